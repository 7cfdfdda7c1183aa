/*
 * roadrunner_oracle.c - TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, scalar fp64 CPU statement of the RoadRunner transit model (H. Parviainen,
 * arXiv:2009.08500; citations are PAPER.md line numbers).  It exists to check the CUDA library
 * (paper_2009_08500_b200/) and to be timed beside it by bench.py's cpu_baseline leg.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.  It
 * shares no code, header, table or constant with the CUDA path and neither imports the other.
 *
 * Layers:
 *   L1  "direct" Eq. (5):  F = (Istar - (w.l) a(c,k)) / Istar with the weight vector w computed at
 *       exactly the requested (c,k).
 *   L2  "interpolated" model: (k,g) weight tensor built once, per-pv table
 *       T = W.ldp, per-point g-interpolation, Keplerian
 *       separation, supersampling and heterogeneous light curves.
 * The L0 truth (Eq. (2) by quadrature) lives in oracle/truth.py.
 *
 * Readings of the paper where it is silent are numbered R1..R12 in DESIGN.md section 3 and named
 * in the comments below.  No blocking, fusion or reordering: every function is the formula.
 *
 * Pins (tests/test_oracle_*.py): lens area vs closed forms, 40-digit values and quadrature;
 * weights sum / support / c=0 closed form; uniform disk F = 1 - a/pi; L1 vs L0 quadrature <= 1e-8;
 * Istar vs analytic integrals; Kepler residual, e=0 equivalence, z(t0) = b; flux invariants;
 * supersampling vs an expanded time array; heterogeneous indexing vs per-light-curve evaluation.
 * Parity unpinned (nothing in the paper fixes them beyond the error band it quotes): the choice
 * zm = edge mean (R1), the default resolutions (R2), the midpoint sub-sample placement (R7).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define OR_PI 3.14159265358979323846264338327950288

/* ---- step 1: z grid (reading R1: zm is the arithmetic mean of the edges) ------ */
void oracle_z_grid(double zcut, int nzin, int nzlimb, double *ze, double *zm, double *mu)
{
    int nz = nzin + nzlimb;
    for (int j = 0; j <= nzin; ++j)                 /* inner region: constant dz */
        ze[j] = (double)j * zcut / (double)nzin;
    double mucut = sqrt(1.0 - zcut * zcut);
    for (int m = 1; m <= nzlimb; ++m) {             /* outer region: constant dmu */
        double mue = mucut * (1.0 - (double)m / (double)nzlimb);
        ze[nzin + m] = sqrt(1.0 - mue * mue);
    }
    ze[nz] = 1.0;
    for (int j = 0; j < nz; ++j) {
        zm[j] = 0.5 * (ze[j] + ze[j + 1]);
        mu[j] = sqrt(1.0 - zm[j] * zm[j]);
    }
}

/* ---- step 2: circle-circle intersection area (textbook lens, reading R9) ----
 * Radii r1, r2, centre distance d.  Partial overlap: the two circular sectors minus the kite,
 *   area = r1^2*alpha + r2^2*beta - D/2,  D = sqrt((-d+r1+r2)(d+r1-r2)(d-r1+r2)(d+r1+r2)) = 4*triangle
 *   alpha = atan2(D, d^2+r1^2-r2^2), beta = atan2(D, d^2+r2^2-r1^2)   (half-angles at the centres)
 * which is the acos form with cos(alpha) = (d^2+r1^2-r2^2)/(2 d r1), sin(alpha) = D/(2 d r1); the
 * atan2 form keeps full precision at the contact points where acos loses half its digits. */
double oracle_lens_area(double r1, double r2, double d)
{
    if (d >= r1 + r2) return 0.0;
    double rmin = r1 < r2 ? r1 : r2;
    if (d <= fabs(r1 - r2)) return OR_PI * rmin * rmin;
    double D = sqrt((-d + r1 + r2) * (d + r1 - r2) * (d - r1 + r2) * (d + r1 + r2));
    double alpha = atan2(D, (d - r2) * (d + r2) + r1 * r1);
    double beta = atan2(D, (d - r1) * (d + r1) + r2 * r2);
    return r1 * r1 * alpha + r2 * r2 * beta - 0.5 * D;
}

/* The same area in the acos form most textbooks print; used only by a pin that cross-checks the
 * two away from the contact points. */
double oracle_lens_area_acos(double r1, double r2, double d)
{
    if (d >= r1 + r2) return 0.0;
    double rmin = r1 < r2 ? r1 : r2;
    if (d <= fabs(r1 - r2)) return OR_PI * rmin * rmin;
    double D = sqrt((-d + r1 + r2) * (d + r1 - r2) * (d - r1 + r2) * (d + r1 + r2));
    return r1 * r1 * acos((d * d + r1 * r1 - r2 * r2) / (2.0 * d * r1))
         + r2 * r2 * acos((d * d + r2 * r2 - r1 * r1) / (2.0 * d * r2)) - 0.5 * D;
}

/* ---- step 3: weight vector w(c,k) (Fig. 1) ----------------------------------------
 * w_j = [A(ze[j+1]) - A(ze[j])] / a(c,k), A(r) = area common to the planet disc (radius k, centre
 * distance c) and the stellar disc of radius r; a(c,k) = A(1).  Reading R5: at c >= 1+k (a = 0)
 * the limit is taken - all weight in the outermost annulus. */
void oracle_weights(double c, double k, const double *ze, int nz, double *w)
{
    double a = oracle_lens_area(1.0, k, c);
    if (!(a > 0.0)) {
        for (int j = 0; j < nz; ++j) w[j] = 0.0;
        w[nz - 1] = 1.0;
        return;
    }
    for (int j = 0; j < nz; ++j) {
        double Ahi = oracle_lens_area(ze[j + 1], k, c);
        double Alo = (ze[j] > 0.0) ? oracle_lens_area(ze[j], k, c) : 0.0;
        w[j] = (Ahi - Alo) / a;
    }
}

/* ---- step 4: (k,g) weight tensor W[nk][ng][nz] -------------------------
 * k_ik = k0 + ik*dk, dk = (k1-k0)/(nk-1); g_ig = ig*dg, dg = 1/(ng-1); c = g_ig*(1+k_ik). */
void oracle_weight_tensor(int nk, double k0, double k1, int ng, const double *ze, int nz, double *W)
{
    double dk = (k1 - k0) / (double)(nk - 1);
    double dg = 1.0 / (double)(ng - 1);
    for (int ik = 0; ik < nk; ++ik) {
        double k = k0 + ik * dk;
        for (int ig = 0; ig < ng; ++ig) {
            double g = (ig == ng - 1) ? 1.0 : ig * dg;
            oracle_weights(g * (1.0 + k), k, ze, nz, W + ((size_t)ik * ng + ig) * nz);
        }
    }
}

/* ---- step 5: per-(pv,passband) table T[row][ik][ig] = sum_j W[ik][ig][j]*ldp[row][j] ----------
 * ("ldw = dot(w, ldp)", :131 for both bracketing k rows; the full table is kept). */
void oracle_ld_table(const double *W, int nk, int ng, int nz, const double *ldp, int64_t nrows,
                     double *T)
{
    for (int64_t r = 0; r < nrows; ++r)
        for (int n = 0; n < nk * ng; ++n) {
            double s = 0.0;
            for (int j = 0; j < nz; ++j) s += W[(size_t)n * nz + j] * ldp[r * nz + j];
            T[r * (int64_t)(nk * ng) + n] = s;
        }
}

/* ---- step 6: Istar = 2 pi int_0^1 z I(z) dz on the model's own annuli (Eq. (2); reading R6) ----
 * Istar = pi * sum_j ldp[j] * (ze[j+1]^2 - ze[j]^2): same bins and mid-bin samples as the weights. */
void oracle_istar(const double *ze, int nz, const double *ldp, int64_t nrows, double *istar)
{
    for (int64_t r = 0; r < nrows; ++r) {
        double s = 0.0;
        for (int j = 0; j < nz; ++j) s += ldp[r * nz + j] * (ze[j + 1] * ze[j + 1] - ze[j] * ze[j]);
        istar[r] = OR_PI * s;
    }
}

/* ---- L1 direct model, Eq. (5) ------------------------------------------------ */
double oracle_direct_flux(double k, double c, const double *ze, int nz, const double *ldp,
                          double istar)
{
    double a = oracle_lens_area(1.0, k, c);
    if (!(a > 0.0)) return 1.0;
    double *w = (double *)malloc(sizeof(double) * (size_t)nz);
    oracle_weights(c, k, ze, nz, w);
    double ip = 0.0;
    for (int j = 0; j < nz; ++j) ip += w[j] * ldp[j];
    free(w);
    return (istar - ip * a) / istar;
}

/* ---- step 8: Kepler's equation E - e sin E = M (reading R8) ----------------
 * Newton from E0 = M + e sin M, safeguarded by bisection on the bracket [M-e, M+e] (f is
 * increasing), until |dE| <= 1e-15 or 50 iterations.  Returns the iteration count. */
int oracle_kepler(double M, double e, double *Eout)
{
    double lo = M - e, hi = M + e;
    double E = M + e * sin(M);
    int it = 0;
    for (; it < 50; ++it) {
        double f = E - e * sin(E) - M;
        if (f > 0.0) hi = E; else lo = E;
        double En = E - f / (1.0 - e * cos(E));
        if (!(En >= lo && En <= hi)) En = 0.5 * (lo + hi);   /* Newton left the bracket: bisect */
        double dE = En - E;
        E = En;
        if (fabs(dE) <= 1e-15) { ++it; break; }
    }
    *Eout = E;
    return it;
}

/* Sky-projected planet-star separation z at time t in units of the stellar radius, and whether the
 * planet is on the observer's side of the star.  t0 = time of inferior conjunction (true anomaly
 * f = pi/2 - w), p period, a semi-major axis / stellar radius, inc inclination, e, w (radians). */
double oracle_separation(double t, double t0, double p, double a, double inc, double e, double w,
                         int *in_front)
{
    double phi = 2.0 * OR_PI * (t - t0) / p;
    if (e == 0.0) {                                   /* circular: closed form */
        double s = sin(phi), c = cos(phi), ci = cos(inc);
        *in_front = c > 0.0;
        return a * sqrt(s * s + c * c * ci * ci);
    }
    double ftr = 0.5 * OR_PI - w;                     /* true anomaly at inferior conjunction */
    double Etr = 2.0 * atan2(sqrt(1.0 - e) * sin(0.5 * ftr), sqrt(1.0 + e) * cos(0.5 * ftr));
    double Mtr = Etr - e * sin(Etr);
    double M = Mtr + phi;
    M = M - 2.0 * OR_PI * floor((M + OR_PI) / (2.0 * OR_PI));      /* to [-pi, pi) */
    double E;
    oracle_kepler(M, e, &E);
    double f = 2.0 * atan2(sqrt(1.0 + e) * sin(0.5 * E), sqrt(1.0 - e) * cos(0.5 * E));
    double r = a * (1.0 - e * e) / (1.0 + e * cos(f));
    double swf = sin(w + f), si = sin(inc);
    *in_front = swf > 0.0;
    return r * sqrt(1.0 - swf * swf * si * si);
}

/* ---- step 9: one sub-sample's flux from the table (reading R10) ---- */
/* kw = the radius ratio the limb-darkening weights are taken at: k itself, or the mean of the pv's
 * radius ratios over the passbands (transmission-spectroscopy shortcut, reading
 * R13: the weight array - its g axis included - is that of a planet of radius kw; the passband's
 * own k sets the transit's extent and the intersection area). */
double oracle_flux_from_table_kw(double z, double k, double kw, const double *T /*[nk][ng]*/,
                                 int nk, double k0, double k1, int ng, double istar)
{
    if (z >= 1.0 + k) return 1.0;
    double dk = (k1 - k0) / (double)(nk - 1), dg = 1.0 / (double)(ng - 1);
    double x = (kw - k0) / dk;
    int ik = (int)floor(x);
    if (ik > nk - 2) ik = nk - 2;
    if (ik < 0) ik = 0;
    double ak = x - ik;
    double y = (z / (1.0 + kw)) / dg;      /* the weights belong to a planet of radius kw at z */
    if (y > (double)(ng - 1)) y = (double)(ng - 1);   /* 1+kw <= z < 1+k: limb node (R5, R13) */
    int ig = (int)floor(y);
    if (ig > ng - 2) ig = ng - 2;
    double ag = y - ig;
    const double *T0 = T + (size_t)ik * ng, *T1 = T + (size_t)(ik + 1) * ng;
    double ip = (1.0 - ak) * ((1.0 - ag) * T0[ig] + ag * T0[ig + 1])
              + ak * ((1.0 - ag) * T1[ig] + ag * T1[ig + 1]);
    double ap = oracle_lens_area(1.0, k, z);
    return (istar - ip * ap) / istar;
}

double oracle_flux_from_table(double z, double k, const double *T /*[nk][ng]*/, int nk, double k0,
                              double k1, int ng, double istar)
{
    return oracle_flux_from_table_kw(z, k, k, T, nk, k0, k1, ng, istar);
}

/* Per-pv validity (reading R12): bit 0 k outside [k0,k1]; bit 1 e outside [0,1); bit 2 a <= 0;
 * bit 3 p <= 0; bit 4 a non-finite parameter. */
int oracle_pv_status(const double *pv, int nkpb, double k0, double k1)
{
    int st = 0;
    for (int q = 0; q < nkpb + 6; ++q) if (!isfinite(pv[q])) st |= 16;
    if (st) return st;
    for (int q = 0; q < nkpb; ++q) if (pv[q] < k0 || pv[q] > k1) st |= 1;
    const double *o = pv + nkpb;   /* t0 p a i e w */
    if (o[4] < 0.0 || o[4] >= 1.0) st |= 2;
    if (o[2] <= 0.0) st |= 4;
    if (o[1] <= 0.0) st |= 8;
    return st;
}

void oracle_evaluate_mk(const double *times, const int32_t *lc_index, int64_t npt,
                        const int32_t *passband_index, const int32_t *supersampling,
                        const double *exposure_time, int32_t nlc,
                        const double *pv, int32_t nkpb, int64_t npv,
                        const double *T, const double *istar,
                        int32_t npb, int32_t nk, double k0, double k1, int32_t ng,
                        int32_t mean_k_weights,
                        double *flux, int32_t *status, double *z_out, int32_t nthreads);

/* ---- steps 7-10: the whole L2 evaluation ---------------------------------------------------------
 * flux[npv][npt]; z_out (optional) [npv][nsub], nsub = sum over exposures of their ns, sub-samples
 * of exposure i stored contiguously in exposure order; behind-the-star sub-samples store -z.
 * Sub-sample times (reading R7): t_{i,s} = times[i] + exptime*((s+0.5)/ns - 0.5). */
void oracle_evaluate(const double *times, const int32_t *lc_index, int64_t npt,
                     const int32_t *passband_index, const int32_t *supersampling,
                     const double *exposure_time, int32_t nlc,
                     const double *pv, int32_t nkpb, int64_t npv,
                     const double *T /*[npv][npb][nk][ng]*/, const double *istar /*[npv][npb]*/,
                     int32_t npb, int32_t nk, double k0, double k1, int32_t ng,
                     double *flux, int32_t *status, double *z_out, int32_t nthreads)
{
    oracle_evaluate_mk(times, lc_index, npt, passband_index, supersampling, exposure_time, nlc, pv,
                       nkpb, npv, T, istar, npb, nk, k0, k1, ng, 0, flux, status, z_out, nthreads);
}

/* mean_k_weights != 0: PAPER.md:188-190, LD weights at the mean of the pv's radius ratios. */
void oracle_evaluate_mk(const double *times, const int32_t *lc_index, int64_t npt,
                        const int32_t *passband_index, const int32_t *supersampling,
                        const double *exposure_time, int32_t nlc,
                        const double *pv, int32_t nkpb, int64_t npv,
                        const double *T, const double *istar,
                        int32_t npb, int32_t nk, double k0, double k1, int32_t ng,
                        int32_t mean_k_weights,
                        double *flux, int32_t *status, double *z_out, int32_t nthreads)
{
    (void)nlc;
    int64_t nsub = 0;
    for (int64_t i = 0; i < npt; ++i) nsub += supersampling[lc_index[i]];
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t v = 0; v < npv; ++v) {
        const double *row = pv + v * (nkpb + 6);
        const double *o = row + nkpb;
        double t0 = o[0], p = o[1], a = o[2], inc = o[3], e = o[4], w = o[5];
        int st = oracle_pv_status(row, nkpb, k0, k1);
        if (status) status[v] = st;
        if (st) {
            for (int64_t i = 0; i < npt; ++i) flux[v * npt + i] = NAN;
            if (z_out) for (int64_t q = 0; q < nsub; ++q) z_out[v * nsub + q] = NAN;
            continue;
        }
        int64_t q = 0;
        for (int64_t i = 0; i < npt; ++i) {
            int l = lc_index[i];
            int pb = passband_index[l];
            int ns = supersampling[l];
            double tau = exposure_time[l];
            double k = row[nkpb == 1 ? 0 : pb];
            double kw = k;
            if (mean_k_weights) {
                kw = 0.0;
                for (int q = 0; q < nkpb; ++q) kw += row[q];
                kw /= (double)nkpb;
            }
            const double *Tvp = T + ((size_t)v * npb + pb) * (size_t)(nk * ng);
            double is = istar[v * npb + pb];
            double sum = 0.0;
            for (int s = 0; s < ns; ++s) {
                double t = times[i] + tau * ((s + 0.5) / (double)ns - 0.5);
                int front;
                double z = oracle_separation(t, t0, p, a, inc, e, w, &front);
                if (z_out) z_out[v * nsub + q++] = front ? z : -z;
                sum += front ? oracle_flux_from_table_kw(z, k, kw, Tvp, nk, k0, k1, ng, is) : 1.0;
            }
            flux[v * npt + i] = sum / (double)ns;        /* mean over sub-samples */
            if (!isfinite(times[i])) flux[v * npt + i] = NAN;   /* reading R15: no time, no flux */
        }
    }
}

/* ==== direct model ==========================================
 * The paper's default: no k grid.  Per (pv, passband) the weights are computed at the pv's own k,
 * `dg, w = calculate_weights(k, ze, ng)`, and `ldw = dot(w, ldp)`; per point only
 * the g interpolation of PAPER.md:101-105 remains.  Same g nodes and g = 1 limit (R5) as the table
 * model; any k > 0 is valid. */
void oracle_direct_rows(const double *ze, int nz, int ng, const double *k /*[nrows]*/,
                        const double *ldp /*[nrows][nz]*/, int64_t nrows, double *rows /*[nrows][ng]*/)
{
    double dg = 1.0 / (double)(ng - 1);
    double *w = (double *)malloc(sizeof(double) * (size_t)nz);
    for (int64_t r = 0; r < nrows; ++r)
        for (int ig = 0; ig < ng; ++ig) {
            double g = (ig == ng - 1) ? 1.0 : ig * dg;
            oracle_weights(g * (1.0 + k[r]), k[r], ze, nz, w);
            double s = 0.0;
            for (int j = 0; j < nz; ++j) s += w[j] * ldp[r * nz + j];
            rows[r * ng + ig] = s;                      /* ldw = dot(w, ldp) */
        }
    free(w);
}

/* One sub-sample's flux from a direct-model row (reading R10 for the last cell). */
double oracle_flux_from_row_kw(double z, double k, double kw, const double *ldw /*[ng]*/, int ng,
                               double istar)
{
    if (z >= 1.0 + k) return 1.0;
    double dg = 1.0 / (double)(ng - 1);
    double y = (z / (1.0 + kw)) / dg;
    if (y > (double)(ng - 1)) y = (double)(ng - 1);
    int ig = (int)floor(y);
    if (ig > ng - 2) ig = ng - 2;
    double ag = y - ig;
    double ip = (1.0 - ag) * ldw[ig] + ag * ldw[ig + 1];
    double ap = oracle_lens_area(1.0, k, z);
    return (istar - ip * ap) / istar;
}

double oracle_flux_from_row(double z, double k, const double *ldw /*[ng]*/, int ng, double istar)
{
    return oracle_flux_from_row_kw(z, k, k, ldw, ng, istar);
}

/* The whole direct-model evaluation: as oracle_evaluate, with rows[npv][npb][ng] from
 * oracle_direct_rows in place of the table, and k > 0 the only limit on k (status bit 0).
 * mean_k_weights: the rows were built at the pv's mean k (reading R13). */
void oracle_evaluate_direct(const double *times, const int32_t *lc_index, int64_t npt,
                            const int32_t *passband_index, const int32_t *supersampling,
                            const double *exposure_time, const double *pv, int32_t nkpb,
                            int64_t npv, const double *rows, const double *istar, int32_t npb,
                            int32_t ng, int32_t mean_k_weights, double *flux, int32_t *status,
                            int32_t nthreads)
{
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t v = 0; v < npv; ++v) {
        const double *row = pv + v * (nkpb + 6);
        const double *o = row + nkpb;
        double t0 = o[0], p = o[1], a = o[2], inc = o[3], e = o[4], w = o[5];
        int st = oracle_pv_status(row, nkpb, 1e-300, 1e300);
        if (status) status[v] = st;
        if (st) {
            for (int64_t i = 0; i < npt; ++i) flux[v * npt + i] = NAN;
            continue;
        }
        for (int64_t i = 0; i < npt; ++i) {
            int l = lc_index[i];
            int pb = passband_index[l];
            int ns = supersampling[l];
            double tau = exposure_time[l];
            double k = row[nkpb == 1 ? 0 : pb];
            double kw = k;
            if (mean_k_weights) {
                kw = 0.0;
                for (int q = 0; q < nkpb; ++q) kw += row[q];
                kw /= (double)nkpb;
            }
            const double *ldw = rows + ((size_t)v * npb + pb) * (size_t)ng;
            double is = istar[v * npb + pb];
            double sum = 0.0;
            for (int s = 0; s < ns; ++s) {
                double t = times[i] + tau * ((s + 0.5) / (double)ns - 0.5);
                int front;
                double z = oracle_separation(t, t0, p, a, inc, e, w, &front);
                sum += front ? oracle_flux_from_row_kw(z, k, kw, ldw, ng, is) : 1.0;
            }
            flux[v * npt + i] = sum / (double)ns;
            if (!isfinite(times[i])) flux[v * npt + i] = NAN;   /* reading R15 */
        }
    }
}

/* ==== small-planet approximation (reading R14) ====================
 * "If the planet is small enough, the weighted average can be replaced with the limb darkening
 * value evaluated at the centre of the planet."  The profile is known at the bin means zm (R1):
 * its value at z is the linear interpolant over zm, held constant before the first and after the
 * last node (a centre beyond the limb sees the limb sample, consistent with R5).  In the row
 * formalism of PAPER.md:97-105 the node g_ig holds the profile at z = g_ig (1+k). */
double oracle_profile_at(double z, const double *zm, const double *ldp, int nz)
{
    if (z <= zm[0]) return ldp[0];
    if (z >= zm[nz - 1]) return ldp[nz - 1];
    int j = 0;
    while (zm[j + 1] <= z) ++j;                        /* zm[j] <= z < zm[j+1] */
    double a = (z - zm[j]) / (zm[j + 1] - zm[j]);
    return (1.0 - a) * ldp[j] + a * ldp[j + 1];
}

/* Direct-model rows with the small-planet approximation for rows whose k <= k_small
 * (k_small <= 0: never). */
void oracle_direct_rows_sp(const double *ze, const double *zm, int nz, int ng, const double *k,
                           const double *ldp, int64_t nrows, double k_small, double *rows)
{
    double dg = 1.0 / (double)(ng - 1);
    for (int64_t r = 0; r < nrows; ++r) {
        if (k_small > 0.0 && k[r] <= k_small) {
            for (int ig = 0; ig < ng; ++ig) {
                double g = (ig == ng - 1) ? 1.0 : ig * dg;
                rows[r * ng + ig] = oracle_profile_at(g * (1.0 + k[r]), zm, ldp + r * nz, nz);
            }
        } else {
            oracle_direct_rows(ze, nz, ng, k + r, ldp + r * nz, 1, rows + r * ng);
        }
    }
}

/* Direct-model rows[npv][npb][ng] straight from the parameter vectors: the weight radius of row
 * (pv, pb) is the pv's k for that passband, or, with mean_k_weights, the mean of the pv's radius
 * ratios (reading R13).  Rows of pvs whose k is not finite and > 0 (reading R12:
 * NaN flux rows, never read by oracle_evaluate_direct) are filled with NaN. */
void oracle_direct_rows_pv(const double *ze, const double *zm, int nz, int ng, const double *pv,
                           int32_t nkpb, int32_t npb, int64_t npv, int32_t mean_k_weights,
                           const double *ldp /*[npv][npb][nz]*/, double k_small,
                           double *rows /*[npv][npb][ng]*/)
{
    for (int64_t v = 0; v < npv; ++v) {
        const double *row = pv + v * (nkpb + 6);
        int ok = 1;
        double kmean = 0.0;
        for (int q = 0; q < nkpb; ++q) {
            if (!isfinite(row[q]) || !(row[q] > 0.0)) ok = 0;
            kmean += row[q];
        }
        kmean /= (double)nkpb;
        for (int pb = 0; pb < npb; ++pb) {
            int64_t r = v * npb + pb;
            if (!ok) {
                for (int ig = 0; ig < ng; ++ig) rows[r * ng + ig] = NAN;
                continue;
            }
            double k = mean_k_weights ? kmean : row[nkpb == 1 ? 0 : pb];
            oracle_direct_rows_sp(ze, zm, nz, ng, &k, ldp + r * nz, 1, k_small, rows + r * ng);
        }
    }
}

