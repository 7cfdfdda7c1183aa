/*
 * roadrunner.h - C-ABI of the B200-native RoadRunner transit-model library
 *                (libroadrunner_b200.so, sm_100a CUDA kernels behind plain C entry points).
 *
 * The method is H. Parviainen, "RoadRunner: a fast and flexible exoplanet transit model"
 * (arXiv:2009.08500).  Citations below are PAPER.md line numbers (section / equation); readings
 * of the paper where it is silent are numbered R1..R15 in DESIGN.md section 3.
 *
 * The two calls of the problem statement are
 *     build_ld_table(ldp[npv x npb x nz])                                   -> rr_build_ld_table
 *     evaluate(times, lc_index, passband_index, supersampling, exposure_time,
 *              pv[npv x npar]) -> flux[npv x npt]                  -> rr_set_data + rr_evaluate
 * following the paper's call pattern "set_data once, evaluate many times";
 * rr_evaluate_flat is the one-call form with the problem statement's flat argument list.
 *
 * Conventions (every entry point)
 *   - extern "C", plain pointers and sizes; no C++ or torch types cross the boundary.
 *   - A pointer named d_* is a DEVICE pointer, h_* a HOST pointer.  All are owned by the caller;
 *     the library never frees or keeps them beyond the call unless stated (rr_set_data copies).
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls are
 *     asynchronous on that stream unless stated.
 *   - Return value: 0 = ok; a negative RR_E* code = argument/state error detected on the host
 *     before anything was launched; <= -1000 = CUDA error (-1000 - cudaError_t).
 *     rr_error_string() names any code.  No exception crosses the ABI.
 *   - There is no CPU fallback: without a CUDA device every compute call fails with a CUDA error.
 *   - A ctx is not thread-safe and keeps ONE set of per-evaluation buffers for the device-pointer
 *     API: calls on the same ctx must be issued from one host thread at a time and, if they go to
 *     different streams, ordered by the caller (two evaluations in flight need two contexts).  In
 *     steady state (same npv, same data) rr_build_ld_table* and rr_evaluate allocate nothing and
 *     synchronise nothing, so a step can be captured into a CUDA graph.
 *
 * Per-parameter-vector validity (reading R12): a parameter vector whose k is outside [k0,k1] (in
 * RR_TABLE_DIRECT mode: k <= 0), whose
 * e is outside [0,1), whose a <= 0 or p <= 0, or that holds a non-finite value gets an all-NaN
 * flux row and a non-zero status word (bits below); the call itself still returns 0, so that a
 * sampler does not lose its other walkers.
 */
#ifndef ROADRUNNER_B200_H
#define ROADRUNNER_B200_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- codes ------------------------------------------------------------------------------- */
#define RR_FP64 0
#define RR_FP32 1
#define RR_MIXED 2           /* the paper's proposed scheme: z and Ip*Ap in fp32; their
                                average over the sub-samples, 1 - avg/Istar and the stored flux in
                                fp64.  ldp, istar, table: fp32; flux: fp64                        */

#define RR_OK            0
#define RR_ENULL        -1   /* a required pointer is NULL                                     */
#define RR_ECONFIG      -2   /* rr_config out of range                                         */
#define RR_ESIZE        -3   /* a size is <= 0 or inconsistent (npar, npv, npt, nlc)           */
#define RR_EINDEX       -4   /* lc_index / passband_index / supersampling out of range         */
#define RR_ESTATE       -5   /* call order: evaluate before set_data / build_ld_table, or npv  */
#define RR_EALLOC       -6   /* device or host allocation failed                               */
#define RR_ESCRATCH     -7   /* rr_orbit_z_noalloc: problem exceeds the static scratch array   */
#define RR_ECUDA_BASE   -1000

/* status bits written per parameter vector (reading R12) */
#define RR_PV_K_RANGE    1   /* some k outside [k0, k1]            */
#define RR_PV_E_RANGE    2   /* e outside [0, 1)                   */
#define RR_PV_A_RANGE    4   /* a <= 0                             */
#define RR_PV_P_RANGE    8   /* p <= 0                             */
#define RR_PV_NONFINITE 16   /* a NaN or infinity in the row       */

/* how rr_build_ld_table / rr_evaluate share kernel 1's work (rr_set_table_mode) */
#define RR_TABLE_LAZY     0  /* default: keep the profile, build at rr_evaluate only the two
                                bracketing k rows each pv's k needs, collapsed */
#define RR_TABLE_FULL     1  /* rr_build_ld_table builds the whole T[npv][npb][nk][ng]            */
#define RR_TABLE_DIRECT   2  /* the paper's direct model: no k grid; at
                                rr_evaluate the weights are computed at each pv's own k and contracted
                                with its profile (g interpolation only); any k > 0 is valid        */

/* named limb-darkening laws (rr_build_ld_table_law); x = 1 - mu */
#define RR_LD_UNIFORM       0  /* I = 1                                                nldc 0  */
#define RR_LD_LINEAR        1  /* 1 - u x                                                   1  */
#define RR_LD_QUADRATIC     2  /* 1 - u1 x - u2 x^2                                         2  */
#define RR_LD_QUADRATIC_TRI 3  /* quadratic with u1 = 2 sqrt(q1) q2, u2 = sqrt(q1)(1 - 2 q2) 2  */
#define RR_LD_GENERAL       4  /* 1 - sum_{n=1..N} c_n (1 - mu^n)                        N<=64  */
#define RR_LD_NONLINEAR     5  /* 1 - sum_{n=1..4} c_n (1 - mu^(n/2))                       4  */
#define RR_LD_LOGARITHMIC   6  /* 1 - u1 x - u2 mu ln mu                                    2  */
#define RR_LD_EXPONENTIAL   7  /* 1 - u1 x - u2 / (1 - e^mu)   (Istar by reading R6)        2  */
#define RR_LD_POWER2        8  /* 1 - c (1 - mu^alpha)                                      2  */
#define RR_LD_POWER2_PM     9  /* power-2 with c = 1 - h1 + h2, alpha = log2(c / h2)        2  */

/* supersample reduction layout of the fused flux kernel (rr_set_reduction) */
#define RR_REDUCE_AUTO    0  /* library picks per light curve from ns and the amount of work    */
#define RR_REDUCE_THREAD  1  /* one thread per exposure, in-thread loop over its sub-samples    */
#define RR_REDUCE_SHUFFLE 2  /* sub-samples across lanes, warp-shuffle sum       */

typedef struct rr_ctx rr_ctx;   /* opaque; owned by the library */

/* Resolution of the model: what the paper's RoadRunnerModel constructor fixes
 * (PAPER.md:83-92 z grid; :116-122 (k,g) weight table).                                        */
typedef struct {
  int32_t nzin;      /* radial bins of constant dz  on [0, zcut]                 (>= 1)          */
  int32_t nzlimb;    /* radial bins of constant dmu on [zcut, 1]; nz = nzin+nzlimb (>= 1)        */
  double  zcut;      /* 0 < zcut < 1                                                             */
  int32_t ng;        /* nodes of g = z/(1+k) on [0,1], g_i = i/(ng-1)            (>= 2)          */
  int32_t nk;        /* nodes of the radius ratio, k_i = k0 + i (k1-k0)/(nk-1)   (>= 2)          */
  double  k0, k1;    /* 0 < k0 < k1                                                              */
  int32_t npb;       /* passbands                                                (>= 1)          */
  int32_t nkpb;      /* 1 = one k per parameter vector; npb = one k per passband  */
  int32_t precision; /* RR_FP64, RR_FP32 (type of ldp, istar, the table and flux) or RR_MIXED    */
} rr_config;

/* ---- life cycle ------------------------------------------------------------------------------
 * rr_create builds, on the current CUDA device, the z grid ze[nz+1], zm[nz], mu[nz]
 * (zm = edge mean, reading R1) and the geometry weight tensor W[nk][ng][nz]
 * (g = 1 node = limit, reading R5) in fp64.  Synchronous.          */
int rr_create(const rr_config *cfg, rr_ctx **out);
int rr_destroy(rr_ctx *ctx);
const char *rr_error_string(int code);

/* Grid read-back (host arrays, fp64): the caller samples its limb-darkening law at mu[nz]
 * (PAPER.md:89, :98).  h_W (optional diagnostics) receives W[nk][ng][nz].  Synchronous.         */
int rr_get_mu(const rr_ctx *ctx, double *h_mu /*[nz]*/);
int rr_get_ze(const rr_ctx *ctx, double *h_ze /*[nz+1]*/);
int rr_get_weights(const rr_ctx *ctx, double *h_W /*[nk][ng][nz]*/);

/* ---- data: paper's tm.set_data(times, lcids, pbids, nsamples, exptimes), PAPER.md:230-236 -----
 * d_times[npt]          mid-exposure times (days), fp64, any order; a NaN or infinite time gives
 *                       NaN flux for that exposure (reading R15)
 * d_lc_index[npt]       light-curve index of each exposure, 0 <= . < nlc
 * h_passband_index[nlc] passband of each light curve, 0 <= . < npb     (reading R11: per light
 *                       curve, as in the paper; per-point passband = passband_index[lc_index[i]])
 * h_supersampling[nlc]  sub-samples per exposure, >= 1
 * h_exposure_time[nlc]  exposure time (days), >= 0; sub-sample s of n sits at
 *                       t + tau*((s+1/2)/n - 1/2)                               (reading R7)
 * The library copies all five and runs the heterogeneous-dispatch kernels (DESIGN.md section 6,
 * kernel 4), which cut the exposure axis into tiles of one light curve each (uniform ns, tau,
 * passband; at most 1024 R exposures, R = clamp((8 + ns/2)/ns, 1, 8), and at most 0.1 d at the
 * run's mean cadence, in multiples of 128) with their time range.  Synchronous on `stream` (it reads back the tile count).
 * RR_EINDEX if any index is out of range (nothing is kept then).                                */
int rr_set_data(rr_ctx *ctx, const double *d_times, const int32_t *d_lc_index, int64_t npt,
                const int32_t *h_passband_index, const int32_t *h_supersampling,
                const double *h_exposure_time, int32_t nlc, void *stream);

/* ---- kernel 1: LD table, PAPER.md:98-99, :127-131 -----------------------------------------------
 * d_ldp[npv][npb][nz]  the limb-darkening profile sampled at mu[nz] (ctx precision)
 * d_istar[npv][npb]    optional disk-integrated brightness (ctx precision); NULL = reading R6:
 *                      Istar = pi sum_j ldp[j] (ze[j+1]^2 - ze[j]^2)            (Eq. (2))
 * The table is T[npv][npb][nk][ng] = sum_j W[ik][ig][j] ldp[pv][pb][j]; fp64 accumulation in both
 * precisions.  The paper's evaluate needs, per (pv, passband), only the two rows that bracket the
 * pv's k: ldw = (1-ak) dot(w[ik], ldp) + ak dot(w[ik+1], ldp).  This call does
 * not receive k, so:
 *   RR_TABLE_LAZY (default)  copies ldp into a buffer owned by ctx and computes Istar; the next
 *                            rr_evaluate, which knows k, builds exactly those collapsed rows
 *                            ldw[npv][npb][ng] (2/nk of the table's arithmetic) before the flux kernel;
 *   RR_TABLE_FULL            builds all of T here (a [npv npb] x [nk ng] x [nz] product) and
 *                            rr_evaluate collapses the two rows while staging them.
 * Both give the same flux to rounding (tested).  Buffers are owned by ctx and grown as needed.   */
int rr_build_ld_table(rr_ctx *ctx, const void *d_ldp, const void *d_istar, int64_t npv,
                      void *stream);
/* Named laws on the device: evaluates the law RR_LD_* with the
 * coefficients d_ldc[npv][npb][nldc] (fp64, device) at mu[nz] into a profile buffer owned by ctx,
 * takes Istar = 2 pi int_0^1 mu I dmu in closed form ("integrated analytically", PAPER.md:156;
 * RR_LD_EXPONENTIAL has none: reading R6), and then behaves as rr_build_ld_table in the current
 * table mode.  The paper names the laws without printing them: the forms above are the textbook
 * ones of its footnote 4.  RR_ESIZE if nldc does not fit the law.  Asynchronous on `stream`
 * (buffers grow only when a larger npv arrives).                                                 */
int rr_build_ld_table_law(rr_ctx *ctx, int32_t law, const double *d_ldc, int32_t nldc, int64_t npv,
                          void *stream);
/* RR_TABLE_*; takes effect at the next rr_build_ld_table.  RR_TABLE_DIRECT needs nz <= 2000.     */
int rr_set_table_mode(rr_ctx *ctx, int32_t mode);
/* Transmission-spectroscopy shortcut (meaningful with nkpb = npb): on != 0 takes
 * the LD weights of every passband at the MEAN of the pv's radius ratios (one weight array per pv);
 * each passband keeps its own k for g = z/(1+k) and for the intersection area (reading R13).
 * Takes effect at the next rr_evaluate.                                                          */
int rr_set_mean_k_weights(rr_ctx *ctx, int32_t on);
/* Small-planet approximation (reading R14): for rows whose weight radius is
 * <= k_threshold the mean occulted brightness is replaced by the profile's value at the planet's
 * centre (linear interpolation of ldp over the bin means zm, constant beyond the first and last
 * node).  k_threshold = 0 (default) switches it off.  Needs RR_TABLE_LAZY or RR_TABLE_DIRECT
 * (rr_evaluate returns RR_ESTATE on a full table).  Takes effect at the next rr_evaluate.        */
int rr_set_small_planet(rr_ctx *ctx, double k_threshold);
/* Orbit evaluation of the fp64 flux kernel for eccentric orbits (default on != 0): per parameter
 * vector, z^2 over the two halves of its transit window is fitted once per rr_evaluate by two
 * degree-12 polynomials through 26 exact Kepler solves, and every sub-sample
 * evaluates the polynomial instead of solving Kepler's equation; a parameter vector whose polynomials
 * have not converged (Chebyshev tail above 1e-12: wide windows of close-in, very eccentric orbits)
 * and every fp32 / mixed kernel keep the per-sub-sample solve.  Difference to the per-sub-sample
 * solve: <= ~1e-11 in z^2, ~1e-13 in flux (tested).  on = 0: always solve.  Takes effect at the next
 * rr_evaluate.                                                                                    */
int rr_set_orbit_poly(rr_ctx *ctx, int32_t on);
/* Lens area of the flux kernels between the contacts (default on != 0): per (parameter vector,
 * radius ratio <= 0.32) the area a(z, k) on the ingress / egress interval is fitted once per
 * rr_evaluate by two degree-12 polynomials through 26 exact evaluations of the two-sectors-minus-kite
 * area (reading R9) and every sub-sample evaluates the polynomial; larger k
 * take the exact form.  Difference to the exact form: <= 2.5e-13 in area, <= 1e-13 in flux (tested).
 * on = 0: always the exact form (two arctangents per ingress sub-sample).  Takes effect at the next
 * rr_evaluate.                                                                                    */
int rr_set_lens_poly(rr_ctx *ctx, int32_t on);
/* Diagnostics: device pointers to the full table (built on demand in lazy mode; synchronous) and
 * Istar of the last rr_build_ld_table (ctx precision), or NULL.                                 */
const void *rr_table_ptr(rr_ctx *ctx);
const void *rr_istar_ptr(const rr_ctx *ctx);
/* Copies the full table T[npv][npb][nk][ng] (built on demand in lazy mode) and Istar[npv][npb] to
 * host arrays (ctx precision; either may be NULL).  Synchronous (device-wide).                   */
int rr_get_table(rr_ctx *ctx, void *h_T, void *h_istar);
/* Diagnostics (lazy / direct mode, after an rr_evaluate): the collapsed rows ldw[npv][npb][ng] the
 * flux kernel staged (ctx precision) -> host array.  Synchronous (device-wide).                  */
int rr_get_rows(const rr_ctx *ctx, void *h_rows);

/* ---- kernels 2+3+4: evaluate, PAPER.md:101-107, :128-131, :214, :220 ---------------------------
 * d_pv[npv][npar]   fp64 rows [k_0..k_{nkpb-1}, t0, p, a, i, e, w], npar = nkpb + 6: the order of
 *                   the paper's evaluate(k, ldc, t0, p, a, i, e, w) with ldc replaced by ldp.
 *                   t0 = time of inferior conjunction, p period (days), a = semi-major axis /
 *                   stellar radius, i inclination and w argument of periastron in radians.
 * d_flux[npv][npt]  out, ctx precision, row-major, exposure order of d_times.
 * d_status[npv]     out, optional (NULL): status bits above.
 * npv must equal the npv of the last rr_build_ld_table.                                         */
int rr_evaluate(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, void *d_flux,
                int32_t *d_status, void *stream);

/* One-call form with the problem statement's flat argument list: rr_set_data (synchronous) then
 * rr_evaluate.                                                                                  */
int rr_evaluate_flat(rr_ctx *ctx, const double *d_times, const int32_t *d_lc_index, int64_t npt,
                     const int32_t *h_passband_index, const int32_t *h_supersampling,
                     const double *h_exposure_time, int32_t nlc, const double *d_pv, int32_t npar,
                     int64_t npv, void *d_flux, int32_t *d_status, void *stream);

/* ---- kernel 2 alone: projected separation, for tests and diagnostics -------
 * d_z[npv][nsub], nsub = sum over exposures of their ns (rr_num_subsamples), sub-samples of an
 * exposure contiguous, exposure order; fp64 in both precisions of ctx unless fp32_math != 0, in
 * which case the fp32 orbit arithmetic of the RR_FP32 flux kernel is used and widened.  A
 * sub-sample with the planet behind the star stores -z.  Rows of invalid pvs are NaN.  Needs
 * rr_set_data; not rr_build_ld_table.                                                           */
int rr_orbit_z(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, double *d_z,
               int32_t fp32_math, void *stream);
/* The same WITHOUT ANY ALLOCATION, for callers that cannot call cudaMalloc (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid it).  rr_orbit_z keeps its scratch - the per-pv
 * orbit and radius-ratio constants its prep kernel writes - in buffers the ctx grows with cudaMalloc
 * when a larger npv arrives; this call keeps it in ONE static device array of
 * RR_NOALLOC_SCRATCH_BYTES (2 MiB; every GPU that loads the library holds it until exit) and calls
 * no cudaMalloc, cudaFree or allocating library routine.  Arguments, output and arithmetic are those
 * of rr_orbit_z (same kernels).  Limit: 256-aligned(200 npv) + 72 npv nkpb <= RR_NOALLOC_SCRATCH_BYTES,
 * i.e. npv <= 7709 with one radius ratio per parameter vector; beyond it the call returns RR_ESCRATCH
 * and launches nothing.  Must be called with the ctx's device current (RR_ESTATE otherwise).  The
 * array is shared by every call on that device and keeps the last call's contents; nothing in it
 * needs clearing (each call writes the entries it reads before it reads them), but calls that overlap
 * on the GPU - different streams, or several contexts on one device - race on it: serialise them.
 * Asynchronous on `stream`.  Needs rr_set_data.                                                   */
#define RR_NOALLOC_SCRATCH_BYTES (2 << 20)
int rr_orbit_z_noalloc(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, double *d_z,
                       int32_t fp32_math, void *stream);
int64_t rr_num_subsamples(const rr_ctx *ctx);   /* < 0: no data set */
int64_t rr_num_tiles(const rr_ctx *ctx);        /* dispatch tiles of the current data; < 0: none */

/* Dispatch read-back for tests (host arrays of rr_num_tiles entries each): first exposure, number
 * of exposures and light curve of every tile, and its [tmin, tmax] time range.  Synchronous.    */
int rr_get_tiles(const rr_ctx *ctx, int32_t *h_start, int32_t *h_count, int32_t *h_lc,
                 double *h_tmin, double *h_tmax);

/* Supersample reduction layout (RR_REDUCE_*); read at every rr_evaluate.                        */
int rr_set_reduction(rr_ctx *ctx, int32_t mode);

/* ---- whole step with HOST buffers (the end-to-end call) --------------------------------------------
 * h_ldp[npv][npb][nz], h_pv[npv][npar] -> h_flux[npv][npt], h_status[npv] (optional).  Runs
 * rr_build_ld_table + rr_evaluate over chunks of parameter vectors on two internal streams so
 * that the host<->device copies of one chunk overlap the kernels of the next.  Host buffers may be
 * pageable or pinned (pinned ones copy faster).  h_ldp in the ctx input precision (fp32 in RR_FP32
 * and RR_MIXED), h_flux in the flux precision (fp32 only in RR_FP32).  Honours the table mode, the
 * mean-k and the small-planet settings.  Needs rr_set_data.  Synchronous.  Afterwards the host-path
 * buffers hold the LAST chunks only (rr_get_table / rr_get_rows refer to the device-pointer API).   */
int rr_evaluate_host(rr_ctx *ctx, const void *h_ldp, const double *h_pv, int32_t npar, int64_t npv,
                     void *h_flux, int32_t *h_status);

/* ---- measurement aids (bench.py) ---------------------------------------------------------------
 * Counters of the last rr_evaluate on this ctx, filled by the flux kernel when enabled with
 * rr_enable_counters(ctx, 1) (adds atomics; keep off when timing): h_counts[0] sub-samples of
 * evaluated tiles skipped as out of the transit window (sub-samples of tiles filled whole are not
 * counted: total - [0] - [1] - [2]), [1] evaluated circular, [2] evaluated eccentric, [3] of those
 * with z < 1+k in front of the star, [4] of those in ingress/egress (lens area), [5] sincos
 * evaluations of the Kepler solver, [6] tiles (per pv) filled without evaluation, [7] tiles (per
 * pv) evaluated, [8] of [2] those evaluated through the orbit polynomials (no solve).  Synchronous. */
int rr_enable_counters(rr_ctx *ctx, int32_t on);
int rr_get_counters(const rr_ctx *ctx, int64_t *h_counts /*[9]*/);
/* Number of kernel launches the library has made on this ctx since creation.                     */
int64_t rr_launch_count(const rr_ctx *ctx);
/* Device time of the kernels inside rr_evaluate, by CUDA events recorded on the caller's stream
 * around them (rr_enable_kernel_timing(ctx, 1); at most 4096 calls are kept between reads).
 * rr_get_kernel_times sums, over the rr_evaluate calls since the last read, h_ms[0] = the lazy row
 * builder (kernel 1's share at evaluate time; 0 in RR_TABLE_FULL mode) and h_ms[1] = the fused
 * flux kernel, and returns the number of calls in *h_calls.  Synchronous.                        */
int rr_enable_kernel_timing(rr_ctx *ctx, int32_t on);
int rr_get_kernel_times(rr_ctx *ctx, double *h_ms /*[2]*/, int64_t *h_calls);
/* FP64 / FP32 FMA pipe peak of the current device, measured with a register-resident FMA chain
 * (DESIGN.md section 7): returns thread-level FMA instructions per second in *h_fma_per_s.
 * Synchronous.                                                                                   */
int rr_measure_fma_peak(int32_t precision, double *h_fma_per_s, void *stream);

/* ---- test aid: the device math of the hot path, element by element ------------------------------
 * The flux kernel's own square root, division, arctangents, sin / cos - 1 polynomials and table-cell
 * split (csrc/rr_math.cuh; ranges and error bounds in DESIGN.md section 6) applied to d_a[n] (and
 * d_b[n] for the two-argument functions), in fp64 or - fp32_math != 0 - in the fp32 arithmetic of the
 * RR_FP32 kernel (inputs rounded to fp32, results widened).  d_out1 (optional) receives the second
 * result of RR_PROBE_SINCOSM1 (cos x - 1) and RR_PROBE_CELL (the weight a = y - floor y).
 * Asynchronous on `stream`.  Tests compare the results with 50-digit arithmetic.                  */
#define RR_PROBE_SQRT3          0  /* sqrt(a), a > 0: seed + one third-order step                  */
#define RR_PROBE_SQRT           1  /* sqrt(a), any a (0 for a <= 0): seed + two Goldschmidt steps  */
#define RR_PROBE_DIV3           2  /* a / b, b > 0                                                 */
#define RR_PROBE_RCP            3  /* 1 / a to ~1e-12 (fp64) / ~1e-7 (fp32)                        */
#define RR_PROBE_ATAN_T         4  /* atan(a), |a| <= tan(pi/8)                                    */
#define RR_PROBE_ATAN_QUADRANT  5  /* atan(sqrt(b/a)) in [0, pi/2] from S = a > 0, P = b >= 0      */
#define RR_PROBE_ATAN2_POS      6  /* atan2(a, b), a >= 0: the angle in [0, pi]                    */
#define RR_PROBE_SINCOSM1       7  /* sin a, cos a - 1, |a| <= 0.5                                 */
#define RR_PROBE_CELL           8  /* floor(a) and a - floor(a), 0 <= a < 2^31                     */
int rr_math_probe(int32_t op, int32_t fp32_math, const double *d_a, const double *d_b, int64_t n,
                  double *d_out0, double *d_out1, void *stream);

#ifdef __cplusplus
}
#endif
#endif /* ROADRUNNER_B200_H */
