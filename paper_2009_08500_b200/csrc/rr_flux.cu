// rr_flux.cu - kernels 2 and 3: orbit -> projected separation z, and the fused supersampled flux.
//   per-pv prep      validity (reading R12), k-interpolation index, orbit
//                    constants at inferior conjunction, and the transit window in orbital phase
//   rr_orbit_kernel  kernel 2 alone: z for every sub-sample (tests / diagnostics)
//   rr_flux_kernel   kernels 2+3 fused, one block per (parameter vector, chunk of dispatch tiles):
//                    PAPER.md:101-107 (g interpolation, area, flux), :131 (k-collapsed table
//                    row), :214 (supersampling), :220 (orbit parameters); template <R, O>:
//                    R = arithmetic of z and ip*ap, O = sub-sample sum and stored flux
//                    (double/double, float/float, float/double = RR_MIXED)
// Orbit formulation (kernel 2).  Time enters as the phase u = (t - t0)/p in turns,
// reduced in fp64.  z < 1+k in front of the star is only possible in a window around conjunction
// computed per pv; everything outside it has flux 1 exactly and costs a compare.  Inside, Kepler's
// equation is solved for d = E - E_tr (E_tr = eccentric anomaly at inferior conjunction):
//   G(d) = d - e [sin(E_tr + d) - sin E_tr] - dM = 0,
// with every difference from E_tr formed from sin d and cos d - 1, so that the result keeps RELATIVE
// accuracy for small d.  That is what lets the fp32 variant work (a direct fp32 solve for E loses
// a*eps(E) ~ 4e-6 in z), and it removes atan2 and the true anomaly from the path: the sky position
// is linear in (cos d - 1, sin d) with per-pv coefficients.
// Solver: a 4th-order series-reversion starter (exact derivatives of G at d = 0 are per-pv
// constants) and Halley steps, the first accepted for ~91 % of sub-samples: a step below a per-pv
// tolerance bounds the remaining error by ~2e-15 (fp64) and is applied by a second-order rotation of
// (sin d, cos d - 1), so one sincos suffices; anything else (|d| > 0.5, e near 1 at periastron) goes
// to a bracketed Halley/bisection loop.  sin d, cos d - 1 on |d| <= 0.5 are Taylor polynomials with
// their coefficients in constant memory (rr_math.cuh).  Circular orbits in fp64: sin/cos once per
// exposure, one plane rotation per further sub-sample.
// Round 2: out-of-window runs of flux = 1 go out as TMA bulk copies from a block-resident buffer of
// ones (rr_fill_ones_bulk); the fp32 and mixed kernels take two exposures per thread with packed
// FFMA2 arithmetic (rr_tile_pairs) when the tiles are longer than a block; the lens area between the
// contacts (rr_lens_fit) and z^2 over the transit window of an eccentric pv (rr_zpoly_fit)
// come from per-pv degree-12 polynomials fitted through exact evaluations once per rr_evaluate.
#include <algorithm>
#include <mutex>

#include "rr_common.cuh"
#include "rr_math.cuh"
#include "rr_lens_poly.cuh"

// flux is written once and never re-read: streaming stores keep W, times and the rows in L2
#define RR_STORE(p, v) __stcs((p), (v))

// Dynamic shared memory of rr_flux_kernel and rr_orbit_kernel.  Global scope: the PTX symbol is
// "rr_dyn", which the inline loads of Cst<> name directly.
extern __shared__ __align__(16) unsigned char rr_dyn[];

namespace {

#ifndef RR_FLUX_THREADS
#define RR_FLUX_THREADS 128     // measured: 128 x 8 blocks/SM beats 256 x 4 by 5 % (finer barriers, tail)
#endif
constexpr int FT = RR_FLUX_THREADS;   // threads per flux block
#ifndef RR_FLUX_MIN_BLOCKS
#define RR_FLUX_MIN_BLOCKS 8    // resident blocks per SM the register budget (64) is set for
#endif
#ifndef RR_ROBUST_INLINE
#define RR_ROBUST_INLINE __forceinline__   // measured: 2 % faster than a call (fewer spills)
#endif
#ifndef RR_FLUX_WAVES
#define RR_FLUX_WAVES 64        // waves of blocks wanted before the tile axis is left uncut (with the
                                // bulk fill: config 4 64 = 128 waves, config 3 0.7 % slower, the sparse
                                // cadence of 4b 14 % faster than with 128: per-block set-up)
#endif

// ---- per-pv prep ---------------------------------------------------------------------------------
__global__ void rr_pv_prep_kernel(const double *__restrict__ pv, int64_t npv, int nkpb, int nk,
                                  double k0, double k1, double kmin, double kmax_ok, int ng,
                                  int fp32, int mean_k, int row_pad,
                                  RRPvOrbit *__restrict__ pvo, RRPvBand *__restrict__ pvb,
                                  int32_t *__restrict__ status_out) {
  int64_t v = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (v >= npv) return;
  const int npar = nkpb + 6;
  const double *row = pv + v * npar;
  const double *o = row + nkpb;
  double t0 = o[0], p = o[1], a = o[2], inc = o[3], e = o[4], w = o[5];
  int st = 0;
  for (int q = 0; q < npar; ++q)
    if (!isfinite(row[q])) st |= RR_PV_NONFINITE;
  if (!st) {
    for (int q = 0; q < nkpb; ++q)
      if (row[q] < kmin || row[q] > kmax_ok) st |= RR_PV_K_RANGE;
    if (e < 0.0 || e >= 1.0) st |= RR_PV_E_RANGE;
    if (a <= 0.0) st |= RR_PV_A_RANGE;
    if (p <= 0.0) st |= RR_PV_P_RANGE;
  }
  int st_k = 0;
  RRPvOrbit po;
  po.circular = (e == 0.0);
  double kmax = 0.0;
  const double dk = (k1 - k0) / (double)(nk - 1);
  double kmean = 0.0;
  for (int q = 0; q < nkpb; ++q) kmean += row[q];
  kmean /= (double)nkpb;
  for (int q = 0; q < nkpb; ++q) {
    double k = row[q];
    RRPvBand b;
    b.k = k;
    b.opk = 1.0 + k;
    b.omk = fabs(1.0 - k);
    double rmin = fmin(1.0, k);
    b.afull = RR_PI * rmin * rmin;
    b.k2 = k * k;
    const double kw = mean_k ? kmean : k;
    b.kw = kw;
    b.gscale = (double)(ng - 1) / (1.0 + kw);   // the g axis of the weights is that of radius kw
    // mean-k weights: y = z gscale reaches (ng-1)(1+k)/(1+kw); the staged row is padded up to there
    if (!(b.gscale * (1.0 + k) < (double)(ng + row_pad) - 1.5)) st_k = 1;
    double x = (kw - k0) / dk;
    int ik = (int)floor(x);
    ik = min(max(ik, 0), nk - 2);
    b.ik = ik;
    b.ak = x - (double)ik;
    b.lens_ok = (k > 0.0 && k <= RR_LENS_KMAX) ? 1 : 0;
    pvb[v * nkpb + q] = b;
    kmax = fmax(kmax, k);
  }
  if (st_k && !st) st = RR_PV_K_RANGE;
  if (status_out) status_out[v] = st;
  po.status = st;
  po.t0 = t0;
  po.inv_p = 1.0 / p;
  double ci = cos(inc);
  po.zc0 = a * a * ci * ci;
  po.zc1 = a * a * (1.0 - ci * ci);
  po.aci2 = po.zc0;
  po.e = e;
  double sw, cw;
  sincos(w, &sw, &cw);
  if (po.circular) { sw = 0.0; cw = 1.0; }      // w is irrelevant for e = 0
  const double beta = sqrt((1.0 - e) * (1.0 + e));
  const double den = 1.0 + e * sw;
  const double sE = beta * cw / den;            // sin, cos of E at true anomaly pi/2 - w
  const double cE = (e + sw) / den;
  po.sE = sE;
  po.cE = cE;
  // G(d) = d - e [sE (cos d - 1) + cE sin d] - dM:  G' = A, G'' = B, G''' = C, G'''' = -B at d = 0
  const double A = 1.0 - e * cE, B = e * sE, C = e * cE;
  po.A = A;
  po.B = B;
  po.C = C;
  po.invA = 1.0 / A;
  {
    // reversion of y = d + (b/2) d^2 + (c/6) d^3 - (b/24) d^4, y = dM/A, b = B/A, c = C/A
    const double b = B / A, c = C / A;
    po.c2 = -0.5 * b;
    po.c3 = 0.5 * b * b - c / 6.0;
    po.c4 = -0.625 * b * b * b + (5.0 / 12.0) * b * c + b / 24.0;
  }
  // Halley's error after a step of size s is ~K s^3, K <= (e/(1-e))^2/4 + e/(6(1-e)), and the
  // accepted step is applied to (sin, cos - 1) to second order (error s^3/6): with
  // s <= 2e-5 (1-e) both are below 2e-15 (fp64); fp32 works to 1e-3 (1-e) -> 4e-10.
  po.tol = (fp32 ? 1e-3 : 2e-5) * (1.0 - e);
  // sky position from (cm, s) = (cos d - 1, sin d):  sin E - sin E_tr = sE cm + cE s,
  // cos E - cos E_tr = cE cm - sE s;  x/a = cw dC - beta sw dS,  y/a = rho_tr + beta cw dS + sw dC
  const double bsw = beta * sw, bcw = beta * cw;
  po.X1 = a * (cw * cE - bsw * sE);
  po.X2 = -a * (cw * sE + bsw * cE);
  po.Y0 = (1.0 - e) * (1.0 + e) / den;           // r(t0)/a
  po.Y1 = bcw * sE + sw * cE;
  po.Y2 = bcw * cE - sw * sE;
  // Transit window.  z^2 = r^2 (c2 sin^2 i + cos^2 i), c2 = cos^2(w+f), so z < 1+k needs
  //   c2 < q2 = ((1+k)^2 / r^2 - cos^2 i) / sin^2 i   with any lower bound r_lo of r on the window,
  // i.e. w+f within h = asin(sqrt(q2)) of pi/2 (in front of the star); q2 <= 0: no transit at
  // all.  r_lo starts at a(1-e) and is raised to the minimum of r over the window found so far
  // (the in-transit set stays inside every window of the sequence, by induction), which matters
  // for eccentric orbits that transit far from periastron: up to (1+e)/(1-e) narrower.
  double u_lo = -0.5, u_hi = 0.5;
  if (!st) {
    const double ci2 = ci * ci, om = 1.0 - ci2;
    const double ftr = 0.5 * RR_PI - w;            // true anomaly at inferior conjunction
    double r_lo = a * (1.0 - e), h = 0.0;
    bool full = false;
    for (int it = 0; it < 4; ++it) {
      const double Q = (1.0 + kmax) / r_lo, Q2 = Q * Q;
      const double q2 = om > 1e-12 ? (Q2 - ci2) / om : (Q2 > ci2 ? 2.0 : -1.0);
      if (q2 >= 0.999998) { full = true; break; }
      h = q2 > 0.0 ? asin(sqrt(q2)) : 0.0;
      if (po.circular) break;
      const double fa = ftr - h, fb = ftr + h;     // r is smallest where cos f is largest
      double cosmax = fmax(cos(fa), cos(fb));
      if (ceil(fa / RR_TWOPI) <= floor(fb / RR_TWOPI)) cosmax = 1.0;   // periastron inside
      const double rn = a * (1.0 - e) * (1.0 + e) / (1.0 + e * cosmax);
      if (!(rn > r_lo * (1.0 + 1e-9))) break;
      r_lo = rn;
    }
    if (!full) {
      if (po.circular) {
        u_hi = h / RR_TWOPI;
        u_lo = -u_hi;
      } else {
        double sq1 = sqrt(1.0 - e), sq2 = sqrt(1.0 + e);
        double Etr = 2.0 * atan2(sq1 * sin(0.5 * ftr), sq2 * cos(0.5 * ftr));
        double fh = ftr + h, fl = ftr - h;
        double Eh = 2.0 * atan2(sq1 * sin(0.5 * fh), sq2 * cos(0.5 * fh));
        double El = 2.0 * atan2(sq1 * sin(0.5 * fl), sq2 * cos(0.5 * fl));
        double dEh = Eh - Etr, dEl = El - Etr;
        dEh -= RR_TWOPI * floor(dEh / RR_TWOPI);   // [0, 2pi)
        dEl -= RR_TWOPI * ceil(dEl / RR_TWOPI);    // (-2pi, 0]
        double dMh = dEh - e * (sin(Etr + dEh) - sin(Etr));
        double dMl = dEl - e * (sin(Etr + dEl) - sin(Etr));
        u_hi = dMh / RR_TWOPI;
        u_lo = dMl / RR_TWOPI;
      }
      u_hi = u_hi * (1.0 + 1e-9) + 1e-9;
      u_lo = u_lo * (1.0 + 1e-9) - 1e-9;
      if (!(u_hi - u_lo < 0.999) || !(u_hi > 0.0) || !(u_lo < 0.0)) { u_lo = -0.5; u_hi = 0.5; }
    }
  }
  po.u_mid = 0.5 * (u_lo + u_hi);
  po.hwid = 0.5 * (u_hi - u_lo);
  po.zpoly_ok = 0;
  po.pad = 0;
  pvo[v] = po;
}

// ---- lens area between the contacts as two polynomials per (pv, radius ratio) -------------------------
// For x = (z - (1-k)) / (2k) in (0, 1):  a(z) = pi k^2 - x^(3/2) g0(x) for x <= 1/2 and
// a(z) = y^(3/2) g1(y), y = 1 - x, for x > 1/2, with g0, g1 analytic (the area is analytic in the angle
// theta, x = sin^2(theta/2)): degree-12 interpolants at the Chebyshev nodes of [0, 1/2] reproduce the
// area to 2e-13 for k <= 0.32 (tests/test_device_poly.py).  One warp per (pv, k) (rr_poly_fit_kernel): lanes 0..12 and
// 13..25 evaluate the exact area (two sectors minus the kite, reading R9) at the nodes of the two
// halves; the node values become monomial coefficients in w = 4x - 1 through the matrix RR_LENS_M.
// The flux kernel then pays one square root and a Horner chain per ingress / egress sub-sample
// instead of a square root, two divisions and two arctangents (60 -> 23 FP64 instructions).
__device__ __forceinline__ void rr_lens_fit(const RRPvBand *__restrict__ pvb, int64_t row, int lane,
                                            double *__restrict__ lens) {
  const RRPvBand b = pvb[row];
  if (!b.lens_ok) return;                         // the flux kernel takes the exact form
  const int half = lane >= RR_LENS_N ? 1 : 0, i = lane - half * RR_LENS_N;
  double g = 0.0;
  if (lane < 2 * RR_LENS_N) {
    const double k = b.k, x = RR_LENS_X[i];
    const double omks = 1.0 - k, opk = 1.0 + k;
    const double z = half ? opk - 2.0 * k * x : omks + 2.0 * k * x;
    const double A = opk - z, B = z + omks, C = z - omks, D = z + opk;
    const double AB = fabs(A * B), S = fabs(C * D), Q = B * D;
    const double kite = rr_sqrt3_pos(AB * S);
    const double h1 = rr_atan_quadrant<double>(kite, Q, fabs(A * C));
    const double h2 = rr_atan_quadrant<double>(kite, S, AB);
    const double ap = fma(h1, 2.0, fma(2.0 * b.k2, h2, -0.5 * kite));
    g = (half ? ap : b.afull - ap) * RR_LENS_XI15[i];
  }
  // coefficient j of this lane's half: sum_i M[j][i] g_i
  double a = 0.0;
#pragma unroll
  for (int q = 0; q < RR_LENS_N; ++q) {
    const double gq = __shfl_sync(0xffffffffu, g, half * RR_LENS_N + q);
    if (lane < 2 * RR_LENS_N) a = fma(RR_LENS_M[i * RR_LENS_N + q], gq, a);
  }
  double *out = lens + (row * 2 + half) * RR_LENS_PITCH;
  if (lane < 2 * RR_LENS_N) out[i] = a;
  if (lane >= 2 * RR_LENS_N && lane < 2 * RR_LENS_N + 2) lens[(row * 2 + (lane - 2 * RR_LENS_N)) * RR_LENS_PITCH + RR_LENS_N] = 0.0;
}

// ---- per-(tile, pv) constants, staged in shared memory (8-byte slots: a double, or the float twice) ----
// Read with volatile loads at the point of use: they are warp-uniform broadcasts that ride in the
// issue slots the half-rate FP64 pipe leaves free, and keeping ~25 of them out of registers is what
// lets 8 blocks of 128 threads share an SM.  The loads name the dynamic shared array by its PTX
// symbol (rr_dyn, declared at global scope so that the name is not mangled) with an immediate
// offset: ptxas then addresses them off the shared-window base it keeps in a UNIFORM register
// (LDS [UR+imm]); round 1 passed the address in a vector register, which ptxas rematerialised
// with S2R/LEA at every use (5 instructions per sub-sample).
enum {
  K_ZC0, K_ZC1,           // circular (pair)
  K_CD, K_SD,             // circular: cos, sin of the phase step between sub-samples (pair)
  K_C4, K_C3,             // starter (pair)
  K_C2, K_KY,             // (pair)
  K_B, K_C,               // (pair)
  K_A, K_TOL,             // (pair)
  K_X1, K_X2,             // (pair)
  K_Y1, K_Y2,             // (pair)
  K_Y0, K_ACI2,           // (pair)
  K_E, K_SE,              // robust solver path (pair)
  K_CE, K_OPK2,           // (1+k)^2
  K_OMK2, K_AFULL,        // (1-k)^2, pi min(1,k)^2 (pair)
  K_GSCALE, K_OPK,        // (ng-1)/(1+kw), 1+k (pair)
  K_OMKS, K_K2,           // 1-k (signed), k^2 (pair)
  K_2K2, K_SCALE,         // 2 k^2, 1/(Istar ns) (pair)
  K_INV2K, K_XOFF,        // x = z K_INV2K + K_XOFF = (z - (1-k)) / (2k): lens polynomials (pair)
  K_LENSOK, K_ZOK,        // != 0: the staged lens polynomials hold for this k / the z^2 polynomials for this pv
  K_INVHW, K_PAD2,        // 1 / hwid
  K_TOTAL,
  K_COUNT = K_SCALE,      // entries rr_stage_constants writes
  K_SMEM = (K_TOTAL + 3) & ~3   // 16-byte multiple in both precisions
};
static_assert(K_CD % 2 == 0 && K_C4 % 2 == 0 && K_E % 2 == 0 && K_OMK2 % 2 == 0 && K_INV2K % 2 == 0 &&
              K_GSCALE % 2 == 0 && K_OMKS % 2 == 0 && K_2K2 % 2 == 0, "pairs");
template <typename T> struct Vec2T;
template <> struct Vec2T<double> { using type = double2; };
template <> struct Vec2T<float> { using type = float2; };

// Shared memory of the flux and orbit kernels (all dynamic, the kernels have no static shared
// memory): cst[K_SMEM] (8-byte slots) | tile flags (16 B) | ldw2[ldw_len] (node, slope) pairs.
// How the loads are addressed (template parameter M of Cst):
//   RR_SM_SYMBOL  by the PTX symbol rr_dyn + immediate: ptxas derives the shared-window base where it
//                 needs it (S2UR + ULEA, or S2R + LEA inside loops: 3-5 instructions per use site)
//   RR_SM_HELD    off a base address held in one register, made opaque to ptxas by a warp shuffle
//                 so that it is neither rematerialised nor copy-propagated away (costs a register)
//   RR_SM_ABS     absolute shared::cta addresses RR_SMEM_ABS + offset as immediates: one LDS per load,
//                 no address arithmetic, no register.  rr_dyn starts at the bytes the runtime reserves
//                 (cudaDevAttrReservedSharedMemoryPerBlock = 1024 on sm_100) because these kernels
//                 have no static shared memory; rr_create verifies that with a probe kernel (and
//                 falls back to RR_SM_SYMBOL otherwise), and every block re-checks and traps.
// Measured (config 4, flux kernel): fp64 symbol 5.75 ms, held 6.07 ms (the 64-register budget is full:
// the held register spills); fp32 symbol 3.93 ms, held 3.83 ms.
enum { RR_SM_SYMBOL = 0, RR_SM_HELD = 1, RR_SM_ABS = 2 };
#define RR_SMEM_ABS 1024
#ifndef RR_SM_FALLBACK_F64
#define RR_SM_FALLBACK_F64 RR_SM_SYMBOL
#endif
#ifndef RR_SM_FALLBACK_F32
#define RR_SM_FALLBACK_F32 RR_SM_HELD
#endif
// Every constant has an 8-byte slot in both precisions: a double, or - fp32 kernels - the float twice,
// so that one 8-byte load gives the packed (c, c) operand of the two-exposures-per-thread FFMA2 path
// and the scalar fp32 paths read its first half.
template <typename R, int M> struct Cst {
  static constexpr int ES = (int)sizeof(R);
  static constexpr int CS = 8;                       // bytes per constant slot
  static constexpr int OFF_FLAGS = K_SMEM * CS, OFF_LENS = OFF_FLAGS + 16,
                       OFF_ZPOLY = OFF_LENS + 2 * RR_LENS_PITCH * 8,    // lens polynomials: 2 x 14 doubles
                       OFF_ROW = OFF_ZPOLY + 2 * RR_LENS_PITCH * 8;    // z^2 polynomials: 2 x 14 doubles
  static constexpr int AB = (M == RR_SM_ABS ? RR_SMEM_ABS : 0);
  unsigned sb;   // RR_SM_HELD: shared-window address of rr_dyn; RR_SM_ABS: 0
  __device__ __forceinline__ Cst() {
    if constexpr (M == RR_SM_HELD) {
      sb = __shfl_sync(0xffffffffu, (unsigned)__cvta_generic_to_shared(rr_dyn), 0);
    } else {
      sb = 0;
      if constexpr (M == RR_SM_ABS)
        if ((unsigned)__cvta_generic_to_shared(rr_dyn) != RR_SMEM_ABS) __trap();
    }
  }
  static __device__ __forceinline__ void store(int slot, double v) {
    if constexpr (ES == 8) reinterpret_cast<double *>(rr_dyn)[slot] = v;
    else reinterpret_cast<float2 *>(rr_dyn)[slot] = make_float2((float)v, (float)v);
  }
  static __device__ __forceinline__ unsigned *flags() {
    return reinterpret_cast<unsigned *>(rr_dyn + OFF_FLAGS);
  }
  template <int I> __device__ __forceinline__ R get() const {
    R v;
    if constexpr (M == RR_SM_SYMBOL) {
      if constexpr (ES == 8)
        asm volatile("ld.volatile.shared.f64 %0, [rr_dyn+%1];" : "=d"(v) : "n"(CS * I));
      else
        asm volatile("ld.volatile.shared.f32 %0, [rr_dyn+%1];" : "=f"(v) : "n"(CS * I));
    } else {
      if constexpr (ES == 8)
        asm volatile("ld.volatile.shared.f64 %0, [%1+%2];" : "=d"(v) : "r"(sb), "n"(AB + CS * I));
      else
        asm volatile("ld.volatile.shared.f32 %0, [%1+%2];" : "=f"(v) : "r"(sb), "n"(AB + CS * I));
    }
    return v;
  }
  // two neighbouring constants (I even) with one 16-byte shared load
  template <int I> __device__ __forceinline__ void pair(double &a, double &b) const {
    static_assert(I % 2 == 0, "pair");
    if constexpr (M == RR_SM_SYMBOL)
      asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [rr_dyn+%2];" : "=d"(a), "=d"(b) : "n"(CS * I));
    else
      asm volatile("ld.volatile.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(a), "=d"(b)
                   : "r"(sb), "n"(AB + CS * I));
  }
  // fp32: the same load, as packed pairs (c, c) ...
  template <int I> __device__ __forceinline__ void pair2(float2 &a, float2 &b) const {
    static_assert(I % 2 == 0, "pair");
    unsigned long long u, w;
    if constexpr (M == RR_SM_SYMBOL)
      asm volatile("ld.volatile.shared.v2.b64 {%0, %1}, [rr_dyn+%2];" : "=l"(u), "=l"(w) : "n"(CS * I));
    else
      asm volatile("ld.volatile.shared.v2.b64 {%0, %1}, [%2+%3];" : "=l"(u), "=l"(w)
                   : "r"(sb), "n"(AB + CS * I));
    a = make_float2(__uint_as_float((unsigned)u), __uint_as_float((unsigned)(u >> 32)));
    b = make_float2(__uint_as_float((unsigned)w), __uint_as_float((unsigned)(w >> 32)));
  }
  template <int I> __device__ __forceinline__ float2 get2() const {
    unsigned long long u;
    if constexpr (M == RR_SM_SYMBOL)
      asm volatile("ld.volatile.shared.b64 %0, [rr_dyn+%1];" : "=l"(u) : "n"(CS * I));
    else
      asm volatile("ld.volatile.shared.b64 %0, [%1+%2];" : "=l"(u) : "r"(sb), "n"(AB + CS * I));
    return make_float2(__uint_as_float((unsigned)u), __uint_as_float((unsigned)(u >> 32)));
  }
  // ... or as scalars (first halves)
  template <int I> __device__ __forceinline__ void pair(float &a, float &b) const {
    float2 x, y;
    pair2<I>(x, y);
    a = x.x;
    b = y.x;
  }
  // coefficients 2m, 2m+1 of the lens polynomial of the half at byte offset hoff (0 or 8 PITCH)
  static __device__ __forceinline__ double *lens() { return reinterpret_cast<double *>(rr_dyn + OFF_LENS); }
  template <int MM, int OFF = OFF_LENS>
  __device__ __forceinline__ void lens2(unsigned hoff, double &a, double &b) const {
    if constexpr (M == RR_SM_SYMBOL) {
      const double2 v = reinterpret_cast<const double2 *>(rr_dyn + OFF + hoff)[MM];
      a = v.x;
      b = v.y;
    } else {
      asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(a), "=d"(b)
                   : "r"(sb + hoff), "n"(AB + OFF + 16 * MM));
    }
  }
  static __device__ __forceinline__ double *zpoly() { return reinterpret_cast<double *>(rr_dyn + OFF_ZPOLY); }
  // degree-12 polynomial of the half at byte offset hoff of the region OFF (lens or z^2), at w
  template <int OFF> __device__ __forceinline__ double poly12(unsigned hoff, double w) const {
    double c0, c1, p;
    lens2<6, OFF>(hoff, p, c1);               // c12 (c13 = 0)
    lens2<5, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    lens2<4, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    lens2<3, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    lens2<2, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    lens2<1, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    lens2<0, OFF>(hoff, c0, c1); p = fma(p, w, c1); p = fma(p, w, c0);
    return p;
  }
  // fp32 kernels: the same polynomial from coefficients staged as floats (16 per half, hoff 0 or 64)
  template <int MM, int OFF> __device__ __forceinline__ float4 coef4f(unsigned hoff) const {
    float4 v;
    if constexpr (M == RR_SM_SYMBOL) {
      v = reinterpret_cast<const float4 *>(rr_dyn + OFF + hoff)[MM];
    } else {
      asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4+%5];"
                   : "=f"(v.x), "=f"(v.y), "=f"(v.z), "=f"(v.w)
                   : "r"(sb + hoff), "n"(AB + OFF + 16 * MM));
    }
    return v;
  }
  template <int OFF> __device__ __forceinline__ float poly12f(unsigned hoff, float w) const {
    const float4 c3 = coef4f<3, OFF>(hoff), c2 = coef4f<2, OFF>(hoff), c1 = coef4f<1, OFF>(hoff),
                 c0 = coef4f<0, OFF>(hoff);
    float p = c3.x;                                  // c12
    p = fmaf(p, w, c2.w); p = fmaf(p, w, c2.z); p = fmaf(p, w, c2.y); p = fmaf(p, w, c2.x);
    p = fmaf(p, w, c1.w); p = fmaf(p, w, c1.z); p = fmaf(p, w, c1.y); p = fmaf(p, w, c1.x);
    p = fmaf(p, w, c0.w); p = fmaf(p, w, c0.z); p = fmaf(p, w, c0.y); p = fmaf(p, w, c0.x);
    return p;
  }
  // table cell ig of the staged row: node ldw[ig] and slope ldw[ig+1] - ldw[ig], one load
  using R2 = typename Vec2T<R>::type;
  static __device__ __forceinline__ R2 *row() { return reinterpret_cast<R2 *>(rr_dyn + OFF_ROW); }
  __device__ __forceinline__ void cell(int ig, R &l0, R &sl) const {
    if constexpr (M == RR_SM_SYMBOL) {
      const R2 v = row()[ig];
      l0 = v.x;
      sl = v.y;
    } else {
      const unsigned a = sb + (unsigned)(2 * ES) * (unsigned)ig;
      constexpr int off = AB + OFF_ROW;
      if constexpr (ES == 8)
        asm volatile("ld.shared.v2.f64 {%0, %1}, [%2+%3];" : "=d"(l0), "=d"(sl) : "r"(a), "n"(off));
      else
        asm volatile("ld.shared.v2.f32 {%0, %1}, [%2+%3];" : "=f"(l0), "=f"(sl) : "r"(a), "n"(off));
    }
  }
};

// rr_create's probe: the shared::cta address of rr_dyn in a kernel without static shared memory
__global__ void rr_smem_probe_kernel(unsigned *out) {
  if (threadIdx.x == 0) out[0] = (unsigned)__cvta_generic_to_shared(rr_dyn);
}

template <typename R>
__device__ __forceinline__ void rr_stage_constants(const RRPvOrbit &o, const RRPvBand &b, double du,
                                                   bool lens_on = false, bool zpoly_on = false) {
  const int t = threadIdx.x;
  double v = 0.0;
  switch (t) {
    // (library calls on two lanes: a polynomial here changed the register allocation of the whole
    // kernel and cost the sparse cadence 4b 10 %)
    case K_CD: v = cospi(2.0 * du); break;   case K_SD: v = sinpi(2.0 * du); break;
    case K_ZC0: v = o.zc0 + (sizeof(R) == 8 ? RR_TINY_D : 1e-30); break;   // z^2 > 0
    case K_ZC1: v = o.zc1; break;
    case K_E: v = o.e; break;           case K_SE: v = o.sE; break;
    case K_CE: v = o.cE; break;         case K_A: v = o.A; break;
    case K_B: v = o.B; break;           case K_C: v = o.C; break;
    case K_KY: v = RR_TWOPI * o.invA; break;
    case K_C2: v = o.c2; break;         case K_C3: v = o.c3; break;
    case K_C4: v = o.c4; break;         case K_TOL: v = o.tol; break;
    case K_X1: v = o.X1; break;         case K_X2: v = o.X2; break;
    case K_Y0: v = o.Y0; break;         case K_Y1: v = o.Y1; break;
    case K_Y2: v = o.Y2; break;         case K_ACI2: v = o.aci2; break;
    case K_OPK: v = b.opk; break;       case K_OPK2: v = b.opk * b.opk; break;
    case K_OMKS: v = 1.0 - b.k; break;  case K_AFULL: v = b.afull; break;
    case K_K2: v = b.k2; break;         case K_GSCALE: v = b.gscale; break;
    case K_OMK2: v = b.omk * b.omk; break;
    case K_2K2: v = 2.0 * b.k2; break;
    case K_INV2K: v = 0.5 / b.k; break;  case K_XOFF: v = -(1.0 - b.k) * (0.5 / b.k); break;
    case K_LENSOK: v = lens_on ? 1.0 : 0.0; break;
    case K_ZOK: v = zpoly_on ? 1.0 : 0.0; break;
    case K_INVHW: v = 1.0 / o.hwid; break;
    default: break;
  }
  if (t < K_COUNT || (t >= K_INV2K && t <= K_INVHW)) Cst<R, RR_SM_SYMBOL>::store(t, v);
}

// ---- kernel 2, robust path: bracketed Halley / bisection for G(d) = 0, any dM ------------------------
// Stores (sin d, cos d - 1) of the root; returns the number of sincos evaluations.
template <typename R>
__device__ RR_ROBUST_INLINE int rr_kepler_robust(R e, R sE, R cE, R dM, R *s_out, R *cm1_out) {
  // root bracketed by E in [M - e, M + e]  <=>  d in [dM - e sE - e, dM - e sE + e]
  const R mid = fma(-e, sE, dM);
  R lo = mid - e, hi = mid + e;
  R d = dM / fma(-e, cE, (R)1);
  d = fmin(fmax(d, lo), hi);
  // Halley steps converge cubically: the error after a step of size s is ~K s^3 with
  // K <= (e/(1-e))^2/4 + e/(6(1-e)); stop when that is below the working epsilon.
  const R tol = (sizeof(R) == 8 ? (R)3e-6 : (R)1e-3) * ((R)1 - e);
  R sh, ch, s = (R)0, c = (R)1, cm1 = (R)0, dd = (R)0;
  int it = 0;
  for (; it < 60; ++it) {
    rr_sincos((R)0.5 * d, &sh, &ch);
    s = (R)2 * sh * ch;
    cm1 = (R)-2 * sh * sh;
    c = (R)1 + cm1;
    R g = (d - dM) - e * fma(sE, cm1, cE * s);
    R gp = (R)1 - e * fma(cE, c, -sE * s);       // 1 - e cos E
    R gpp = e * fma(sE, c, cE * s);              // e sin E
    if (g > (R)0) hi = d; else lo = d;
    R dn = d - ((R)2 * g * gp) / fma((R)2 * gp, gp, -g * gpp);   // Halley
    if (!(dn >= lo && dn <= hi)) dn = (R)0.5 * (lo + hi);        // left the bracket: bisect
    dd = dn - d;
    d = dn;
    if (fabs(dd) <= tol) { ++it; break; }
  }
  // rotate (sin, cos - 1) of the last evaluated d by the last small step dd, to second order
  const R hdd2 = (R)0.5 * dd * dd;
  *s_out = s + c * dd - s * hdd2;
  *cm1_out = cm1 - s * dd - c * hdd2;
  return it;
}

// ---- z^2 over the transit window as two polynomials per parameter vector (fp64 kernel) ---------------
// For an eccentric orbit with a transit window [u_mid - hwid, u_mid + hwid] the squared separation is
// an analytic function of the phase; on each half of the window, t' = |w| / hwid in [0, 1], it is
// interpolated by a degree-12 polynomial at the Chebyshev nodes (the tables of the lens polynomials:
// nodes 2 RR_LENS_X, matrix RR_LENS_M).  One warp per parameter vector: lanes 0..12 / 13..25 solve
// Kepler's equation exactly (bracketed Halley) at the nodes of the two halves.
// The polynomials are used only if their Chebyshev tails |c12| + |c11| are below RR_ZPOLY_TAIL
// (wide windows of close-in, very eccentric orbits do not converge: those pvs keep the per-sub-sample
// solve).  Per sub-sample the flux kernel then pays 15 FP64 instructions instead of 53.
#ifndef RR_ZPOLY_TAIL
#define RR_ZPOLY_TAIL 1e-12
#endif
__device__ __forceinline__ void rr_zpoly_fit(RRPvOrbit *__restrict__ pvo, int64_t v, int lane,
                                             double *__restrict__ zpoly) {
  const RRPvOrbit po = pvo[v];
  if (po.status || po.circular || !(po.hwid < 0.49)) return;     // (zpoly_ok stays 0)
  const int half = lane >= RR_LENS_N ? 1 : 0, i = lane - half * RR_LENS_N;
  double g = 0.0;
  if (lane < 2 * RR_LENS_N) {
    const double w = (half ? 2.0 : -2.0) * RR_LENS_X[i] * po.hwid;  // phase from the window centre
    const double dM = RR_TWOPI * (w + po.u_mid);
    double s, cm1;
    rr_kepler_robust<double>(po.e, po.sE, po.cE, dM, &s, &cm1);
    const double xs = fma(po.X1, cm1, po.X2 * s);
    const double ys = po.Y0 + fma(po.Y1, cm1, po.Y2 * s);
    g = fma(xs, xs, po.aci2 * ys * ys);
  }
  double a = 0.0;
#pragma unroll
  for (int q = 0; q < RR_LENS_N; ++q) {
    const double gq = __shfl_sync(0xffffffffu, g, half * RR_LENS_N + q);
    if (lane < 2 * RR_LENS_N) a = fma(RR_LENS_M[i * RR_LENS_N + q], gq, a);
  }
  // Chebyshev tail from the two leading monomial coefficients: c12 = a12 / 2^11, c11 = a11 / 2^10
  double tail = 0.0;
  if (lane < 2 * RR_LENS_N && i == RR_LENS_N - 1) tail = fabs(a) * (1.0 / 2048.0);
  if (lane < 2 * RR_LENS_N && i == RR_LENS_N - 2) tail = fabs(a) * (1.0 / 1024.0);
  if (!(a == a) || fabs(a) > 1e300) tail = 1.0;                   // not finite: no polynomial
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) tail += __shfl_xor_sync(0xffffffffu, tail, o);
  double *out = zpoly + (v * 2 + half) * RR_LENS_PITCH;
  if (lane < 2 * RR_LENS_N) out[i] = a;
  if (lane >= 2 * RR_LENS_N && lane < 2 * RR_LENS_N + 2)
    zpoly[(v * 2 + (lane - 2 * RR_LENS_N)) * RR_LENS_PITCH + RR_LENS_N] = 0.0;
  if (lane == 0 && tail <= RR_ZPOLY_TAIL) pvo[v].zpoly_ok = 1;
}

// One launch for both fits: warps [0, nrows) take the lens polynomials of the (pv, k) rows, warps
// [nrows, nrows + npv) the z^2 polynomials of the parameter vectors (either part may be absent).
__global__ void rr_poly_fit_kernel(const RRPvBand *__restrict__ pvb, int64_t nrows,
                                   double *__restrict__ lens, RRPvOrbit *__restrict__ pvo, int64_t npv,
                                   double *__restrict__ zpoly) {
  const int64_t w = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  const int64_t nl = lens ? nrows : 0;
  if (w < nl) rr_lens_fit(pvb, w, lane, lens);
  else if (zpoly && w - nl < npv) rr_zpoly_fit(pvo, w - nl, lane, zpoly);
}

// ---- kernel 2 core: squared separation at reduced phase ur (turns, relative to t0) ----------------------
// Returns z^2; front = planet between observer and star.  iters counts sincos evaluations.
template <typename R, bool CIRC, int M>
__device__ __forceinline__ R rr_separation2(const Cst<R, M> K, double ur, bool &front, int &iters) {
  if (CIRC) {
    // e = 0: z^2 = a^2 (sin^2 phi + cos^2 phi cos^2 i) = a^2 cos^2 i + a^2 sin^2 i sin^2 phi
    R s;
    if (fabs(ur) <= 0.07949995994567871) {             // 0x3FB45A1C'00000000: 2 pi u <= 0.4995
      R cm1;
      rr_sincosm1_small((R)(RR_TWOPI * ur), s, cm1);
    } else {
      s = rr_sinpi((R)(2.0 * ur));
    }
    front = fabs(ur) < 0.25;
    R zc0, zc1;
    K.template pair<K_ZC0>(zc0, zc1);
    return fma(s * s, zc1, zc0);
  }
  R s2, cm2;
  bool done = false;
  R dM;
  {
    R c4, c3, c2, ky, B, C, A, tol;
    K.template pair<K_C4>(c4, c3);
    K.template pair<K_C2>(c2, ky);
    const R y = (R)ur * ky;                            // dM / A
    R d = y * fma(y, fma(y, fma(y, c4, c3), c2), (R)1);
    K.template pair<K_B>(B, C);
    K.template pair<K_A>(A, tol);
    // 2 pi ur: fp64 takes it from y (one FP64 instruction, no 64-bit constant); fp32 rounds the
    // fp64 product once (y A would add two fp32 roundings to the Kepler residual)
    dM = sizeof(R) == 8 ? y * A : (R)(RR_TWOPI * ur);
    // Halley steps from the series starter while d stays in the polynomial range; the first one
    // is accepted for ~94 % of config 4's eccentric sub-samples
#pragma unroll 1
    for (int it = 0; it < 3 && fabs(d) <= (R)RR_TRIG_SMALL; ++it) {
      R s, cm1, t, g;
      if constexpr (sizeof(R) == 8) {
        rr_sincosm1_small(d, s, cm1);
        t = fma(B, cm1, C * s);                    // e [sin E - sin E_tr]
        g = (d - dM) - t;
      } else {
        // fp32: d - t = A d - C (sin d - d) - B (cos d - 1), A = 1 - e cos E_tr rounded once from
        // fp64.  Formed this way the residual carries eps |dM| instead of eps |d| ~ eps |dM| / A
        // (the direct form loses 1/(1 - e) near a periastron transit: 4e-7 in flux at e = 0.99).
        R sres;
        rr_sincosm1_small(d, s, cm1, sres);
        const R bc = B * cm1;
        t = fma(C, s, bc);
        g = fma(A, d, -dM) - fma(C, sres, bc);
      }
      const R gp = A - fma(C, cm1, -B * s);        // 1 - e cos E
      const R gpp = B + t;                         // e sin E
      // Halley: -2 g g' / (2 g'^2 - g g'') = -(g g') / (g'^2 - g g''/2)
      const R dd = -(g * gp) * rr_rcp(fma((R)-0.5 * g, gpp, gp * gp));
      iters += 1;
      if (fabs(dd) <= tol) {
        // (sin, cos - 1) of d + dd, second order in dd
        const R c = (R)1 + cm1;
        const R h2 = (R)0.5 * dd * dd;
        s2 = fma(-s, h2, fma(c, dd, s));
        cm2 = fma(-c, h2, fma(-s, dd, cm1));
        done = true;
        break;
      }
      d += dd;
    }
  }
  if (!done) {
    R e, sE;
    K.template pair<K_E>(e, sE);
    iters += rr_kepler_robust<R>(e, sE, K.template get<K_CE>(), (R)(RR_TWOPI * ur), &s2, &cm2);
  }
  R X1, X2, Y1, Y2, Y0, aci2;
  K.template pair<K_X1>(X1, X2);
  K.template pair<K_Y1>(Y1, Y2);
  K.template pair<K_Y0>(Y0, aci2);
  const R xs = fma(X1, cm2, X2 * s2);
  const R ys = Y0 + fma(Y1, cm2, Y2 * s2);
  front = ys > (R)0;
  const R tiny = sizeof(R) == 8 ? (R)RR_TINY_D : (R)1e-30f;       // z^2 > 0: the sqrt seed stays finite
  return fma(xs, xs, fma(aci2 * ys, ys, tiny));
}

// ---- kernel 3 core: occulted light ip * ap of one sub-sample with z < 1+k ------
// Table cell of y = g/dg in [0, ng-1]: lower node ig and weight ag = y - ig.  The staged row carries
// one extra cell (node ldw[ng-1], slope 0), so that y = ng-1 (z = 1+k to rounding) needs no clamp
// (reading R10: the same value as cell ng-2 with ag = 1).
__device__ __forceinline__ void rr_cell(double y, int &ig, double &ag) {
  ig = __double2int_rd(y);                   // conversion unit, not the FP64 pipe; the index and the
  ag = y - floor(y);                         // weight do not wait for each other
}
__device__ __forceinline__ void rr_cell(float y, int &ig, float &ag) {
  ig = (int)y;
  ag = y - (float)ig;
}

// kmode (block-uniform, decided once per tile): bit 0: k^2 <= 1/2; bit 1: the staged lens
// polynomials hold (fp64 kernel, k <= RR_LENS_KMAX).
template <typename R, int M>
__device__ __forceinline__ R rr_deficit(const Cst<R, M> K, R z2, int &ningress, int kmode) {
  const bool ksmall = (kmode & 1) != 0;
  // the constants first: their shared-memory latency passes under the square root
  R gscale, opk, omk2, afull;
  K.template pair<K_GSCALE>(gscale, opk);
  K.template pair<K_OMK2>(omk2, afull);
  const R z = rr_sqrt3(z2);                 // z2 > 0: both orbit branches add 2^-1000
  int ig;
  R ag;
  rr_cell(z * gscale, ig, ag);
  R l0, sl;
  K.cell(ig, l0, sl);                      // ldw[ig], ldw[ig+1] - ldw[ig]
  const R ip = fma(ag, sl, l0);             // mean occulted brightness
  R ap;
  if (z2 <= omk2) {
    ap = afull;                             // planet (or star) fully inside the other disc
  } else if (kmode & 2) {
    // Between the contacts, polynomial form (rr_lens_fit): x = (z - (1-k)) / (2k),
    //   a = pi k^2 - x^(3/2) g0(4x - 1)  for x <= 1/2,   a = y^(3/2) g1(4y - 1), y = 1 - x, else.
    if constexpr (sizeof(R) == 8) {
      double inv2k, xoff;
      K.template pair<K_INV2K>(inv2k, xoff);
      const double x = fma(z, inv2k, xoff);
      const bool lo = x <= 0.5;
      const double xx = fabs(lo ? x : 1.0 - x);
      const unsigned hoff = lo ? 0u : (unsigned)(RR_LENS_PITCH * 8);
      const double w = fma(xx, 4.0, -1.0);
      const double sq = rr_sqrt3_pos(xx);
      const double p = K.template poly12<Cst<R, M>::OFF_LENS>(hoff, w);
      const double t = xx * sq;
      ap = lo ? fma(-t, p, afull) : t * p;
    } else {
      float inv2k, xoff;
      K.template pair<K_INV2K>(inv2k, xoff);
      const float x = fmaf(z, inv2k, xoff);
      const bool lo = x <= 0.5f;
      const float xx = fabsf(lo ? x : 1.0f - x);
      const float p = K.template poly12f<Cst<R, M>::OFF_LENS>(lo ? 0u : 64u, fmaf(xx, 4.0f, -1.0f));
      const float t = xx * rr_sqrt_core(xx + 1e-30f);
      ap = fmaxf(lo ? fmaf(-t, p, afull) : t * p, 0.0f);
    }
    ++ningress;
  } else {
    // Lens of the unit disc and the disc of radius k at distance z (reading R9): two sectors minus
    // the kite.  With A = 1+k-z, B = z+1-k, C = z-1+k, D = z+1+k (all >= 0 here):
    //   kite = sqrt(A B C D) = 4 x area of the triangle (1, k, z),
    //   half-angle at the star's centre   th1/2 = atan(kite / (B D))   [tan^2 = A C / (B D)],
    //   half-angle at the planet's centre th2/2 = atan(kite / (C D))   [tan^2 = A B / (C D)],
    // the half-angle formulas of the triangle: both arguments are >= 0 (no sign cases), th1/2 <=
    // asin(k)/2 needs no octant reduction for k^2 <= 1/2 and th2/2 in [0, pi/2] needs one of three
    // cases.  ap = th1 + k^2 th2 - kite/2.
    const R omks = K.template get<K_OMKS>();
    const R A = opk - z, B = z + omks, C = z - omks, D = z + opk;
    const R AB = fabs(A * B), S = fabs(C * D), Q = B * D;
    const R kite = rr_sqrt3_pos(AB * S);
    const R tk2 = K.template get<K_2K2>();
    // (the k^2 > 1/2 case is a path of its own so that the common one is a single basic block:
    // the two arctangents are independent and interleave)
    if (ksmall) {                           // k^2 <= 1/2, decided once per tile
      const R h1 = rr_atan_t(rr_div3(kite, Q));
      const R h2 = rr_atan_quadrant<R>(kite, S, AB);
      ap = fma(h1, (R)2, fma(tk2, h2, (R)-0.5 * kite));
    } else {
      const R h1 = rr_atan_quadrant<R>(kite, Q, fabs(A * C));
      const R h2 = rr_atan_quadrant<R>(kite, S, AB);
      ap = fma(h1, (R)2, fma(tk2, h2, (R)-0.5 * kite));
    }
    // fp32: the three terms cancel at the first contact; keep ap >= 0 so that flux <= 1 (RR_MIXED
    // stores the sum in fp64, where a deficit of -1e-13 would show)
    if constexpr (sizeof(R) == 4) ap = fmaxf(ap, 0.0f);
    ++ningress;
  }
  return ip * ap;
}

struct FluxParams {
  const double *times;
  const RRTile *tiles;
  const RRLc *lcs;
  const RRPvOrbit *pvo;
  const RRPvBand *pvb;
  const void *T;        // full table (RR_TABLE_FULL) or NULL
  const void *rows;     // collapsed rows ldw[npv][npb][ng] (RR_TABLE_LAZY) or NULL
  const void *istar;
  const double *lens;   // lens-area polynomials [npv][nkpb][2][RR_LENS_PITCH] (fp64 kernel) or NULL
  const double *zpoly;  // z^2 polynomials [npv][2][RR_LENS_PITCH] (fp64 kernel) or NULL
  void *flux;
  unsigned long long *counters;
  int64_t npt, npv, ntiles;
  int npb, nkpb, nk, ng;
  int shuffle_min_ns;   // light curves with ns >= this use the lanes-over-sub-samples layout
  int ldw_len;          // staged row length: ng + 1, or more with mean-k weights, where g of a
                        // passband with k > kw passes the last node (reading R13): limb value
  unsigned ones_off;    // byte offset in rr_dyn of the block's buffer of ones (bulk fill)
  unsigned nchunks;     // blocks per parameter vector
  unsigned chunk_len;   // dispatch tiles per block
};

template <typename R> __device__ __forceinline__ R rr_nan();
template <> __device__ __forceinline__ double rr_nan<double>() { return __longlong_as_double(0x7ff8000000000000LL); }
template <> __device__ __forceinline__ float rr_nan<float>() { return __int_as_float(0x7fc00000); }

// Coalesced, 16-byte-vectorised constant fill of out[0..count).
template <typename R>
__device__ __forceinline__ void rr_fill(R *out, int64_t count, R val) {
  constexpr int VN = 16 / sizeof(R);
  uintptr_t addr = reinterpret_cast<uintptr_t>(out);
  int64_t head = (int64_t)(((16 - (addr & 15)) & 15) / sizeof(R));
  if (head > count) head = count;
  if ((int64_t)threadIdx.x < head) out[threadIdx.x] = val;
  const int64_t nvec = (count - head) / VN;
  if (sizeof(R) == 8) {
    double2 v = make_double2((double)val, (double)val);
    double2 *o = reinterpret_cast<double2 *>(out + head);
#pragma unroll 4
    for (int64_t i = threadIdx.x; i < nvec; i += FT) RR_STORE(o + i, v);
  } else {
    float4 v = make_float4((float)val, (float)val, (float)val, (float)val);
    float4 *o = reinterpret_cast<float4 *>(out + head);
#pragma unroll 4
    for (int64_t i = threadIdx.x; i < nvec; i += FT) RR_STORE(o + i, v);
  }
  const int64_t done = head + nvec * VN;
  if ((int64_t)threadIdx.x < count - done) out[done + threadIdx.x] = val;
}

// Out-of-window runs (flux = 1) written by the TMA engine: a block keeps RR_ONES_BYTES of ones in
// shared memory and ONE thread issues bulk copies shared -> global (cp.async.bulk, <= RR_ONES_BYTES
// each) for the 16-byte-aligned body of the run; head and tail elements go out as plain stores.  The
// other threads go straight on to the next in-window tile: the fill costs the SM one instruction per
// 8 kB instead of a 16-byte store per thread (config 4 writes 10.9 of its 13.1 GB this way).
#ifndef RR_ONES_BYTES
#define RR_ONES_BYTES 8192
#endif
#ifndef RR_BULK_FILL
#define RR_BULK_FILL 1
#endif
// Block-uniform call: writes the ones and makes them visible to the async proxy.
template <typename O>
__device__ __forceinline__ void rr_ones_setup(unsigned char *ones_p) {
  for (int i = threadIdx.x; i < RR_ONES_BYTES / (int)sizeof(O); i += FT)
    reinterpret_cast<O *>(ones_p)[i] = (O)1;
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
  __syncthreads();
}
template <typename O>
__device__ __forceinline__ void rr_fill_ones_bulk(O *out, int64_t count, unsigned ones_smem) {
  const uintptr_t addr = reinterpret_cast<uintptr_t>(out);
  int64_t head = (int64_t)(((16 - (addr & 15)) & 15) / sizeof(O));
  if (head > count) head = count;
  if ((int64_t)threadIdx.x < head) out[threadIdx.x] = (O)1;
  const int64_t body = ((count - head) * (int64_t)sizeof(O)) & ~(int64_t)15;      // bytes
  if (threadIdx.x == 0 && body > 0) {
    const char *dst = reinterpret_cast<const char *>(out + head);
    // flux is never re-read: evict-first in L2, so that W, the times and the rows stay (config 4
    // 0.8 %, config 4b 4 % faster than with the default policy)
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    for (int64_t off = 0; off < body; off += RR_ONES_BYTES) {
      const unsigned n = (unsigned)min((int64_t)RR_ONES_BYTES, body - off);
      asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
                   :: "l"(dst + off), "r"(ones_smem), "r"(n), "l"(pol) : "memory");
    }
    asm volatile("cp.async.bulk.commit_group;" ::: "memory");
  }
  const int64_t done = head + body / (int64_t)sizeof(O);
  if ((int64_t)threadIdx.x < count - done) out[done + threadIdx.x] = (O)1;
}

// Occulted light of the sub-sample at phase w (turns, measured from the window centre).
// cnt: 0 skipped, 1 circular, 2 eccentric, 3 occulting, 4 ingress, 5 sincos evaluations of the solver
template <typename R, bool COUNT, bool CIRC, bool NOWRAP, int M>
__device__ __forceinline__ R rr_subsample(const Cst<R, M> K, double w, double u_mid, double hwid,
                                          bool need_front, int kmode, unsigned long long *cnt) {
  // NOWRAP (block-uniform): hwid + 2 hw < 1/2, so |w| < 1/2 already and the reduction is a no-op
  const double wr = NOWRAP ? w : w - rr_round(w);
  R def = (R)0;
  if (fabs(wr) <= hwid) {
    bool front = true;
    int it = 0, ing = 0;
    R z2;
    if (!CIRC && (kmode & 4)) {
      // z^2 from the pv's polynomials over its transit window (rr_zpoly_fit): t' = |w| / hwid
      if constexpr (!CIRC && sizeof(R) == 8) {
        const double t = wr * K.template get<K_INVHW>();
        const unsigned hoff = t < 0.0 ? 0u : (unsigned)(RR_LENS_PITCH * 8);
        z2 = fabs(K.template poly12<Cst<R, M>::OFF_ZPOLY>(hoff, fma(fabs(t), 2.0, -1.0))) + RR_TINY_D;
      } else if constexpr (!CIRC) {
        const float t = (float)wr * K.template get<K_INVHW>();
        z2 = fabsf(K.template poly12f<Cst<R, M>::OFF_ZPOLY>(t < 0.0f ? 0u : 64u,
                                                             fmaf(fabsf(t), 2.0f, -1.0f))) + 1e-30f;
      }
      if (COUNT) cnt[6]++;
    } else {
      z2 = rr_separation2<R, CIRC, M>(K, wr + u_mid, front, it);
    }
    // inside a transit window (hwid < 1/2) the true anomaly is within a quarter turn of
    // conjunction: the planet is in front, and the test is only needed without a window
    bool occ = z2 < K.template get<K_OPK2>();
    if (need_front) occ = occ && front;
    if (occ) {
      def = rr_deficit<R, M>(K, z2, ing, kmode);
      if (COUNT) { cnt[3]++; cnt[4] += ing; }
    }
    if (COUNT) { cnt[CIRC ? 1 : 2]++; cnt[5] += it; }
  } else if (COUNT) {
    cnt[0]++;
  }
  return def;
}

// Mid-exposure time through the read-only path (global address space known, L1-cacheable: every pv
// block on the SM reads the same times).
__device__ __forceinline__ double rr_ld_time(uintptr_t p) {
#ifdef RR_TIME_GENERIC
  return *reinterpret_cast<const double *>(p);
#else
  double t;
  asm volatile("ld.global.nc.f64 %0, [%1];" : "=d"(t) : "l"(p));
  return t;
#endif
}

// ---- two exposures per thread ---------------------------------------------------------------------------
// fp32 / mixed kernels: packed FFMA2 arithmetic (one instruction, two exposures).  fp64 kernel
// (eccentric tiles; circular ones keep their rotation recurrence): two scalar instructions per
// operation, but one load of every constant and coefficient, one branch, one loop for the pair, and two
// independent dependency chains per warp.
// (ax, ay): the element is inside the transit window at this sub-sample.  An inactive element is
// given the phase 0, computes along and is masked out; nothing here can fault on its values.
#ifndef RR_FP32_PAIRS
#define RR_FP32_PAIRS 1
#endif
#ifndef RR_LENS_POLY
#define RR_LENS_POLY 1
#endif
#ifndef RR_ZPOLY
#define RR_ZPOLY 1
#endif
#ifndef RR_FP64_PAIRS
#define RR_FP64_PAIRS 0   // measured twice: with the direct formulation (80 registers, 6 blocks per SM)
                          // config 4 5.09 -> 5.56 ms, config 3 7.56 -> 9.04; with the polynomial paths
                          // 3.85 -> 4.22 ms at 6, 7 or 8 blocks per SM.  Kept as a build option.
#endif
// two neighbouring constants as pairs (c, c): fp32 from the doubled slots, fp64 splat in registers
template <int I, typename R, int M>
__device__ __forceinline__ void rr_pairP(const Cst<R, M> K, typename PairT<R>::type &a,
                                         typename PairT<R>::type &b) {
  if constexpr (sizeof(R) == 4) {
    K.template pair2<I>(a, b);
  } else {
    R x, y;
    K.template pair<I>(x, y);
    a = splat<R>(x);
    b = splat<R>(y);
  }
}
template <int I, typename R, int M>
__device__ __forceinline__ typename PairT<R>::type rr_getP(const Cst<R, M> K) {
  if constexpr (sizeof(R) == 4) return K.template get2<I>();
  else return splat<R>(K.template get<I>());
}

// degree-12 polynomial of the first (lo) or second half of the region OFF, in the working precision
template <int OFF, typename R, int M>
__device__ __forceinline__ R rr_polyR(const Cst<R, M> K, bool lo, R w) {
  if constexpr (sizeof(R) == 8) return K.template poly12<OFF>(lo ? 0u : (unsigned)(RR_LENS_PITCH * 8), w);
  else return K.template poly12f<OFF>(lo ? 0u : 64u, w);
}

// The phases come as dM = 2 pi ur in the working precision (rr_tile_pairs).
template <typename R, bool CIRC, int M>
__device__ __forceinline__ typename PairT<R>::type
rr_separation2_pair(const Cst<R, M> K, typename PairT<R>::type dM, bool ax, bool ay, bool &fx,
                    bool &fy) {
  using P = typename PairT<R>::type;
  if (CIRC) {
    P s;
    const P am = abs2(dM);
    if (am.x <= (R)0.4995 && am.y <= (R)0.4995) {
      P cm1, sres;
      rr_sincosm1_small2(dM, s, cm1, sres);
    } else {
      s = mk2((R)sin((double)dM.x), (R)sin((double)dM.y));
    }
    fx = am.x < (R)1.5707963;
    fy = am.y < (R)1.5707963;
    P zc0, zc1;
    rr_pairP<K_ZC0>(K, zc0, zc1);
    return fma2(mul2(s, s), zc1, zc0);
  }
  P s2 = splat<R>((R)0), cm2 = splat<R>((R)0);
  bool okx = !ax, oky = !ay;
  {
    P c4, c3, c2, ky, B, C, A, tol;
    rr_pairP<K_C4>(K, c4, c3);
    rr_pairP<K_C2>(K, c2, ky);
    const P y = mul2(dM, mul2(ky, splat<R>((R)0.15915494309189535)));   // dM / A (K_KY = 2 pi / A)
    P d = mul2(y, fma2(y, fma2(y, fma2(y, c4, c3), c2), splat<R>((R)1)));
    rr_pairP<K_B>(K, B, C);
    rr_pairP<K_A>(K, A, tol);
    // Halley steps for the pair until every active element has accepted its step (an element that
    // accepted earlier just takes one more, smaller, step)
#pragma unroll 1
    for (int it = 0; it < 3; ++it) {
      const P ad = abs2(d);
      if ((ax && !(ad.x <= (R)RR_TRIG_SMALL)) || (ay && !(ad.y <= (R)RR_TRIG_SMALL))) break;
      P s, cm1, sres;
      rr_sincosm1_small2(d, s, cm1, sres);
      const P bc = mul2(B, cm1);
      const P t = fma2(C, s, bc);                                           // e [sin E - sin E_tr]
      P g;
      if constexpr (sizeof(R) == 8) g = sub2(sub2(d, dM), t);
      else g = sub2(fma2(A, d, neg2(dM)), fma2(C, sres, bc));              // (rr_separation2, fp32)
      const P gp = sub2(A, fma2(C, cm1, neg2(mul2(B, s))));                 // 1 - e cos E
      const P gpp = add2(B, t);                                             // e sin E
      const P dd = mul2(neg2(mul2(g, gp)),
                        rcp2(fma2(mul2(splat<R>((R)-0.5), g), gpp, mul2(gp, gp))));
      const P c = add2(splat<R>((R)1), cm1);
      const P h2 = mul2(mul2(splat<R>((R)0.5), dd), dd);
      s2 = fma2(neg2(s), h2, fma2(c, dd, s));
      cm2 = fma2(neg2(c), h2, fma2(neg2(s), dd, cm1));
      const P add_ = abs2(dd);
      okx = !ax || add_.x <= tol.x;
      oky = !ay || add_.y <= tol.y;
      if (okx && oky) break;
      d = add2(d, dd);
    }
  }
  if (!(okx && oky)) {                           // |d| > 0.5 or no convergence: the bracketed solver
    R e, sE;
    K.template pair<K_E>(e, sE);
    const R cE = K.template get<K_CE>();
    if (!okx) rr_kepler_robust<R>(e, sE, cE, dM.x, &s2.x, &cm2.x);
    if (!oky) rr_kepler_robust<R>(e, sE, cE, dM.y, &s2.y, &cm2.y);
  }
  P X1, X2, Y1, Y2, Y0, aci2;
  rr_pairP<K_X1>(K, X1, X2);
  rr_pairP<K_Y1>(K, Y1, Y2);
  rr_pairP<K_Y0>(K, Y0, aci2);
  const P xs = fma2(X1, cm2, mul2(X2, s2));
  const P ys = add2(Y0, fma2(Y1, cm2, mul2(Y2, s2)));
  fx = ys.x > (R)0;
  fy = ys.y > (R)0;
  const R tiny = sizeof(R) == 8 ? (R)RR_TINY_D : (R)1e-30f;
  return fma2(xs, xs, fma2(mul2(aci2, ys), ys, splat<R>(tiny)));
}

// Occulted light ip * ap of the pair; (ox, oy): z < 1+k in front of the star.
template <typename R, int M>
__device__ __forceinline__ typename PairT<R>::type
rr_deficit_pair(const Cst<R, M> K, typename PairT<R>::type z2, bool ox, bool oy, int kmode) {
  using P = typename PairT<R>::type;
  const bool ksmall = (kmode & 1) != 0;
  P gscale, opk, omk2, afull;
  rr_pairP<K_GSCALE>(K, gscale, opk);
  rr_pairP<K_OMK2>(K, omk2, afull);
  z2 = sel2(ox, oy, z2, splat<R>((R)0.25));     // a masked element stays inside the staged row
  const P z = rr_sqrt2(z2);
  const P yv = mul2(z, gscale);
  int igx, igy;
  P ag;
  rr_cell(yv.x, igx, ag.x);
  rr_cell(yv.y, igy, ag.y);
  R l0x, slx, l0y, sly;
  K.cell(igx, l0x, slx);
  K.cell(igy, l0y, sly);
  const P ip = fma2(ag, mk2(slx, sly), mk2(l0x, l0y));
  const bool inx = ox && z2.x > omk2.x, iny = oy && z2.y > omk2.y;
  P ap = afull;
  if ((inx || iny) && (kmode & 2)) {
    // lens polynomials (rr_deficit): each element with the coefficients of its own half, two scalar
    // chains (packing the coefficients of two different halves costs more than it saves)
    P inv2k, xoff;
    rr_pairP<K_INV2K>(K, inv2k, xoff);
    const P x = fma2(z, inv2k, xoff);
    const bool lox = x.x <= (R)0.5, loy = x.y <= (R)0.5;
    const P xx = abs2(sel2(lox, loy, x, sub2(splat<R>((R)1), x)));
    const P w = fma2(xx, splat<R>((R)4), splat<R>((R)-1));
    const R tiny = sizeof(R) == 8 ? (R)RR_TINY_D : (R)1e-30f;
    const P t = mul2(xx, rr_sqrt2(add2(xx, splat<R>(tiny))));
    const R px = rr_polyR<Cst<R, M>::OFF_LENS>(K, lox, w.x);
    const R py = rr_polyR<Cst<R, M>::OFF_LENS>(K, loy, w.y);
    R lx = lox ? fma(-t.x, px, afull.x) : t.x * px;
    R ly = loy ? fma(-t.y, py, afull.y) : t.y * py;
    if constexpr (sizeof(R) == 4) { lx = fmaxf(lx, 0.0f); ly = fmaxf(ly, 0.0f); }
    ap = mk2(inx ? lx : afull.x, iny ? ly : afull.y);
  } else if (inx || iny) {                      // lens area (rr_deficit), both elements
    const P omks = rr_getP<K_OMKS>(K);
    const P A = sub2(opk, z), B = add2(z, omks), C = sub2(z, omks), D = add2(z, opk);
    const P AB = abs2(mul2(A, B)), S = abs2(mul2(C, D)), Q = mul2(B, D);
    const R tiny = sizeof(R) == 8 ? (R)RR_TINY_D : (R)1e-30f;
    const P kite = rr_sqrt2(add2(mul2(AB, S), splat<R>(tiny)));
    const P tk2 = rr_getP<K_2K2>(K);
    const P h2 = rr_atan_quadrant2(kite, S, AB);
    const P h1 = ksmall ? rr_atan_t2(rr_div3_2(kite, Q))
                        : rr_atan_quadrant2(kite, Q, abs2(mul2(A, C)));
    P lens = fma2(h1, splat<R>((R)2), fma2(tk2, h2, mul2(splat<R>((R)-0.5), kite)));
    if constexpr (sizeof(R) == 4) lens = mk2(fmaxf(lens.x, 0.0f), fmaxf(lens.y, 0.0f));
    ap = sel2(inx, iny, lens, afull);
  }
  return sel2(ox, oy, mul2(ip, ap), splat<R>((R)0));
}

// The thread-per-exposure loop of rr_tile for a pair of exposures i and i + FT.
template <typename R, typename O, bool CIRC, bool NOWRAP, int M>
__device__ __forceinline__ void rr_tile_pairs(const double *__restrict__ times, O *__restrict__ out,
                                              int count, int ns, double t0, double inv_p,
                                              double u_mid, double hwid, double hw, O scale,
                                              const Cst<R, M> K, int kmode) {
  using P = typename PairT<R>::type;
  const bool ksmall = (kmode & 1) != 0;
  constexpr bool ANG = NOWRAP && sizeof(R) == 4;   // fp32 angle step per sub-sample
  const double du = 2.0 * hw / ns, off0 = hw * (1.0 / ns - 1.0), hskip = hwid + hw;
  const bool need_front =
      __shfl_sync(0xffffffffu, (int)(CIRC ? !(hskip + hw < 0.25) : !(hwid < 0.49)), 0) != 0;
  // (lane-0 broadcasts: opaque, or the compiler recomputes both from fp64 in the sub-sample loop)
  const float2 da2 = splat<float>(__shfl_sync(0xffffffffu, (float)(RR_TWOPI * du), 0));
  const float hwa = __shfl_sync(0xffffffffu, (float)(RR_TWOPI * hwid), 0);
  const float inv_hwa = __shfl_sync(0xffffffffu, (float)(1.0 / (RR_TWOPI * hwid)), 0);
  const float inv_hw = __shfl_sync(0xffffffffu, (float)(1.0 / hwid), 0);
  uintptr_t tp = reinterpret_cast<uintptr_t>(times + threadIdx.x);
  uintptr_t op = reinterpret_cast<uintptr_t>(out + threadIdx.x);
  int left = count - (int)threadIdx.x;
  double tna = left > 0 ? rr_ld_time(tp) : 0.0, tnb = left > FT ? rr_ld_time(tp + FT * 8) : tna;
  for (; left > 0; left -= 2 * FT) {
    const bool has1 = left > FT;
    const double ta = tna, tb = tnb;
    // the next pair's times are in flight during this pair
    if (left > 2 * FT) {
      tna = rr_ld_time(tp + 2 * FT * 8);
      tnb = left > 3 * FT ? rr_ld_time(tp + 3 * FT * 8) : tna;
    }
    const double wca = fma(ta - t0, inv_p, -u_mid), wcb = fma(tb - t0, inv_p, -u_mid);
    const double wra = wca - rr_round(wca), wrb = wcb - rr_round(wcb);
    const bool ina = fabs(wra) <= hskip, inb = has1 && fabs(wrb) <= hskip;
    O fa = (wra == wra) ? (O)1 : rr_nan<O>(), fb = (wrb == wrb) ? (O)1 : rr_nan<O>();
    if (ina || inb) {
      O acca = (O)0, accb = (O)0;
      // an exposure outside the window gets a phase that never passes the test: no flag to keep
      double wa = ina ? wra + off0 : 1e30, wb = inb ? wrb + off0 : 1e30;
      const P opk2 = rr_getP<K_OPK2>(K);
      // ANG (fp32, the exposure cannot wrap): the angles 2 pi x phase from the window centre (aw)
      // and from conjunction (am) of the first sub-sample rounded ONCE from fp64, then an fp32 step
      // per sub-sample - 2 eps32 |angle|, the size of the rounding of dM the fp32 solver starts from
      // anyway - instead of six fp64 instructions and two conversions per element
      const float2 aw0 = make_float2(ina ? (float)(RR_TWOPI * wa) : 1e30f, inb ? (float)(RR_TWOPI * wb) : 1e30f);
      const float2 am0 = make_float2((float)(RR_TWOPI * (wra + off0 + u_mid)), (float)(RR_TWOPI * (wrb + off0 + u_mid)));
      float2 fs = splat<float>(0.0f);
      for (int s = 0; s < ns; ++s, wa += du, wb += du) {
        bool ax, ay;
        P dM;
        P tw = splat<R>((R)0);                  // phase from the window centre / hwid
        if constexpr (ANG) {
          const float2 aws = fma2(fs, da2, aw0), aw = abs2(aws);
          ax = aw.x <= hwa;
          ay = aw.y <= hwa;
          const float2 am = fma2(fs, da2, am0);
          fs = add2(fs, splat<float>(1.0f));
          if (!(ax || ay)) continue;
          dM = mk2((R)am.x, (R)am.y);
          tw = mk2((R)(ax ? aws.x * inv_hwa : 0.0f), (R)(ay ? aws.y * inv_hwa : 0.0f));
        } else {
          const double was = NOWRAP ? wa : wa - rr_round(wa), wbs = NOWRAP ? wb : wb - rr_round(wb);
          ax = fabs(was) <= hwid;               // (1e30 - round(1e30) = 0: only without NOWRAP ...
          ay = fabs(wbs) <= hwid;
          if (!NOWRAP) { ax = ax && ina; ay = ay && inb; }   // ... where the flags are needed)
          if (!(ax || ay)) continue;
          dM = mk2((R)(RR_TWOPI * (was + u_mid)), (R)(RR_TWOPI * (wbs + u_mid)));
          if (kmode & 4) {
            const R invhw = K.template get<K_INVHW>();
            tw = mk2(ax ? (R)was * invhw : (R)0, ay ? (R)wbs * invhw : (R)0);
          }
        }
        dM = sel2(ax, ay, dM, splat<R>((R)0));
        bool fx = true, fy = true;
        P z2;
        if (!CIRC && (kmode & 4)) {
          // z^2 of both elements from the pv's polynomials (rr_zpoly_fit), each in its own half
          if constexpr (!CIRC) {
            const R tiny = sizeof(R) == 8 ? (R)RR_TINY_D : (R)1e-30f;
            const R px = rr_polyR<Cst<R, M>::OFF_ZPOLY>(K, tw.x < (R)0, fma(fabs(tw.x), (R)2, (R)-1));
            const R py = rr_polyR<Cst<R, M>::OFF_ZPOLY>(K, tw.y < (R)0, fma(fabs(tw.y), (R)2, (R)-1));
            z2 = mk2(fabs(px) + tiny, fabs(py) + tiny);
          }
        } else {
          z2 = rr_separation2_pair<R, CIRC, M>(K, dM, ax, ay, fx, fy);
        }
        bool ox = ax && z2.x < opk2.x, oy = ay && z2.y < opk2.y;
        if (need_front) { ox = ox && fx; oy = oy && fy; }
        if (ox || oy) {
          const P def = rr_deficit_pair<R, M>(K, z2, ox, oy, kmode);
          acca += (O)def.x;
          accb += (O)def.y;
        }
      }
      // mean of (Istar - ip ap)/Istar over ns; fp64 staged the table already times 1/(Istar ns)
      if (ina) fa = sizeof(R) == 8 ? (O)1 - acca : fma(-acca, scale, (O)1);
      if (inb) fb = sizeof(R) == 8 ? (O)1 - accb : fma(-accb, scale, (O)1);
    }
    RR_STORE(reinterpret_cast<O *>(op), fa);
    if (has1) RR_STORE(reinterpret_cast<O *>(op + FT * sizeof(O)), fb);
    asm volatile("add.u64 %0, %0, %1;" : "+l"(tp) : "n"(2 * FT * 8));
    asm volatile("add.u64 %0, %0, %1;" : "+l"(op) : "n"(2 * FT * (int)sizeof(O)));
  }
}

// The exposures of one tile for one pv.  CIRC: e == 0 (block-uniform).
// R = arithmetic type of z and ip*ap; O = type of the sub-sample sum, the final 1 - sum/(Istar ns)
// and the stored flux (O = double with R = float is RR_MIXED, the scheme of PAPER.md:293).
template <typename R, typename O, bool COUNT, bool CIRC, bool NOWRAP, int M, bool PAIRS>
__device__ __forceinline__ void rr_tile(const double *__restrict__ times, O *__restrict__ out,
                                        int count, int ns, int shuffle, double t0, double inv_p,
                                        double u_mid, double hwid, double hw, O scale,
                                        const Cst<R, M> K, unsigned long long *cnt) {
  const double du = 2.0 * hw / ns;                   // sub-sample spacing, turns
  const double off0 = hw * (1.0 / ns - 1.0);         // first sub-sample offset (reading R7)
  const double hskip = hwid + hw;
  // k^2 <= 1/2 (block-uniform; lane-0 broadcast so that it stays a predicate, not a compare per use)
  const int kmode = __shfl_sync(0xffffffffu, (int)(K.template get<K_K2>() <= (R)0.5) |
                                                 (K.template get<K_LENSOK>() != (R)0 ? 2 : 0) |
                                                 (K.template get<K_ZOK>() != (R)0 ? 4 : 0), 0);
  const bool ksmall = (kmode & 1) != 0;
  if constexpr (PAIRS && !COUNT && !(CIRC && sizeof(R) == 8)) {
    if (!shuffle && count > FT) {   // two exposures per thread (tiles of <= FT exposures, the
                                    // counting build and fp64 circular tiles keep the scalar loop)
      rr_tile_pairs<R, O, CIRC, NOWRAP, M>(times, out, count, ns, t0, inv_p, u_mid, hwid, hw, scale,
                                           K, kmode);
      return;
    }
  }
  if (!shuffle) {
    // ---- one thread per exposure, in-thread loop over its sub-samples ----
    // The time and flux pointers advance by opaque 64-bit adds: otherwise the compiler, short of
    // registers, rebuilds both addresses from the kernel parameters at every exposure (15
    // instructions).
    uintptr_t tp = reinterpret_cast<uintptr_t>(times + threadIdx.x);
    uintptr_t op = reinterpret_cast<uintptr_t>(out + threadIdx.x);
    int left = count - (int)threadIdx.x;             // exposures of this thread still to do, x FT
    double tnext = left > 0 ? rr_ld_time(tp) : 0.0;
    // circular: the in-front test is only needed when the evaluated phases can reach a quarter turn
    // (lane-0 broadcast: opaque, or the compiler recomputes the fp64 test in the inner loop)
    const bool need_front =
        __shfl_sync(0xffffffffu, (int)(CIRC ? !(hskip + hw < 0.25) : !(hwid < 0.49)), 0) != 0;
    while (left > 0) {
      const double tcur = tnext;
      left -= FT;
      asm volatile("add.u64 %0, %0, %1;" : "+l"(tp) : "n"(FT * 8));
      if (left > 0) tnext = rr_ld_time(tp);            // in flight during this exposure
      const double wc = fma(tcur - t0, inv_p, -u_mid);
      const double wr = wc - rr_round(wc);           // exposure centre from the window centre
      O f;
      if (!(fabs(wr) <= hskip)) {
        f = (wr == wr) ? (O)1 : rr_nan<O>();         // out of the window; NaN time: reading R15
        if (COUNT) cnt[0] += ns;
      } else {
        O acc = (O)0;
        if (CIRC && sizeof(R) == 8) {
          // circular orbit, fp64: sin and cos of the first sub-sample's phase, then one plane
          // rotation per sub-sample (constant phase step); no per-sub-sample window test is
          // needed, outside the window z >= 1+k by construction.  (fp32 keeps the polynomial per
          // sub-sample: a rotation's ABSOLUTE rounding error times a is too much for z there.)
          const double ur0 = (wr + off0) + u_mid;
          R sn, cs;
          if (fabs(ur0) <= 0.07949995994567871) {    // 0x3FB45A1C'00000000: 2 pi u <= 0.4995
            R cm1;
            rr_sincosm1_small((R)(RR_TWOPI * ur0), sn, cm1);
            cs = (R)1 + cm1;
          } else {
            double s_, c_;
            sincospi(2.0 * ur0, &s_, &c_);
            sn = (R)s_;
            cs = (R)c_;
          }
          R zc0, zc1, cd, sd;
          K.template pair<K_ZC0>(zc0, zc1);
          K.template pair<K_CD>(cd, sd);
          const R opk2 = K.template get<K_OPK2>();
          for (int s = 0; s < ns; ++s) {
            const R z2 = fma(sn * sn, zc1, zc0);     // zc0 carries +2^-1000: z2 > 0
            bool occ = z2 < opk2;
            if (need_front) occ = occ && cs > (R)0;
            // the next sub-sample's rotation first: independent work under the deficit's latency
            const R s1 = fma(sn, cd, cs * sd);
            cs = fma(cs, cd, -sn * sd);
            sn = s1;
            if (occ) {
              int ing = 0;
              acc += rr_deficit<R, M>(K, z2, ing, kmode);
              if (COUNT) { cnt[3]++; cnt[4] += ing; }
            }
          }
          if (COUNT) cnt[1] += ns;
        } else {
          double w = wr + off0;
          for (int s = 0; s < ns; ++s, w += du)
            acc += rr_subsample<R, COUNT, CIRC, NOWRAP, M>(K, w, u_mid, hwid, need_front, kmode, cnt);
        }
        // mean of (Istar - ip ap)/Istar over ns; fp64 staged the table already times 1/(Istar ns)
        f = sizeof(R) == 8 ? (O)1 - acc : fma(-acc, scale, (O)1);
      }
      RR_STORE(reinterpret_cast<O *>(op), f);
      asm volatile("add.u64 %0, %0, %1;" : "+l"(op) : "n"(FT * (int)sizeof(O)));
    }
  } else {
    // ---- sub-samples across lanes, warp-shuffle sum ----
    int G = 1;
    while (G < ns && G < 32) G <<= 1;               // lanes per exposure
    const int sl = threadIdx.x & (G - 1);
    const int per_pass = FT / G;
    for (int base = 0; base < count; base += per_pass) {
      const int i = base + (threadIdx.x / G);
      const bool live = i < count;
      O acc = (O)0;
      double wr = 0.0;
      if (live) {
        const double wc = fma(times[i] - t0, inv_p, -u_mid);
        wr = wc - rr_round(wc);
        if (fabs(wr) <= hskip) {
          const double w0 = wr + off0;
          for (int s = sl; s < ns; s += G)
            acc += rr_subsample<R, COUNT, CIRC, false, M>(K, fma(du, (double)s, w0), u_mid, hwid, true,
                                                          kmode, cnt);
        } else if (COUNT) {
          for (int s = sl; s < ns; s += G) cnt[0]++;
        }
      }
      for (int o = G >> 1; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
      if (live && sl == 0)
        out[i] = (wr == wr) ? (sizeof(R) == 8 ? (O)1 - acc : fma(-acc, scale, (O)1)) : rr_nan<O>();
    }
  }
}

// One block per (parameter vector, chunk of consecutive dispatch tiles).  Block = FT threads.
// The pv's constants are staged once per block, the k-collapsed table row once per light curve the
// chunk meets; tiles outside the transit window are merged into contiguous runs and written as
// flux = 1 by TMA bulk copies (rr_fill_ones_bulk), without touching the orbit.
// Shared memory (rr_dyn): cst[K_SMEM] (constants, 8-byte slots) | ldw2[ldw_len] (node, slope)
// pairs of the k-collapsed table row.
// MODE 0: plain; 1: with the class counters (bench.py's op count); 2: fp32 kernels with the
// two-exposures-per-thread FFMA2 loop for tiles longer than a block (the launcher picks it when the
// tiles of the data are, on average, longer than 1.5 FT exposures; a kernel of its own because the
// extra code costs the scalar loop registers: the sparse cadence 4b ran 8 % slower with both in one).
#ifndef RR_FP64_PAIR_BLOCKS
#define RR_FP64_PAIR_BLOCKS 6   // resident blocks per SM of the fp64 pair kernel (80 registers)
#endif
#ifndef RR_FP32_PAIR_BLOCKS
#define RR_FP32_PAIR_BLOCKS RR_FLUX_MIN_BLOCKS
#endif
template <typename R, typename O, int MODE, int M>
__global__ void __launch_bounds__(FT, MODE != 2 ? RR_FLUX_MIN_BLOCKS
                                                : (sizeof(R) == 8 ? RR_FP64_PAIR_BLOCKS
                                                                  : RR_FP32_PAIR_BLOCKS))
rr_flux_kernel(const FluxParams P) {
  constexpr bool COUNT = MODE == 1;
  constexpr bool PAIRS = MODE == 2;
  const Cst<R, M> K;
  using R2 = typename Cst<R, M>::R2;
  unsigned *tflags = Cst<R, M>::flags();
  unsigned long long cnt[7] = {0, 0, 0, 0, 0, 0, 0};
  unsigned long long cfill = 0, ceval = 0;

#if RR_BULK_FILL
  // ones for the bulk fill, after the staged row (16-byte aligned); written at the block's first fill
  unsigned char *ones_p = rr_dyn + P.ones_off;
  const unsigned ones_smem = (unsigned)__cvta_generic_to_shared(ones_p);
  bool ones_ready = false;
#endif
  const unsigned v = blockIdx.x / P.nchunks;
  const unsigned chunk = blockIdx.x - v * P.nchunks;
  const int64_t tl0 = (int64_t)chunk * P.chunk_len;
  const int64_t tl1 = min(tl0 + (int64_t)P.chunk_len, P.ntiles);
  const RRPvOrbit &po = P.pvo[v];
  O *row = reinterpret_cast<O *>(P.flux) + (int64_t)v * P.npt;
  if (po.status) {                                     // reading R12: NaN row
    const RRTile a = P.tiles[tl0], b = P.tiles[tl1 - 1];
    rr_fill<O>(row + a.start, (int64_t)b.start + b.count - a.start, rr_nan<O>());
    return;
  }
  const double t0 = po.t0, inv_p = po.inv_p, u_mid = po.u_mid, hwid = po.hwid;
  const int circular = po.circular;
  int desc_lc = -1, staged_lc = -1;                    // light curve of lc / of the staged table
  RRLc lc;
  double hw = 0.0;                                     // half an exposure, in turns
  O scale = (O)0;
  int64_t f0 = -1, f1 = 0;                             // pending run of exposures with flux 1

  for (int64_t base = tl0; base < tl1; base += FT) {
    const int ngrp = (int)min((int64_t)FT, tl1 - base);
    // Each thread tests ONE tile of the group against the transit window (modulo one turn): the
    // phases of the tile, measured from the window centre, lie in [wa, wb]; n = first turn whose
    // window can end after wa.  Out-of-window tiles get flux 1 without evaluation.
    bool in = false;
    if ((int)threadIdx.x < ngrp) {
      const RRTile *tp = P.tiles + base + threadIdx.x;
      const double hwt = 0.5 * P.lcs[tp->lc].exptime * inv_p;
      const double wa = fma(tp->tmin - t0, inv_p, -u_mid) - hwt;
      const double wb = fma(tp->tmax - t0, inv_p, -u_mid) + hwt;
      in = !(ceil(wa - hwid) - hwid > wb);
    }
    const unsigned mask = __ballot_sync(0xffffffffu, in);
    __syncthreads();                                   // the previous group's flags are consumed
    if ((threadIdx.x & 31) == 0) tflags[threadIdx.x >> 5] = mask;
    __syncthreads();
    const int nwords = (ngrp + 31) >> 5;
    int pos = 0;
    while (pos < ngrp) {
      int q = ngrp;                                    // next in-window tile at or after pos
      for (int w = pos >> 5; w < nwords; ++w) {
        unsigned bits = tflags[w];
        if (w == (pos >> 5)) bits &= 0xffffffffu << (pos & 31);
        if (bits) { q = (w << 5) + __ffs(bits) - 1; break; }
      }
      if (q > pos) {                                   // tiles pos .. q-1: extend the pending run
        const RRTile *ta = P.tiles + base + pos, *tb = P.tiles + base + q - 1;
        if (f0 < 0) f0 = ta->start;
        f1 = (int64_t)tb->start + tb->count;
        if (COUNT) cfill += (threadIdx.x == 0) ? (unsigned long long)(q - pos) : 0ull;
      }
      if (q >= ngrp) break;
      pos = q + 1;
      if (f0 >= 0) {
#if RR_BULK_FILL
        if (!ones_ready) { rr_ones_setup<O>(ones_p); ones_ready = true; }
        rr_fill_ones_bulk<O>(row + f0, f1 - f0, ones_smem);
#else
        rr_fill<O>(row + f0, f1 - f0, (O)1);
#endif
        f0 = -1;
      }
      const RRTile *tp = P.tiles + base + q;
      // warp-uniform by construction; the lane-0 broadcast lets ptxas keep them (and the tile's base
      // pointers) in uniform registers
      const int tstart = __shfl_sync(0xffffffffu, tp->start, 0);
      const int tcount = __shfl_sync(0xffffffffu, tp->count, 0);
      const int tlc = __shfl_sync(0xffffffffu, tp->lc, 0);
      if (tlc != desc_lc) {
        lc = P.lcs[tlc];
        desc_lc = tlc;
        hw = 0.5 * lc.exptime * inv_p;
      }
      if (COUNT) ceval += (threadIdx.x == 0);
      if (tlc != staged_lc) {
        // stage the k-collapsed table row ldw[ng] as (node, slope) cells, and the
        // constants, in shared memory
        const int kb = (P.nkpb == 1) ? 0 : lc.pb;
        const RRPvBand &pb = P.pvb[(int64_t)v * P.nkpb + kb];
        const int64_t trow = (int64_t)v * P.npb + lc.pb;
        R2 *ldw2 = Cst<R, M>::row();
        // fp64: the cells carry the factor 1/(Istar ns), so that flux = 1 - sum(ip ap) needs no
        // final scaling; fp32 keeps it apart (one rounding less on the occulted light)
        const double sc_d = 1.0 / ((double)reinterpret_cast<const R *>(P.istar)[trow] * lc.ns);
        const R sc = sizeof(R) == 8 ? (R)sc_d : (R)1;
        __syncthreads();
        if (P.rows) {                                  // lazy mode: the row was collapsed for this k
          const R *rw = reinterpret_cast<const R *>(P.rows) + trow * (int64_t)P.ng;
          for (int ig = threadIdx.x; ig < P.ldw_len; ig += FT) {
            const R a = rw[min(ig, P.ng - 1)], b = rw[min(ig + 1, P.ng - 1)];
            R2 c;
            c.x = a * sc;
            c.y = (b - a) * sc;
            ldw2[ig] = c;
          }
        } else {
          const R *T0 = reinterpret_cast<const R *>(P.T) + (trow * P.nk + pb.ik) * (int64_t)P.ng;
          const R *T1 = T0 + P.ng;
          const R ak = (R)pb.ak;
          for (int ig = threadIdx.x; ig < P.ldw_len; ig += FT) {
            const int jg = min(ig, P.ng - 1), jh = min(ig + 1, P.ng - 1);   // cells >= ng-1: flat
            const R a = fma(ak, T1[jg] - T0[jg], T0[jg]), b = fma(ak, T1[jh] - T0[jh], T0[jh]);
            R2 c;
            c.x = a * sc;
            c.y = (b - a) * sc;
            ldw2[ig] = c;
          }
        }
        const bool lens_on = P.lens != nullptr && pb.lens_ok != 0;
        if constexpr (sizeof(R) == 8) {
          if (lens_on && threadIdx.x < 2 * RR_LENS_PITCH)
            Cst<R, M>::lens()[threadIdx.x] =
                P.lens[((int64_t)v * P.nkpb + kb) * (2 * RR_LENS_PITCH) + threadIdx.x];
        } else {              // fp32 kernels: the coefficients rounded to fp32, 16 floats per half
          if (lens_on && threadIdx.x < 32) {
            const int half = threadIdx.x >> 4, j = threadIdx.x & 15;
            reinterpret_cast<float *>(Cst<R, M>::lens())[threadIdx.x] =
                j < RR_LENS_N ? (float)P.lens[((int64_t)v * P.nkpb + kb) * (2 * RR_LENS_PITCH) +
                                              half * RR_LENS_PITCH + j] : 0.0f;
          }
        }
        const bool zpoly_on = P.zpoly != nullptr && po.zpoly_ok != 0;
        if constexpr (sizeof(R) == 8) {
          if (zpoly_on && threadIdx.x >= 32 && threadIdx.x < 32 + 2 * RR_LENS_PITCH)
            Cst<R, M>::zpoly()[threadIdx.x - 32] =
                P.zpoly[(int64_t)v * (2 * RR_LENS_PITCH) + threadIdx.x - 32];
        } else {              // fp32 kernels: the coefficients rounded to fp32, 16 floats per half
          if (zpoly_on && threadIdx.x >= 32 && threadIdx.x < 64) {
            const int half = (threadIdx.x - 32) >> 4, j = threadIdx.x & 15;
            reinterpret_cast<float *>(Cst<R, M>::zpoly())[threadIdx.x - 32] =
                j < RR_LENS_N ? (float)P.zpoly[(int64_t)v * (2 * RR_LENS_PITCH) + half * RR_LENS_PITCH + j]
                              : 0.0f;
          }
        }
        rr_stage_constants<R>(po, pb, 2.0 * hw / lc.ns, lens_on, zpoly_on);
        if (threadIdx.x == K_SCALE) Cst<R, M>::store(K_SCALE, sc_d);
        __syncthreads();
        scale = (O)K.template get<K_SCALE>();
        staged_lc = tlc;
      }
      const int shuffle = lc.ns >= P.shuffle_min_ns;
      const bool nowrap = hwid + 2.0 * hw < 0.499;
      if (circular)
        rr_tile<R, O, COUNT, true, false, M, PAIRS>(P.times + tstart, row + tstart, tcount, lc.ns, shuffle, t0,
                                          inv_p, u_mid, hwid, hw, scale, K, cnt);
      else if (nowrap)
        rr_tile<R, O, COUNT, false, true, M, PAIRS>(P.times + tstart, row + tstart, tcount, lc.ns, shuffle, t0,
                                          inv_p, u_mid, hwid, hw, scale, K, cnt);
      else
        rr_tile<R, O, COUNT, false, false, M, PAIRS>(P.times + tstart, row + tstart, tcount, lc.ns, shuffle, t0,
                                           inv_p, u_mid, hwid, hw, scale, K, cnt);
    }
  }
#if RR_BULK_FILL
  if (f0 >= 0) {
    if (!ones_ready) { rr_ones_setup<O>(ones_p); ones_ready = true; }
    rr_fill_ones_bulk<O>(row + f0, f1 - f0, ones_smem);
  }
  // the bulk copies read the block's shared memory: it must outlive them
  if (ones_ready && threadIdx.x == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
#else
  if (f0 >= 0) rr_fill<O>(row + f0, f1 - f0, (O)1);
#endif
  if (COUNT) {
#pragma unroll
    for (int q = 0; q < 7; ++q) {
      unsigned long long x = cnt[q];
      for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
      if ((threadIdx.x & 31) == 0 && x) atomicAdd(P.counters + (q < 6 ? q : 8), x);
    }
    if (threadIdx.x == 0) {
      if (cfill) atomicAdd(P.counters + 6, cfill);
      if (ceval) atomicAdd(P.counters + 7, ceval);
    }
  }
}

// ---- kernel 2 alone ---------------------------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(FT)
rr_orbit_kernel(const double *__restrict__ times, const RRTile *__restrict__ tiles,
                const RRLc *__restrict__ lcs, const RRPvOrbit *__restrict__ pvo, int64_t ntiles,
                int64_t npv, int64_t nsub, double *__restrict__ zout) {
  const Cst<R, RR_SM_SYMBOL> K;
  const int64_t total = ntiles * npv;
  for (int64_t w = blockIdx.x; w < total; w += gridDim.x) {
    const int64_t v = w / ntiles;
    const int64_t tl = w - v * ntiles;
    const RRTile tile = tiles[tl];
    const RRLc lc = lcs[tile.lc];
    const RRPvOrbit &po = pvo[v];
    const int ns = lc.ns;
    double *out = zout + v * nsub + tile.sub_off;
    const int n = tile.count * ns;
    if (po.status) {
      for (int j = threadIdx.x; j < n; j += FT) out[j] = rr_nan<double>();
      continue;
    }
    RRPvBand nob = {};
    __syncthreads();
    rr_stage_constants<R>(po, nob, 0.0);
    __syncthreads();
    const double hw = 0.5 * lc.exptime * po.inv_p;
    const double du = 2.0 * hw / ns, off0 = hw * (1.0 / ns - 1.0);
    for (int j = threadIdx.x; j < n; j += FT) {
      int i = j / ns, s = j - i * ns;
      double us = fma(du, (double)s, (times[tile.start + i] - po.t0) * po.inv_p + off0);
      double ur = us - rint(us);
      bool front;
      int it = 0;
      R z2 = po.circular ? rr_separation2<R, true, RR_SM_SYMBOL>(K, ur, front, it)
                         : rr_separation2<R, false, RR_SM_SYMBOL>(K, ur, front, it);
      double z = (double)rr_sqrt(z2);
      out[j] = front ? z : -z;
    }
  }
}

// ---- FMA pipe peak (measurement aid) -------------------------------------------------------------
template <typename R>
__global__ void __launch_bounds__(256) rr_fma_peak_kernel(R *out, int iters, R a, R b) {
  R x0 = (R)threadIdx.x, x1 = x0 + 1, x2 = x0 + 2, x3 = x0 + 3, x4 = x0 + 4, x5 = x0 + 5,
    x6 = x0 + 6, x7 = x0 + 7;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  R s = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
  if (s == (R)123456789) out[0] = s;   // never true: keeps the chain alive
}

template <typename R>
int fma_peak_typed(double *h_fma_per_s, cudaStream_t st) {
  R *d = nullptr;
  RR_CUDA(cudaMalloc(&d, sizeof(R)));
  int dev = 0, sms = 0;
  RR_CUDA(cudaGetDevice(&dev));
  RR_CUDA(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  const int blocks = sms * 8, iters = 4096;
  cudaEvent_t e0, e1;
  RR_CUDA(cudaEventCreate(&e0));
  RR_CUDA(cudaEventCreate(&e1));
  double best = 0.0;
  for (int rep = 0; rep < 4; ++rep) {
    RR_CUDA(cudaEventRecord(e0, st));
    rr_fma_peak_kernel<R><<<blocks, 256, 0, st>>>(d, iters, (R)0.999999, (R)1e-6);
    RR_CUDA(cudaEventRecord(e1, st));
    RR_CUDA(cudaEventSynchronize(e1));
    float ms = 0.f;
    RR_CUDA(cudaEventElapsedTime(&ms, e0, e1));
    double rate = (double)blocks * 256.0 * iters * 64.0 / (ms * 1e-3);
    if (rep > 0 && rate > best) best = rate;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  *h_fma_per_s = best;
  return RR_OK;
}

// ---- device math probe (tests): the functions of rr_math.cuh applied element by element ------------
template <typename R>
__global__ void rr_math_probe_kernel(int op, const double *__restrict__ a, const double *__restrict__ b,
                                     int64_t n, double *__restrict__ o0, double *__restrict__ o1) {
  const int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const R x = (R)a[i], y = b ? (R)b[i] : (R)0;
  R r0 = (R)0, r1 = (R)0;
  switch (op) {
    case RR_PROBE_SQRT3: r0 = rr_sqrt3(x); break;
    case RR_PROBE_SQRT: r0 = rr_sqrt(x); break;
    case RR_PROBE_DIV3: r0 = rr_div3(x, y); break;
    case RR_PROBE_RCP: r0 = rr_rcp(x); break;
    case RR_PROBE_ATAN_T: r0 = rr_atan_t(x); break;
    case RR_PROBE_ATAN_QUADRANT: r0 = rr_atan_quadrant<R>(rr_sqrt3_pos(x * y), x, y); break;
    case RR_PROBE_ATAN2_POS: r0 = rr_atan2_pos(x, y); break;
    case RR_PROBE_SINCOSM1: rr_sincosm1_small(x, r0, r1); break;
    case RR_PROBE_CELL: {
      int ig;
      R ag;
      rr_cell(x, ig, ag);
      r0 = (R)ig;
      r1 = ag;
      break;
    }
    default: break;
  }
  o0[i] = (double)r0;
  if (o1) o1[i] = (double)r1;
}

}  // namespace

int rr_math_probe_launch(int op, int fp32, const double *d_a, const double *d_b, int64_t n,
                         double *d_o0, double *d_o1, cudaStream_t st) {
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (fp32) rr_math_probe_kernel<float><<<grid, 256, 0, st>>>(op, d_a, d_b, n, d_o0, d_o1);
  else rr_math_probe_kernel<double><<<grid, 256, 0, st>>>(op, d_a, d_b, n, d_o0, d_o1);
  RR_CUDA(cudaGetLastError());
  return RR_OK;
}

// Extra nodes of the staged table row beyond ng - 1 (all equal to the limb node): 1 normally; with
// mean-k weights and chromatic k, g = z/(1+kw) of a passband with k > kw runs up to (1+k)/(1+kw).
// The mode is that of the table actually built (wk->lazy), not the one set for the next build.
static int rr_row_pad(const rr_ctx *ctx, const RRWork *wk) {
  const rr_config &c = ctx->cfg;
  if (!(ctx->mean_k && c.nkpb > 1)) return 1;
  if (wk->lazy == 2) return c.ng + 2;    // direct model, no k limits: up to k = 1 + 2 kw
  return (int)ceil((c.ng - 1) * (c.k1 - c.k0) / (1.0 + c.k0)) + 3;
}

// ---- host launchers -------------------------------------------------------------------------------
// fp32_tol: Halley acceptance tolerance of the fp32 arithmetic (the RR_FP32 / RR_MIXED flux kernels
// and rr_orbit_z(fp32_math = 1)); the fp64 orbit kernel needs the fp64 one on any ctx.
int rr_pv_prep_launch(rr_ctx *ctx, RRWork *wk, const double *d_pv, int64_t npv,
                      int32_t *d_status, int fp32_tol, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  if (npv > wk->pv_cap) {
    if (wk->pvo) cudaFree(wk->pvo);
    if (wk->pvb) cudaFree(wk->pvb);
    wk->pvo = nullptr;
    wk->pvb = nullptr;
    wk->pv_cap = 0;
    if (wk->lens) cudaFree(wk->lens);
    wk->lens = nullptr;
    if (wk->zpoly) cudaFree(wk->zpoly);
    wk->zpoly = nullptr;
    if (cudaMalloc(&wk->pvo, sizeof(RRPvOrbit) * npv) != cudaSuccess ||
        cudaMalloc(&wk->pvb, sizeof(RRPvBand) * npv * c.nkpb) != cudaSuccess ||
        cudaMalloc(&wk->lens, sizeof(double) * 2 * RR_LENS_PITCH * npv * c.nkpb) != cudaSuccess ||
        cudaMalloc(&wk->zpoly, sizeof(double) * 2 * RR_LENS_PITCH * npv) != cudaSuccess) {
      cudaGetLastError();
      return RR_EALLOC;
    }
    wk->pv_cap = npv;
  }
  // direct model (no k grid): any k > 0 is valid
  const bool direct = wk->lazy == 2;
  rr_pv_prep_kernel<<<(unsigned)((npv + 127) / 128), 128, 0, st>>>(
      d_pv, npv, c.nkpb, c.nk, c.k0, c.k1, direct ? 1e-300 : c.k0, direct ? 1e300 : c.k1, c.ng,
      fp32_tol, ctx->mean_k, rr_row_pad(ctx, wk), wk->pvo, wk->pvb, d_status);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

static unsigned rr_grid_for(int64_t total) {
  const int64_t cap = 0x7fffffffLL;
  return (unsigned)(total < cap ? (total > 0 ? total : 1) : cap);
}

int rr_flux_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, void *d_flux, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  FluxParams P;
  P.times = ctx->d_times;
  P.tiles = ctx->d_tiles;
  P.lcs = ctx->d_lc;
  P.pvo = wk->pvo;
  P.pvb = wk->pvb;
  P.T = wk->lazy ? nullptr : wk->T;
  P.rows = wk->lazy ? wk->rows : nullptr;
  P.istar = wk->istar;
  P.lens = (RR_LENS_POLY && ctx->lens_poly) ? wk->lens : nullptr;   // (fitted in fp64 for every precision)
  P.flux = d_flux;
  P.counters = ctx->d_counters;
  P.npt = ctx->npt;
  P.npv = npv;
  P.ntiles = ctx->ntiles;
  P.npb = c.npb;
  P.nkpb = c.nkpb;
  P.nk = c.nk;
  P.ng = c.ng;
  // Supersample reduction layout.  Thread-per-exposure streams flux fully coalesced and needs no
  // shuffle; lanes-over-sub-samples multiplies the parallelism by ns, which only pays when
  // npv x npt alone cannot fill the GPU.
  const int64_t resident = (int64_t)ctx->sm_count * 2048;
  P.ldw_len = c.ng + rr_row_pad(ctx, wk);
  if (ctx->reduction == RR_REDUCE_THREAD) P.shuffle_min_ns = 0x7fffffff;
  else if (ctx->reduction == RR_REDUCE_SHUFFLE) P.shuffle_min_ns = 2;
  else P.shuffle_min_ns = (npv * ctx->npt < 2 * resident) ? 4 : 0x7fffffff;
  if (ctx->ntiles <= 0 || npv <= 0) return RR_OK;
  // Blocks: one per (pv, chunk of consecutive tiles).  One chunk per pv when the population alone
  // gives every SM RR_FLUX_WAVES waves of blocks (table row and constants staged once per pv);
  // otherwise the tile axis is cut so that about that many waves exist.
  const int64_t want = (int64_t)ctx->sm_count * RR_FLUX_MIN_BLOCKS * RR_FLUX_WAVES;
  int64_t nchunks = (want + npv - 1) / npv;
  // (at least two tiles per block: with one, the per-block set-up shows - config 2 3.5 % slower)
  nchunks = std::max<int64_t>(1, std::min<int64_t>(nchunks, std::max<int64_t>(1, ctx->ntiles / 2)));
  const int64_t chunk_len = (ctx->ntiles + nchunks - 1) / nchunks;
  nchunks = (ctx->ntiles + chunk_len - 1) / chunk_len;
  if (npv * nchunks > 0x7fffffffLL) return RR_ESIZE;
  P.nchunks = (unsigned)nchunks;
  P.chunk_len = (unsigned)chunk_len;
  const unsigned grid = (unsigned)(npv * nchunks);
  size_t smem = (size_t)K_SMEM * 8 + 16 + 4 * RR_LENS_PITCH * 8 +
                (size_t)2 * P.ldw_len * (c.precision != RR_FP64 ? 4 : 8);
  smem = (smem + 15) & ~(size_t)15;
  P.ones_off = (unsigned)smem;
#if RR_BULK_FILL
  smem += RR_ONES_BYTES;
#endif
  if (ctx->counters_on)
    RR_CUDA(cudaMemsetAsync(ctx->d_counters, 0, sizeof(unsigned long long) * 16, st));
  using Kernel = void (*)(const FluxParams);
  const int pi = c.precision == RR_FP32 ? 1 : (c.precision == RR_MIXED ? 2 : 0);
#define RR_KROW(R, O, M)                                                                          \
  {rr_flux_kernel<R, O, 0, M>, rr_flux_kernel<R, O, 1, M>,                                        \
   rr_flux_kernel<R, O, (sizeof(R) == 8 && !RR_FP64_PAIRS) ? 0 : 2, M>}
  static const Kernel kernels[2][3][3] = {
      {RR_KROW(double, double, RR_SM_FALLBACK_F64), RR_KROW(float, float, RR_SM_FALLBACK_F32),
       RR_KROW(float, double, RR_SM_FALLBACK_F32)},
      {RR_KROW(double, double, RR_SM_ABS), RR_KROW(float, float, RR_SM_ABS),
       RR_KROW(float, double, RR_SM_ABS)}};
#undef RR_KROW
  // fp32 kernels: the pair loop when the data's tiles are long enough to give a thread two exposures
  const bool pairs = (pi != 0 ? RR_FP32_PAIRS : RR_FP64_PAIRS) &&
                     2 * ctx->npt > 3 * (int64_t)FT * ctx->ntiles &&
                     ctx->reduction != RR_REDUCE_SHUFFLE;
  const Kernel kern = kernels[ctx->smem_abs ? 1 : 0][pi][ctx->counters_on ? 1 : (pairs ? 2 : 0)];
  P.zpoly = (RR_ZPOLY && ctx->orbit_poly) ? wk->zpoly : nullptr;   // (fitted in fp64 for every precision)
  if (P.zpoly || P.lens) {  // the per-pv polynomials (lens area, z^2 over the transit window): one launch
    const int64_t nrows = npv * c.nkpb, nw = (P.lens ? nrows : 0) + (P.zpoly ? npv : 0);
    rr_poly_fit_kernel<<<(unsigned)((nw * 32 + 255) / 256), 256, 0, st>>>(
        wk->pvb, nrows, P.lens ? wk->lens : nullptr, wk->pvo, npv, P.zpoly ? wk->zpoly : nullptr);
    RR_LAUNCH_CHECK(ctx);
  }
  if (smem > 48 * 1024)     // large ng, or mean-k padding: opt in to more dynamic shared memory
    RR_CUDA(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  kern<<<grid, FT, smem, st>>>(P);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

int rr_orbit_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, double *d_z, int fp32_math,
                    cudaStream_t st) {
  const int64_t total = ctx->ntiles * npv;
  if (total <= 0) return RR_OK;
  const unsigned grid = rr_grid_for(total);
  if (fp32_math)
    rr_orbit_kernel<float><<<grid, FT, K_SMEM * 8 + 16 + 4 * RR_LENS_PITCH * 8, st>>>(ctx->d_times, ctx->d_tiles, ctx->d_lc, wk->pvo,
                                                ctx->ntiles, npv, ctx->nsub, d_z);
  else
    rr_orbit_kernel<double><<<grid, FT, K_SMEM * 8 + 16 + 4 * RR_LENS_PITCH * 8, st>>>(ctx->d_times, ctx->d_tiles, ctx->d_lc,
                                                 wk->pvo, ctx->ntiles, npv, ctx->nsub, d_z);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

// ---- allocation-free entry point (rr_orbit_z_noalloc): kernel 2 alone, scratch in a static array ----
// Some callers cannot call cudaMalloc (code under CUDA graph capture, tight serving loops, harnesses
// that forbid it).  rr_orbit_z's scratch - the per-pv orbit and radius-ratio constants the prep kernel
// writes and the orbit kernel reads - normally lives in buffers the ctx grows with cudaMalloc; here it
// lives in ONE file-scope device array of RR_NOALLOC_SCRATCH_BYTES (2 MiB), which every GPU that loads
// the library holds until exit.  Layout: RRPvOrbit[npv] | (256-byte aligned) RRPvBand[npv nkpb].
// In host code `rr_noalloc_scratch` is a host-side stand-in, not a device address: its device address
// is taken once per device with cudaGetSymbolAddress (rr_noalloc_setup, from rr_create, with the
// ctx's device current) and handed to the kernels.  Every call on a device shares the array, which
// keeps the last call's contents: nothing in it needs to start at zero (the prep kernel writes every
// entry the orbit kernel reads, for exactly the npv rows of this call, before it reads them, on the
// same stream), but two calls that overlap on the GPU (different streams, or different contexts on
// one device) race on it.
static_assert(sizeof(RRPvOrbit) == 200 && sizeof(RRPvBand) == 72,
              "roadrunner.h states the no-alloc limit with these sizes");
static __device__ __align__(256) unsigned char rr_noalloc_scratch[RR_NOALLOC_SCRATCH_BYTES];

int rr_noalloc_setup(rr_ctx *ctx) {
  static std::mutex mu;
  static void *addr[64] = {nullptr};               // device address of the array, per device
  std::lock_guard<std::mutex> lock(mu);
  const int d = ctx->device;                       // the current device (rr_create)
  void *p = (d >= 0 && d < 64) ? addr[d] : nullptr;
  if (!p) {
    RR_CUDA(cudaGetSymbolAddress(&p, rr_noalloc_scratch));
    if (d >= 0 && d < 64) addr[d] = p;
  }
  ctx->noalloc_scratch = p;
  return RR_OK;
}

// As rr_pv_prep_launch + rr_orbit_launch with pvo / pvb in the static scratch.  No allocation.
int rr_orbit_noalloc_launch(rr_ctx *ctx, const double *d_pv, int64_t npv, double *d_z, int fp32_math,
                            cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const uint64_t off_b = ((uint64_t)sizeof(RRPvOrbit) * (uint64_t)npv + 255u) & ~(uint64_t)255u;
  const uint64_t need = off_b + (uint64_t)sizeof(RRPvBand) * (uint64_t)npv * (uint64_t)c.nkpb;
  if (npv > (1 << 24) || need > (uint64_t)RR_NOALLOC_SCRATCH_BYTES) return RR_ESCRATCH;
  int dev = -1;
  RR_CUDA(cudaGetDevice(&dev));
  if (!ctx->noalloc_scratch || dev != ctx->device) return RR_ESTATE;   // the address is per device
  RRPvOrbit *pvo = reinterpret_cast<RRPvOrbit *>(ctx->noalloc_scratch);
  RRPvBand *pvb = reinterpret_cast<RRPvBand *>(static_cast<unsigned char *>(ctx->noalloc_scratch) + off_b);
  const RRWork *wk = &ctx->work[0];                // table mode of the device-pointer API (k limits)
  const bool direct = wk->lazy == 2;
  rr_pv_prep_kernel<<<(unsigned)((npv + 127) / 128), 128, 0, st>>>(
      d_pv, npv, c.nkpb, c.nk, c.k0, c.k1, direct ? 1e-300 : c.k0, direct ? 1e300 : c.k1, c.ng,
      fp32_math != 0, ctx->mean_k, rr_row_pad(ctx, wk), pvo, pvb, nullptr);
  RR_LAUNCH_CHECK(ctx);
  const int64_t total = ctx->ntiles * npv;
  if (total <= 0) return RR_OK;
  const unsigned grid = rr_grid_for(total);
  const size_t smem = K_SMEM * 8 + 16 + 4 * RR_LENS_PITCH * 8;
  if (fp32_math)
    rr_orbit_kernel<float><<<grid, FT, smem, st>>>(ctx->d_times, ctx->d_tiles, ctx->d_lc, pvo,
                                                   ctx->ntiles, npv, ctx->nsub, d_z);
  else
    rr_orbit_kernel<double><<<grid, FT, smem, st>>>(ctx->d_times, ctx->d_tiles, ctx->d_lc, pvo,
                                                    ctx->ntiles, npv, ctx->nsub, d_z);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

// 1 if rr_dyn sits at shared::cta address RR_SMEM_ABS in a kernel without static shared memory
// (what the RR_SM_ABS kernels assume), 0 if not; < 0: error.  Synchronous; called by rr_create.
int rr_smem_probe(int *abs_ok) {
  unsigned *d = nullptr, h = 0;
  *abs_ok = 0;
  RR_CUDA(cudaMalloc(&d, sizeof(unsigned)));
  rr_smem_probe_kernel<<<1, 32, 256>>>(d);
  cudaError_t e = cudaMemcpy(&h, d, sizeof(unsigned), cudaMemcpyDeviceToHost);
  cudaFree(d);
  if (e != cudaSuccess) return RR_ECUDA_BASE - (int)e;
#ifndef RR_NO_SMEM_ABS
  *abs_ok = h == (unsigned)RR_SMEM_ABS;
#endif
  return RR_OK;
}

int rr_fma_peak_launch(int precision, double *h_fma_per_s, cudaStream_t st) {
  if (precision != RR_FP64) return fma_peak_typed<float>(h_fma_per_s, st);
  return fma_peak_typed<double>(h_fma_per_s, st);
}
