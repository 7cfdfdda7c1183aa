// rr_common.cuh - shared declarations of the CUDA library (product code; no oracle code here).
// Method: H. Parviainen, arXiv:2009.08500 (citations: PAPER.md lines).  Layout: DESIGN.md s5.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/roadrunner.h"

#define RR_PI 3.14159265358979323846264338327950288
#define RR_TWOPI 6.28318530717958647692528676655900577

// ---- device-resident descriptors -----------------------------------------------------------
// Per light curve (kernel 4 input): PAPER.md:230-236.
struct RRLc {
  double exptime;    // exposure time tau (days)
  int32_t ns;        // sub-samples per exposure
  int32_t pb;        // passband
  int32_t tile_len;  // exposures per dispatch tile
  int32_t pad;
};

// One dispatch tile (kernel 4 output): a run of exposures of ONE light curve.
struct RRTile {
  double tmin, tmax;  // range of the mid-exposure times in the tile
  int64_t sub_off;    // index of the tile's first sub-sample in a [nsub] row (rr_orbit_z)
  int32_t start;      // first exposure
  int32_t count;      // exposures in the tile
  int32_t lc;         // light curve
  int32_t pad;
};

// Per parameter vector, orbit part (kernel 2's per-pv work, done once per rr_evaluate by
// rr_pv_prep_kernel).  Phases u are in turns of the orbit relative to t0; E_tr is the eccentric
// anomaly at inferior conjunction (true anomaly pi/2 - w, reading R8); d = E - E_tr.
struct RRPvOrbit {
  double t0, inv_p;
  double u_mid, hwid;   // transit window [u_mid - hwid, u_mid + hwid]: z < 1+k in front of the
                        // star is only possible inside it (hwid = 1/2: no window, whole orbit)
  double zc0, zc1;      // circular: z^2 = zc0 + zc1 sin^2(2 pi u) = a^2 cos^2 i, a^2 sin^2 i
  double e, sE, cE;     // e, sin E_tr, cos E_tr (robust solver path)
  double A, B, C;       // Kepler's equation in d: derivatives at d = 0: 1 - e cE, e sE, e cE
  double invA, c2, c3, c4;  // starter: series reversion d0 = y(1 + y(c2 + y(c3 + y c4))), y = dM/A
  double tol;           // accept the single Halley step when |step| <= tol
  double X1, X2;        // sky x (units of R*) = X1 (cos d - 1) + X2 sin d
  double Y0, Y1, Y2;    // line-of-sight-projected y / a = Y0 + Y1 (cos d - 1) + Y2 sin d; front: > 0
  double aci2;          // a^2 cos^2 i:  z^2 = x^2 + aci2 y^2
  int32_t status;       // RR_PV_* bits; != 0 -> NaN row
  int32_t circular;     // e == 0
  int32_t zpoly_ok;     // 1: z^2 over the transit window from the fitted polynomials (rr_zpoly_fit)
  int32_t pad;
};

// Per (parameter vector, k-band): radius-ratio constants.
struct RRPvBand {
  double k, opk;       // k, 1+k
  double omk;          // |1-k|: z <= omk -> full overlap
  double afull;        // pi * min(1,k)^2
  double k2;           // k^2
  double gscale;       // (ng-1)/(1+k): y = z*gscale is the g coordinate in table cells
  double ak;           // weight of table row ik+1
  double kw;           // radius ratio the LD weights are taken at: k, or the mean of the pv's k over
                       // the passbands (transmission-spectroscopy shortcut)
  int32_t ik;          // lower k row of kw, clamped to nk-2 (reading R10)
  int32_t lens_ok;     // 1: the polynomial form of the lens area holds for this k (rr_lens_fit)
};

// Per-evaluation device buffers: one set for the device-pointer API, one per slot of the
// host-buffer path (so that two chunks can be in flight on two streams).
struct RRWork {
  void *T, *istar;          // kernel 1 output (ctx precision)
  int64_t table_npv;        // npv of the table / profile set last; -1 = none
  int64_t T_cap, istar_cap; // bytes
  // lazy table mode (RR_TABLE_LAZY): the profile is kept and rr_evaluate builds, for every
  // (pv, passband), only the k-collapsed row its k needs
  void *ldp;                // owned copy of the caller's ldp (device API)
  int64_t ldp_cap;
  const void *ldp_src;      // profile the row builder reads: ldp, or the host path's staging
  void *rows;               // ldw[npv][npb][ng], ctx precision
  int64_t rows_cap;
  int32_t *bk;              // row buckets by ik: hist[nk] | cursor[nk] | offs[nk+1] | tileoff[nk+1] | list[M]
  int64_t bk_cap;
  int32_t lazy;             // 0: evaluate from T; 1: from lazy rows; 2: from direct-model rows
  int32_t have_full;        // T holds the full table of the current profile
  RRPvOrbit *pvo;
  RRPvBand *pvb;
  double *lens;             // [npv][nkpb][2][RR_LENS_PITCH]: lens-area polynomials (fp64 kernel)
  double *zpoly;            // [npv][2][RR_LENS_PITCH]: z^2 over the two halves of the transit window
  int64_t pv_cap;
};
#define RR_LENS_PITCH 14    // 13 coefficients + 1 pad: 16-byte multiples per half
#define RR_LENS_KMAX 0.32   // radius ratios up to here take the polynomial form (error <= 2e-13)

// ---- host context -----------------------------------------------------------------------------
struct rr_ctx {
  rr_config cfg;
  int nz;
  int device;
  int sm_count;
  int smem_abs;         // 1: the flux kernels may address shared memory absolutely (rr_smem_probe)
  void *noalloc_scratch; // device address of the static scratch of rr_orbit_z_noalloc on ctx's device
  // geometry (a0)
  double *d_ze, *d_zm, *d_mu, *d_q, *d_W;
  void *d_Wsup;         // int2 [nk][ng]: non-zero range [jlo, jhi) of every weight row
  std::vector<double> h_ze, h_mu;
  // data (kernel 4)
  int64_t npt;
  int32_t nlc;
  double *d_times;
  int32_t *d_lc_index;
  RRLc *d_lc;
  std::vector<RRLc> h_lc;
  RRTile *d_tiles;
  int64_t ntiles, tiles_cap;
  int64_t nsub;
  int64_t *d_scratch;   // dispatch scratch
  int64_t scratch_cap;
  int32_t reduction;
  int32_t table_mode;   // RR_TABLE_LAZY | RR_TABLE_FULL | RR_TABLE_DIRECT
  int32_t mean_k;       // 1: LD weights at the mean k of the passbands
  int32_t orbit_poly;   // 1 (default): z^2 of eccentric pvs from per-pv polynomials where they hold
  int32_t lens_poly;    // 1 (default): lens area between the contacts from per-pv polynomials
  double k_small;       // small-planet approximation for kw <= k_small; 0: off
  // table (kernel 1) and per-pv prep: [0] device API, [1],[2] host-path slots
  RRWork work[3];
  // counters / accounting
  unsigned long long *d_counters;
  int32_t counters_on;
  int64_t launches;
  // per-kernel device timing of rr_evaluate (rr_enable_kernel_timing): event triples
  // (before rows, before flux, after flux) of the calls since the last read
  int32_t timing_on;
  std::vector<cudaEvent_t> tev;
  // host path
  cudaStream_t hs[2];
  cudaEvent_t hev[2];
  void *d_host_stage[2][4];   // per slot: ldp, pv, flux, status
  int64_t host_stage_cap[2][4];
};

// ---- error plumbing -----------------------------------------------------------------------------
#define RR_CUDA(call)                                          \
  do {                                                         \
    cudaError_t _e = (call);                                   \
    if (_e != cudaSuccess) return RR_ECUDA_BASE - (int)_e;     \
  } while (0)

#define RR_LAUNCH_CHECK(ctx)                                   \
  do {                                                         \
    (ctx)->launches++;                                         \
    cudaError_t _e = cudaGetLastError();                       \
    if (_e != cudaSuccess) return RR_ECUDA_BASE - (int)_e;     \
  } while (0)

// ---- internal entry points of the kernel files ---------------------------------------------------
int rr_geometry_build(rr_ctx *ctx);                                            // rr_geometry.cu
int rr_ld_table_launch(rr_ctx *ctx, RRWork *wk, const void *d_ldp,             // rr_ld_table.cu
                       const void *d_istar, int64_t npv, cudaStream_t st);
int rr_ld_profile_launch(rr_ctx *ctx, RRWork *wk, const void *d_ldp, const void *d_istar,
                         int64_t npv, int copy, cudaStream_t st);              // rr_ld_table.cu
int rr_ld_rows_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st);  // rr_ld_table.cu
int rr_ld_full_from_profile(rr_ctx *ctx, RRWork *wk, cudaStream_t st);         // rr_ld_table.cu
int rr_ld_law_launch(rr_ctx *ctx, RRWork *wk, int law, const double *d_ldc, int nc, int64_t npv,
                     cudaStream_t st);                                         // rr_ld_table.cu
int rr_ld_rows_direct_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st);  // rr_geometry.cu
int rr_ld_rows_small_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st);   // rr_geometry.cu
int rr_dispatch_build(rr_ctx *ctx, cudaStream_t st);                           // rr_dispatch.cu
int rr_pv_prep_launch(rr_ctx *ctx, RRWork *wk, const double *d_pv, int64_t npv,
                      int32_t *d_status, int fp32_tol, cudaStream_t st);       // rr_flux.cu
int rr_flux_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, void *d_flux, cudaStream_t st);
int rr_orbit_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, double *d_z, int fp32_math,
                    cudaStream_t st);
int rr_fma_peak_launch(int precision, double *h_fma_per_s, cudaStream_t st);   // rr_flux.cu
int rr_smem_probe(int *abs_ok);                                                // rr_flux.cu
int rr_noalloc_setup(rr_ctx *ctx);                                             // rr_flux.cu
int rr_orbit_noalloc_launch(rr_ctx *ctx, const double *d_pv, int64_t npv, double *d_z,
                            int fp32_math, cudaStream_t st);                   // rr_flux.cu
int rr_math_probe_launch(int op, int fp32, const double *d_a, const double *d_b, int64_t n,
                         double *d_o0, double *d_o1, cudaStream_t st);         // rr_flux.cu
