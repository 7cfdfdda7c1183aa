// rr_api.cu - the C-ABI of include/roadrunner.h: argument checks, buffer ownership, call order.
// Every step of the path runs in the kernels of rr_geometry.cu (a0), rr_ld_table.cu (kernel 1),
// rr_flux.cu (kernels 2+3) and rr_dispatch.cu (kernel 4); this file launches them.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "rr_common.cuh"

#ifndef RR_TILE_UNIT
#define RR_TILE_UNIT 1024  // measured: 1024 beats 512 by 0.5 % and 2048 by 0.7 % (with 128 waves)
#endif

namespace {

// element size of ldp, T, Istar, rows (fp32 in RR_FP32 and RR_MIXED) and of flux (fp32 in RR_FP32)
int esize(const rr_ctx *ctx) { return ctx->cfg.precision != RR_FP64 ? 4 : 8; }
int esize_flux(const rr_ctx *ctx) { return ctx->cfg.precision == RR_FP32 ? 4 : 8; }

void free_work(RRWork *w) {
  if (w->T) cudaFree(w->T);
  if (w->istar) cudaFree(w->istar);
  if (w->pvo) cudaFree(w->pvo);
  if (w->pvb) cudaFree(w->pvb);
  if (w->lens) cudaFree(w->lens);
  if (w->zpoly) cudaFree(w->zpoly);
  if (w->ldp) cudaFree(w->ldp);
  if (w->rows) cudaFree(w->rows);
  if (w->bk) cudaFree(w->bk);
  memset(w, 0, sizeof(*w));
  w->table_npv = -1;
}

void free_data(rr_ctx *ctx) {
  if (ctx->d_times) cudaFree(ctx->d_times);
  if (ctx->d_lc_index) cudaFree(ctx->d_lc_index);
  if (ctx->d_lc) cudaFree(ctx->d_lc);
  ctx->d_times = nullptr;
  ctx->d_lc_index = nullptr;
  ctx->d_lc = nullptr;
  ctx->npt = 0;
  ctx->nlc = 0;
  ctx->ntiles = -1;
  ctx->nsub = -1;
}

// Exposures per dispatch tile for a light curve with ns sub-samples: RR_TILE_UNIT x R, R chosen so
// that a tile carries about 4096 sub-samples.
int tile_len_for(int ns) {
  int r = (8 + ns / 2) / ns;
  r = std::max(1, std::min(8, r));
  return RR_TILE_UNIT * r;
}

// The lazy row builder keeps one profile (nz doubles) in shared memory.
bool lazy_ok(const rr_ctx *ctx) { return ctx->table_mode != RR_TABLE_FULL && ctx->nz <= 2000; }

int grow(void **p, int64_t *cap, int64_t need) {
  if (need <= *cap) return RR_OK;
  if (*p) cudaFree(*p);
  *p = nullptr;
  *cap = 0;
  if (cudaMalloc(p, (size_t)need) != cudaSuccess) {
    cudaGetLastError();
    return RR_EALLOC;
  }
  *cap = need;
  return RR_OK;
}

}  // namespace

extern "C" {

const char *rr_error_string(int code) {
  switch (code) {
    case RR_OK: return "ok";
    case RR_ENULL: return "a required pointer is NULL";
    case RR_ECONFIG: return "rr_config out of range";
    case RR_ESIZE: return "a size is <= 0 or inconsistent";
    case RR_EINDEX: return "lc_index / passband_index / supersampling / exposure_time out of range";
    case RR_ESTATE: return "call order: set_data / build_ld_table first, with the same npv";
    case RR_EALLOC: return "allocation failed";
    case RR_ESCRATCH:
      return "problem too large for the static scratch of the allocation-free entry point "
             "(RR_NOALLOC_SCRATCH_BYTES): use rr_orbit_z";
    default: break;
  }
  if (code <= RR_ECUDA_BASE) return cudaGetErrorString((cudaError_t)(RR_ECUDA_BASE - code));
  return "unknown error";
}

int rr_create(const rr_config *cfg, rr_ctx **out) {
  if (!cfg || !out) return RR_ENULL;
  *out = nullptr;
  if (cfg->nzin < 1 || cfg->nzlimb < 1 || !(cfg->zcut > 0.0 && cfg->zcut < 1.0) || cfg->ng < 2 ||
      cfg->nk < 2 || !(cfg->k0 > 0.0) || !(cfg->k1 > cfg->k0) || !isfinite(cfg->k1) ||
      cfg->npb < 1 || (cfg->nkpb != 1 && cfg->nkpb != cfg->npb) ||
      (cfg->precision != RR_FP64 && cfg->precision != RR_FP32 && cfg->precision != RR_MIXED) ||
      (int64_t)cfg->nzin + cfg->nzlimb > 100000 || cfg->ng > 5600 ||
      (int64_t)cfg->nk * cfg->ng > 0x7fffffffLL / 2)
    return RR_ECONFIG;
  rr_ctx *ctx = new (std::nothrow) rr_ctx();
  if (!ctx) return RR_EALLOC;
  ctx->cfg = *cfg;
  ctx->nz = cfg->nzin + cfg->nzlimb;
  ctx->ntiles = -1;
  ctx->nsub = -1;
  for (auto &w : ctx->work) w.table_npv = -1;
  ctx->reduction = RR_REDUCE_AUTO;
  ctx->table_mode = RR_TABLE_LAZY;
  ctx->orbit_poly = 1;
  ctx->lens_poly = 1;
  int rc = RR_OK;
  cudaError_t e = cudaGetDevice(&ctx->device);
  if (e == cudaSuccess)
    e = cudaDeviceGetAttribute(&ctx->sm_count, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_counters, sizeof(unsigned long long) * 16);
  if (e == cudaSuccess) e = cudaMemset(ctx->d_counters, 0, sizeof(unsigned long long) * 16);
  if (e != cudaSuccess) rc = RR_ECUDA_BASE - (int)e;
  if (rc == RR_OK) rc = rr_smem_probe(&ctx->smem_abs);
  if (rc == RR_OK) rc = rr_noalloc_setup(ctx);   // address of the no-alloc scratch on this device
  if (rc == RR_OK) rc = rr_geometry_build(ctx);
  if (rc != RR_OK) {
    cudaGetLastError();
    rr_destroy(ctx);
    return rc;
  }
  *out = ctx;
  return RR_OK;
}

int rr_destroy(rr_ctx *ctx) {
  if (!ctx) return RR_ENULL;
  cudaDeviceSynchronize();
  for (auto e : ctx->tev) cudaEventDestroy(e);
  ctx->tev.clear();
  free_data(ctx);
  for (auto &w : ctx->work) free_work(&w);
  void *bufs[] = {ctx->d_ze, ctx->d_zm, ctx->d_mu, ctx->d_q, ctx->d_W, ctx->d_Wsup, ctx->d_tiles,
                  ctx->d_scratch, ctx->d_counters};
  for (void *b : bufs)
    if (b) cudaFree(b);
  for (int s = 0; s < 2; ++s) {
    for (int q = 0; q < 4; ++q)
      if (ctx->d_host_stage[s][q]) cudaFree(ctx->d_host_stage[s][q]);
    if (ctx->hs[s]) cudaStreamDestroy(ctx->hs[s]);
    if (ctx->hev[s]) cudaEventDestroy(ctx->hev[s]);
  }
  cudaGetLastError();
  delete ctx;
  return RR_OK;
}

int rr_get_mu(const rr_ctx *ctx, double *h_mu) {
  if (!ctx || !h_mu) return RR_ENULL;
  memcpy(h_mu, ctx->h_mu.data(), sizeof(double) * ctx->nz);
  return RR_OK;
}

int rr_get_ze(const rr_ctx *ctx, double *h_ze) {
  if (!ctx || !h_ze) return RR_ENULL;
  memcpy(h_ze, ctx->h_ze.data(), sizeof(double) * (ctx->nz + 1));
  return RR_OK;
}

int rr_get_weights(const rr_ctx *ctx, double *h_W) {
  if (!ctx || !h_W) return RR_ENULL;
  size_t n = (size_t)ctx->cfg.nk * ctx->cfg.ng * ctx->nz;
  RR_CUDA(cudaMemcpy(h_W, ctx->d_W, sizeof(double) * n, cudaMemcpyDeviceToHost));
  return RR_OK;
}

int rr_set_reduction(rr_ctx *ctx, int32_t mode) {
  if (!ctx) return RR_ENULL;
  if (mode < RR_REDUCE_AUTO || mode > RR_REDUCE_SHUFFLE) return RR_ECONFIG;
  ctx->reduction = mode;
  return RR_OK;
}

int rr_set_data(rr_ctx *ctx, const double *d_times, const int32_t *d_lc_index, int64_t npt,
                const int32_t *h_passband_index, const int32_t *h_supersampling,
                const double *h_exposure_time, int32_t nlc, void *stream) {
  if (!ctx || !d_times || !d_lc_index || !h_passband_index || !h_supersampling ||
      !h_exposure_time)
    return RR_ENULL;
  if (npt <= 0 || npt > 0x7fffffffLL || nlc <= 0) return RR_ESIZE;
  std::vector<RRLc> lcs((size_t)nlc);
  for (int l = 0; l < nlc; ++l) {
    if (h_passband_index[l] < 0 || h_passband_index[l] >= ctx->cfg.npb) return RR_EINDEX;
    if (h_supersampling[l] < 1 || h_supersampling[l] > (1 << 20)) return RR_EINDEX;
    if (!(h_exposure_time[l] >= 0.0) || !isfinite(h_exposure_time[l])) return RR_EINDEX;
    lcs[l].exptime = h_exposure_time[l];
    lcs[l].ns = h_supersampling[l];
    lcs[l].pb = h_passband_index[l];
    lcs[l].tile_len = tile_len_for(h_supersampling[l]);
    lcs[l].pad = 0;
  }
  cudaStream_t st = (cudaStream_t)stream;
  free_data(ctx);
  cudaError_t e = cudaMalloc(&ctx->d_times, sizeof(double) * npt);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_lc_index, sizeof(int32_t) * npt);
  if (e == cudaSuccess) e = cudaMalloc(&ctx->d_lc, sizeof(RRLc) * nlc);
  if (e != cudaSuccess) {
    cudaGetLastError();
    free_data(ctx);
    return RR_EALLOC;
  }
  ctx->npt = npt;
  ctx->nlc = nlc;
  ctx->h_lc = lcs;
  int rc = RR_OK;
  e = cudaMemcpyAsync(ctx->d_times, d_times, sizeof(double) * npt, cudaMemcpyDeviceToDevice, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(ctx->d_lc_index, d_lc_index, sizeof(int32_t) * npt,
                        cudaMemcpyDeviceToDevice, st);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(ctx->d_lc, ctx->h_lc.data(), sizeof(RRLc) * nlc, cudaMemcpyHostToDevice,
                        st);
  if (e != cudaSuccess) rc = RR_ECUDA_BASE - (int)e;
  if (rc == RR_OK) rc = rr_dispatch_build(ctx, st);
  if (rc != RR_OK) {
    cudaStreamSynchronize(st);
    free_data(ctx);
  }
  return rc;
}

int rr_build_ld_table(rr_ctx *ctx, const void *d_ldp, const void *d_istar, int64_t npv,
                      void *stream) {
  if (!ctx || !d_ldp) return RR_ENULL;
  if (npv <= 0) return RR_ESIZE;
  if (lazy_ok(ctx))
    return rr_ld_profile_launch(ctx, &ctx->work[0], d_ldp, d_istar, npv, 1, (cudaStream_t)stream);
  return rr_ld_table_launch(ctx, &ctx->work[0], d_ldp, d_istar, npv, (cudaStream_t)stream);
}

int rr_build_ld_table_law(rr_ctx *ctx, int32_t law, const double *d_ldc, int32_t nldc, int64_t npv,
                          void *stream) {
  if (!ctx || (!d_ldc && law != RR_LD_UNIFORM)) return RR_ENULL;
  if (npv <= 0) return RR_ESIZE;
  static const int need[] = {0, 1, 2, 2, -1, 4, 2, 2, 2, 2};
  if (law < RR_LD_UNIFORM || law > RR_LD_POWER2_PM) return RR_ECONFIG;
  if (need[law] >= 0 ? nldc != need[law] : (nldc < 1 || nldc > 64)) return RR_ESIZE;
  return rr_ld_law_launch(ctx, &ctx->work[0], law, d_ldc, nldc, npv, (cudaStream_t)stream);
}

int rr_set_small_planet(rr_ctx *ctx, double k_threshold) {
  if (!ctx) return RR_ENULL;
  if (!(k_threshold >= 0.0) || !isfinite(k_threshold)) return RR_ECONFIG;
  ctx->k_small = k_threshold;
  return RR_OK;
}

int rr_set_mean_k_weights(rr_ctx *ctx, int32_t on) {
  if (!ctx) return RR_ENULL;
  ctx->mean_k = on ? 1 : 0;
  return RR_OK;
}

int rr_set_orbit_poly(rr_ctx *ctx, int32_t on) {
  if (!ctx) return RR_ENULL;
  ctx->orbit_poly = on ? 1 : 0;
  return RR_OK;
}

int rr_set_lens_poly(rr_ctx *ctx, int32_t on) {
  if (!ctx) return RR_ENULL;
  ctx->lens_poly = on ? 1 : 0;
  return RR_OK;
}

int rr_set_table_mode(rr_ctx *ctx, int32_t mode) {
  if (!ctx) return RR_ENULL;
  if (mode != RR_TABLE_LAZY && mode != RR_TABLE_FULL && mode != RR_TABLE_DIRECT) return RR_ECONFIG;
  if (mode == RR_TABLE_DIRECT && ctx->nz > 2000) return RR_ECONFIG;
  ctx->table_mode = mode;
  return RR_OK;
}

const void *rr_table_ptr(rr_ctx *ctx) {
  if (!ctx || ctx->work[0].table_npv <= 0) return nullptr;
  // the profile copy of rr_build_ld_table was queued on the caller's stream, which the legacy
  // stream used below does not order with
  if (cudaDeviceSynchronize() != cudaSuccess) return nullptr;
  if (rr_ld_full_from_profile(ctx, &ctx->work[0], nullptr) != RR_OK) return nullptr;
  if (cudaDeviceSynchronize() != cudaSuccess) return nullptr;
  return ctx->work[0].T;
}

const void *rr_istar_ptr(const rr_ctx *ctx) {
  return (ctx && ctx->work[0].table_npv > 0) ? ctx->work[0].istar : nullptr;
}

int rr_get_table(rr_ctx *ctx, void *h_T, void *h_istar) {
  if (!ctx) return RR_ENULL;
  RRWork &w = ctx->work[0];
  if (w.table_npv <= 0) return RR_ESTATE;
  RR_CUDA(cudaDeviceSynchronize());
  if (h_T) {
    int rc = rr_ld_full_from_profile(ctx, &w, nullptr);
    if (rc != RR_OK) return rc;
    RR_CUDA(cudaDeviceSynchronize());
  }
  const size_t rows = (size_t)w.table_npv * ctx->cfg.npb, es = (size_t)esize(ctx);
  if (h_T)
    RR_CUDA(cudaMemcpy(h_T, w.T, rows * ctx->cfg.nk * ctx->cfg.ng * es, cudaMemcpyDeviceToHost));
  if (h_istar) RR_CUDA(cudaMemcpy(h_istar, w.istar, rows * es, cudaMemcpyDeviceToHost));
  return RR_OK;
}

int rr_get_rows(const rr_ctx *ctx, void *h_rows) {
  if (!ctx || !h_rows) return RR_ENULL;
  const RRWork &w = ctx->work[0];
  if (w.table_npv <= 0 || !w.lazy || !w.rows) return RR_ESTATE;
  RR_CUDA(cudaDeviceSynchronize());
  RR_CUDA(cudaMemcpy(h_rows, w.rows, (size_t)w.table_npv * ctx->cfg.npb * ctx->cfg.ng * esize(ctx),
                     cudaMemcpyDeviceToHost));
  return RR_OK;
}

int rr_evaluate(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, void *d_flux,
                int32_t *d_status, void *stream) {
  if (!ctx || !d_pv || !d_flux) return RR_ENULL;
  if (npv <= 0 || npar != ctx->cfg.nkpb + 6) return RR_ESIZE;
  if (ctx->ntiles < 0 || ctx->work[0].table_npv != npv) return RR_ESTATE;
  if (ctx->k_small > 0.0 && !ctx->work[0].lazy) return RR_ESTATE;   // needs the row builders
  cudaStream_t st = (cudaStream_t)stream;
  int rc = rr_pv_prep_launch(ctx, &ctx->work[0], d_pv, npv, d_status,
                             ctx->cfg.precision != RR_FP64, st);
  if (rc != RR_OK) return rc;
  // Kernel timing: a triple of events (before rows, before flux, after flux) joins ctx->tev only
  // when all three were recorded; any failure destroys them here.
  cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
  bool timed = ctx->timing_on && ctx->tev.size() < 3 * 4096;
  if (timed)
    for (auto &e : ev)
      if (cudaEventCreate(&e) != cudaSuccess) { cudaGetLastError(); e = nullptr; timed = false; }
  cudaError_t ce = cudaSuccess;
  if (timed) ce = cudaEventRecord(ev[0], st);
  if (ce == cudaSuccess && ctx->work[0].lazy) rc = rr_ld_rows_launch(ctx, &ctx->work[0], npv, st);
  if (ce == cudaSuccess && rc == RR_OK && ctx->work[0].lazy && ctx->k_small > 0.0)
    rc = rr_ld_rows_small_launch(ctx, &ctx->work[0], npv, st);
  if (ce == cudaSuccess && rc == RR_OK && timed) ce = cudaEventRecord(ev[1], st);
  if (ce == cudaSuccess && rc == RR_OK) rc = rr_flux_launch(ctx, &ctx->work[0], npv, d_flux, st);
  if (ce == cudaSuccess && rc == RR_OK && timed) ce = cudaEventRecord(ev[2], st);
  if (ce != cudaSuccess && rc == RR_OK) rc = RR_ECUDA_BASE - (int)ce;
  if (timed && rc == RR_OK) {
    for (auto e : ev) ctx->tev.push_back(e);
  } else {
    for (auto e : ev)
      if (e) cudaEventDestroy(e);
  }
  return rc;
}

int rr_evaluate_flat(rr_ctx *ctx, const double *d_times, const int32_t *d_lc_index, int64_t npt,
                     const int32_t *h_passband_index, const int32_t *h_supersampling,
                     const double *h_exposure_time, int32_t nlc, const double *d_pv, int32_t npar,
                     int64_t npv, void *d_flux, int32_t *d_status, void *stream) {
  int rc = rr_set_data(ctx, d_times, d_lc_index, npt, h_passband_index, h_supersampling,
                       h_exposure_time, nlc, stream);
  if (rc != RR_OK) return rc;
  return rr_evaluate(ctx, d_pv, npar, npv, d_flux, d_status, stream);
}

int rr_orbit_z(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, double *d_z,
               int32_t fp32_math, void *stream) {
  if (!ctx || !d_pv || !d_z) return RR_ENULL;
  if (npv <= 0 || npar != ctx->cfg.nkpb + 6) return RR_ESIZE;
  if (ctx->ntiles < 0) return RR_ESTATE;
  cudaStream_t st = (cudaStream_t)stream;
  int rc = rr_pv_prep_launch(ctx, &ctx->work[0], d_pv, npv, nullptr, fp32_math != 0, st);
  if (rc != RR_OK) return rc;
  return rr_orbit_launch(ctx, &ctx->work[0], npv, d_z, fp32_math, st);
}

int rr_orbit_z_noalloc(rr_ctx *ctx, const double *d_pv, int32_t npar, int64_t npv, double *d_z,
                       int32_t fp32_math, void *stream) {
  if (!ctx || !d_pv || !d_z) return RR_ENULL;
  if (npv <= 0 || npar != ctx->cfg.nkpb + 6) return RR_ESIZE;
  if (ctx->ntiles < 0) return RR_ESTATE;
  return rr_orbit_noalloc_launch(ctx, d_pv, npv, d_z, fp32_math, (cudaStream_t)stream);
}

int64_t rr_num_subsamples(const rr_ctx *ctx) { return ctx ? ctx->nsub : -1; }
int64_t rr_num_tiles(const rr_ctx *ctx) { return ctx ? ctx->ntiles : -1; }

int rr_get_tiles(const rr_ctx *ctx, int32_t *h_start, int32_t *h_count, int32_t *h_lc,
                 double *h_tmin, double *h_tmax) {
  if (!ctx) return RR_ENULL;
  if (ctx->ntiles < 0) return RR_ESTATE;
  std::vector<RRTile> t((size_t)ctx->ntiles);
  RR_CUDA(cudaMemcpy(t.data(), ctx->d_tiles, sizeof(RRTile) * t.size(), cudaMemcpyDeviceToHost));
  for (size_t i = 0; i < t.size(); ++i) {
    if (h_start) h_start[i] = t[i].start;
    if (h_count) h_count[i] = t[i].count;
    if (h_lc) h_lc[i] = t[i].lc;
    if (h_tmin) h_tmin[i] = t[i].tmin;
    if (h_tmax) h_tmax[i] = t[i].tmax;
  }
  return RR_OK;
}

// Whole step from host buffers: chunks of parameter vectors, two streams, so that the copies of
// one chunk overlap the kernels of the other.
int rr_evaluate_host(rr_ctx *ctx, const void *h_ldp, const double *h_pv, int32_t npar, int64_t npv,
                     void *h_flux, int32_t *h_status) {
  if (!ctx || !h_ldp || !h_pv || !h_flux) return RR_ENULL;
  if (npv <= 0 || npar != ctx->cfg.nkpb + 6) return RR_ESIZE;
  if (ctx->ntiles < 0) return RR_ESTATE;
  if (ctx->k_small > 0.0 && !lazy_ok(ctx)) return RR_ESTATE;   // needs the row builders
  const rr_config &c = ctx->cfg;
  const int64_t es = esize(ctx), esf = esize_flux(ctx);
  for (int s = 0; s < 2; ++s) {
    if (!ctx->hs[s]) RR_CUDA(cudaStreamCreateWithFlags(&ctx->hs[s], cudaStreamNonBlocking));
    if (!ctx->hev[s]) RR_CUDA(cudaEventCreateWithFlags(&ctx->hev[s], cudaEventDisableTiming));
  }
  // chunk: about 256 MB of flux, at least 1 pv
  int64_t chunk = (256LL << 20) / (ctx->npt * esf);
  chunk = std::max<int64_t>(1, std::min(chunk, npv));
  if (chunk > 64) chunk = (chunk / 64) * 64;
  const int64_t ldp_row = (int64_t)c.npb * ctx->nz * es, pv_row = (int64_t)npar * 8,
                flux_row = ctx->npt * esf;
  int rc = RR_OK;
  int64_t n_chunks = (npv + chunk - 1) / chunk;
  for (int64_t ci = 0; ci < n_chunks && rc == RR_OK; ++ci) {
    const int s = (int)(ci & 1);
    const int64_t v0 = ci * chunk, nv = std::min(chunk, npv - v0);
    cudaStream_t st = ctx->hs[s];
    // the slot's previous chunk must have left its staging buffers (same stream: ordered)
    if ((rc = grow(&ctx->d_host_stage[s][0], &ctx->host_stage_cap[s][0], chunk * ldp_row)) ||
        (rc = grow(&ctx->d_host_stage[s][1], &ctx->host_stage_cap[s][1], chunk * pv_row)) ||
        (rc = grow(&ctx->d_host_stage[s][2], &ctx->host_stage_cap[s][2], chunk * flux_row)) ||
        (rc = grow(&ctx->d_host_stage[s][3], &ctx->host_stage_cap[s][3], chunk * 4)))
      break;
    void *d_ldp = ctx->d_host_stage[s][0];
    double *d_pv = (double *)ctx->d_host_stage[s][1];
    void *d_flux = ctx->d_host_stage[s][2];
    int32_t *d_status = (int32_t *)ctx->d_host_stage[s][3];
    // (no early return from here on: copies and kernels of the other slot may still be in flight
    // against the caller's host buffers, and the epilogue below waits for both streams)
    cudaError_t ce = cudaMemcpyAsync(d_ldp, (const char *)h_ldp + v0 * ldp_row, nv * ldp_row,
                                     cudaMemcpyHostToDevice, st);
    if (ce == cudaSuccess)
      ce = cudaMemcpyAsync(d_pv, (const char *)h_pv + v0 * pv_row, nv * pv_row,
                           cudaMemcpyHostToDevice, st);
    if (ce != cudaSuccess) { rc = RR_ECUDA_BASE - (int)ce; break; }
    RRWork *wk = &ctx->work[1 + s];
    if (lazy_ok(ctx)) {   // the staging buffer lives until this chunk's kernels are done
      if ((rc = rr_ld_profile_launch(ctx, wk, d_ldp, nullptr, nv, 0, st)) != RR_OK) break;
    } else if ((rc = rr_ld_table_launch(ctx, wk, d_ldp, nullptr, nv, st)) != RR_OK) {
      break;
    }
    if ((rc = rr_pv_prep_launch(ctx, wk, d_pv, nv, d_status, ctx->cfg.precision != RR_FP64, st)) != RR_OK) break;
    if (wk->lazy && (rc = rr_ld_rows_launch(ctx, wk, nv, st)) != RR_OK) break;
    if (wk->lazy && ctx->k_small > 0.0 && (rc = rr_ld_rows_small_launch(ctx, wk, nv, st)) != RR_OK)
      break;
    if ((rc = rr_flux_launch(ctx, wk, nv, d_flux, st)) != RR_OK) break;
    ce = cudaMemcpyAsync((char *)h_flux + v0 * flux_row, d_flux, nv * flux_row,
                         cudaMemcpyDeviceToHost, st);
    if (ce == cudaSuccess && h_status)
      ce = cudaMemcpyAsync(h_status + v0, d_status, nv * 4, cudaMemcpyDeviceToHost, st);
    if (ce != cudaSuccess) { rc = RR_ECUDA_BASE - (int)ce; break; }
  }
  for (int s = 0; s < 2; ++s) {
    cudaError_t e = cudaStreamSynchronize(ctx->hs[s]);
    if (e != cudaSuccess && rc == RR_OK) rc = RR_ECUDA_BASE - (int)e;
  }
  return rc;
}

int rr_enable_counters(rr_ctx *ctx, int32_t on) {
  if (!ctx) return RR_ENULL;
  ctx->counters_on = on ? 1 : 0;
  return RR_OK;
}

int rr_get_counters(const rr_ctx *ctx, int64_t *h_counts) {
  if (!ctx || !h_counts) return RR_ENULL;
  RR_CUDA(cudaDeviceSynchronize());
  RR_CUDA(cudaMemcpy(h_counts, ctx->d_counters, sizeof(int64_t) * 9, cudaMemcpyDeviceToHost));
  return RR_OK;
}

int64_t rr_launch_count(const rr_ctx *ctx) { return ctx ? ctx->launches : -1; }

int rr_enable_kernel_timing(rr_ctx *ctx, int32_t on) {
  if (!ctx) return RR_ENULL;
  ctx->timing_on = on ? 1 : 0;
  return RR_OK;
}

int rr_get_kernel_times(rr_ctx *ctx, double *h_ms, int64_t *h_calls) {
  if (!ctx || !h_ms || !h_calls) return RR_ENULL;
  h_ms[0] = h_ms[1] = 0.0;
  *h_calls = 0;
  int rc = RR_OK;
  for (size_t i = 0; i + 2 < ctx->tev.size(); i += 3) {
    cudaEvent_t *e = &ctx->tev[i];
    float a = 0.f, b = 0.f;
    cudaError_t err = cudaEventSynchronize(e[2]);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&a, e[0], e[1]);
    if (err == cudaSuccess) err = cudaEventElapsedTime(&b, e[1], e[2]);
    if (err == cudaSuccess) {
      h_ms[0] += a;
      h_ms[1] += b;
      ++*h_calls;
    } else if (rc == RR_OK) {
      rc = RR_ECUDA_BASE - (int)err;
    }
    for (int q = 0; q < 3; ++q) cudaEventDestroy(e[q]);
  }
  ctx->tev.clear();
  return rc;
}

int rr_math_probe(int32_t op, int32_t fp32_math, const double *d_a, const double *d_b, int64_t n,
                  double *d_out0, double *d_out1, void *stream) {
  if (!d_a || !d_out0) return RR_ENULL;
  if (op < RR_PROBE_SQRT3 || op > RR_PROBE_CELL) return RR_ECONFIG;
  const bool two = op == RR_PROBE_DIV3 || op == RR_PROBE_ATAN_QUADRANT || op == RR_PROBE_ATAN2_POS;
  if (two && !d_b) return RR_ENULL;
  if (n <= 0) return RR_ESIZE;
  return rr_math_probe_launch(op, fp32_math != 0, d_a, two ? d_b : nullptr, n, d_out0, d_out1,
                              (cudaStream_t)stream);
}

int rr_measure_fma_peak(int32_t precision, double *h_fma_per_s, void *stream) {
  if (!h_fma_per_s) return RR_ENULL;
  if (precision != RR_FP64 && precision != RR_FP32 && precision != RR_MIXED) return RR_ECONFIG;
  return rr_fma_peak_launch(precision, h_fma_per_s, (cudaStream_t)stream);
}

}  // extern "C"
