// rr_dispatch.cu - kernel 4: heterogeneous-light-curve dispatch.
// The exposure axis (times[npt] tagged with lc_index[npt]) is cut on the device into tiles that
// each hold exposures of ONE light curve, so that a thread block of the flux kernel sees one
// supersampling factor, one exposure time and one passband (reading R11: passband per light curve)
// and no warp diverges on ns.  Tile length depends on the light curve's ns so that tiles carry
// comparable work.  Each tile also gets its [tmin, tmax] time range (lets the flux kernel fill a
// whole out-of-transit tile without evaluating it) and the offset of its first sub-sample.
//
//   1. rr_k4_heads_*    heads of runs of equal lc_index (any order of light curves is allowed;
//                       a light curve may come in several runs), range check of lc_index
//   2. rr_k4_tilecount  tiles per run, exclusive scan -> first tile of every run
//   3. rr_k4_tiles      one thread per tile: binary search of its run, start/count/lc
//   4. rr_k4_ranges     one warp per tile: min/max time; then scan of count*ns -> sub_off
// The scans over runs and tiles (few) run in a single block (chunked, carry in shared memory); the
// walk over the exposures uses the whole GPU.
#include "rr_common.cuh"

namespace {

constexpr int SCAN_T = 1024;

// Block-wide inclusive scan of one value per thread (SCAN_T threads); returns the inclusive prefix,
// *total gets the block total.
__device__ int64_t block_inclusive_scan(int64_t v, int64_t *warp_sums, int64_t *total) {
  int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    int64_t n = __shfl_up_sync(0xffffffffu, v, o);
    if (lane >= o) v += n;
  }
  if (lane == 31) warp_sums[w] = v;
  __syncthreads();
  if (w == 0) {
    int64_t s = warp_sums[lane];
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      int64_t n = __shfl_up_sync(0xffffffffu, s, o);
      if (lane >= o) s += n;
    }
    warp_sums[lane] = s;
  }
  __syncthreads();
  if (w > 0) v += warp_sums[w - 1];
  *total = warp_sums[31];
  __syncthreads();
  return v;
}

// 1. run heads -> seg_start[nseg]; out[0] = nseg, out[1] = error flag.  Three launches so that the
// exposure axis is walked by the whole GPU (one block walked it alone in round 1: 0.10 ms at 10^5
// exposures, 1 ms at 10^6, per rr_set_data and so per rr_evaluate_flat):
//   1a. one block per SCAN_T exposures: number of run heads in the block, range check of lc_index
//   1b. one block: exclusive scan of the per-block counts
//   1c. one block per SCAN_T exposures: scan inside the block, scatter of the run heads
__device__ __forceinline__ int rr_k4_is_head(const int32_t *__restrict__ lc, int64_t i, int64_t npt,
                                             int32_t nlc, int *bad) {
  if (i >= npt) return 0;
  const int32_t l = lc[i];
  if (l < 0 || l >= nlc) *bad = 1;
  return (i == 0 || lc[i - 1] != l) ? 1 : 0;
}

__global__ void __launch_bounds__(SCAN_T)
rr_k4_heads_count(const int32_t *__restrict__ lc, int64_t npt, int32_t nlc,
                  int64_t *__restrict__ blk_count, int64_t *__restrict__ out) {
  int bad = 0;
  const int head = rr_k4_is_head(lc, (int64_t)blockIdx.x * SCAN_T + threadIdx.x, npt, nlc, &bad);
  const int n = __syncthreads_count(head);
  const int anybad = __syncthreads_or(bad);
  if (threadIdx.x == 0) {
    blk_count[blockIdx.x] = n;
    if (anybad) out[1] = 1;                        // (out[0..3] were zeroed by the launcher)
  }
}

__global__ void __launch_bounds__(SCAN_T)
rr_k4_heads_scan(int64_t nblk, const int64_t *__restrict__ blk_count, int64_t *__restrict__ blk_off,
                 int64_t *__restrict__ out) {
  __shared__ int64_t ws[32];
  int64_t carry = 0;
  for (int64_t base = 0; base < nblk; base += SCAN_T) {
    const int64_t b = base + threadIdx.x;
    const int64_t n = b < nblk ? blk_count[b] : 0;
    int64_t tot;
    const int64_t inc = block_inclusive_scan(n, ws, &tot);
    if (b < nblk) blk_off[b] = carry + inc - n;
    carry += tot;
  }
  if (threadIdx.x == 0) out[0] = carry;
}

__global__ void __launch_bounds__(SCAN_T)
rr_k4_heads_scatter(const int32_t *__restrict__ lc, int64_t npt, int32_t nlc,
                    const int64_t *__restrict__ blk_off, int64_t *__restrict__ seg_start) {
  __shared__ int64_t ws[32];
  int bad = 0;
  const int64_t i = (int64_t)blockIdx.x * SCAN_T + threadIdx.x;
  const int64_t head = rr_k4_is_head(lc, i, npt, nlc, &bad);
  int64_t tot;
  const int64_t inc = block_inclusive_scan(head, ws, &tot);
  if (head) seg_start[blk_off[blockIdx.x] + inc - 1] = i;
}

// Tile length of a run of exposures [b, e) of one light curve: at most the light curve's tile_len
// (RR_TILE_UNIT x R exposures, set from ns so that a tile carries ~4096 sub-samples), and no longer
// than RR_TILE_SPAN days at the run's mean cadence |t[e-1] - t[b]| / (e-b-1), in multiples of 128
// exposures (one pass of a flux block), at least 128.  A transit lasts hours: with sparse cadences
// (10^5 exposures two minutes apart) a 3072-exposure tile spans four days, always holds a transit and
// is never skipped; 0.1-day tiles are.  Times in any order are allowed: the span of an unsorted run is
// meaningless, which costs speed, not correctness.
#ifndef RR_TILE_SPAN
#define RR_TILE_SPAN 0.1
#endif
__device__ __forceinline__ int64_t rr_k4_run_tile_len(const double *__restrict__ times, int64_t b,
                                                      int64_t e, int64_t max_len) {
  if (e - b < 2) return max_len;
  const double span = fabs(times[e - 1] - times[b]);
  const double q = RR_TILE_SPAN / span;                       // IEEE division, then one product:
  const double n = (double)(e - b - 1) * q;                   // the tests restate these two roundings
  if (!(n < (double)max_len)) return max_len;                 // also span = 0, NaN, infinite
  const int64_t len = (((int64_t)n + 127) / 128) * 128;
  return len < 128 ? 128 : (len > max_len ? max_len : len);
}

// 2. tiles per run and their exclusive scan; out[2] = ntiles.
__global__ void __launch_bounds__(SCAN_T)
rr_k4_tilecount(const int32_t *__restrict__ lc, const double *__restrict__ times, int64_t npt,
                const RRLc *__restrict__ lcs,
                const int64_t *__restrict__ seg_start, int64_t *__restrict__ tile_off,
                int64_t *__restrict__ out) {
  __shared__ int64_t ws[32];
  int64_t nseg = out[0];
  int64_t carry = 0;
  for (int64_t base = 0; base < nseg; base += SCAN_T) {
    int64_t s = base + threadIdx.x;
    int64_t nt = 0;
    if (s < nseg) {
      int64_t b = seg_start[s], e = (s + 1 < nseg) ? seg_start[s + 1] : npt;
      int64_t len = rr_k4_run_tile_len(times, b, e, lcs[lc[b]].tile_len);
      nt = (e - b + len - 1) / len;
    }
    int64_t tot;
    int64_t inc = block_inclusive_scan(nt, ws, &tot);
    if (s < nseg) tile_off[s] = carry + inc - nt;
    carry += tot;
  }
  if (threadIdx.x == 0) out[2] = carry;
}

// 3. one thread per tile.
__global__ void rr_k4_tiles(const int32_t *__restrict__ lc, const double *__restrict__ times,
                            int64_t npt, const RRLc *__restrict__ lcs, const int64_t *__restrict__ seg_start,
                            const int64_t *__restrict__ tile_off, int64_t nseg, int64_t ntiles,
                            RRTile *__restrict__ tiles) {
  int64_t tl = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (tl >= ntiles) return;
  int64_t lo = 0, hi = nseg - 1;   // last run whose first tile is <= tl
  while (lo < hi) {
    int64_t mid = (lo + hi + 1) >> 1;
    if (tile_off[mid] <= tl) lo = mid; else hi = mid - 1;
  }
  int64_t b = seg_start[lo], e = (lo + 1 < nseg) ? seg_start[lo + 1] : npt;
  int32_t l = lc[b];
  int64_t len = rr_k4_run_tile_len(times, b, e, lcs[l].tile_len);
  int64_t start = b + (tl - tile_off[lo]) * len;
  int64_t count = e - start < len ? e - start : len;
  RRTile r;
  r.tmin = 0.0;
  r.tmax = 0.0;
  r.sub_off = count * (int64_t)lcs[l].ns;   // scanned in step 4
  r.start = (int32_t)start;
  r.count = (int32_t)count;
  r.lc = l;
  r.pad = 0;
  tiles[tl] = r;
}

// 4a. one warp per tile: time range.
__global__ void rr_k4_ranges(const double *__restrict__ times, int64_t ntiles,
                             RRTile *__restrict__ tiles) {
  int64_t tl = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (tl >= ntiles) return;
  int start = tiles[tl].start, count = tiles[tl].count;
  double lo = INFINITY, hi = -INFINITY;
  for (int i = lane; i < count; i += 32) {
    double t = times[start + i];
    lo = fmin(lo, t);
    hi = fmax(hi, t);
    if (!(t == t)) { lo = -INFINITY; hi = INFINITY; }   // NaN time: never skip the tile
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    lo = fmin(lo, __shfl_xor_sync(0xffffffffu, lo, o));
    hi = fmax(hi, __shfl_xor_sync(0xffffffffu, hi, o));
  }
  if (lane == 0) {
    tiles[tl].tmin = lo;
    tiles[tl].tmax = hi;
  }
}

// 4b. exclusive scan of the per-tile sub-sample counts; out[3] = nsub.
__global__ void __launch_bounds__(SCAN_T)
rr_k4_suboff(int64_t ntiles, RRTile *__restrict__ tiles, int64_t *__restrict__ out) {
  __shared__ int64_t ws[32];
  int64_t carry = 0;
  for (int64_t base = 0; base < ntiles; base += SCAN_T) {
    int64_t i = base + threadIdx.x;
    int64_t n = (i < ntiles) ? tiles[i].sub_off : 0;
    int64_t tot;
    int64_t inc = block_inclusive_scan(n, ws, &tot);
    if (i < ntiles) tiles[i].sub_off = carry + inc - n;
    carry += tot;
  }
  if (threadIdx.x == 0) out[3] = carry;
}

}  // namespace

// Needs ctx->d_times, d_lc_index, d_lc, npt, nlc set.  Synchronous on st.
int rr_dispatch_build(rr_ctx *ctx, cudaStream_t st) {
  int64_t npt = ctx->npt;
  // scratch: seg_start[npt] | tile_off[npt] | out[4] | blk_count[nblk] | blk_off[nblk]
  const int64_t nblk = (npt + SCAN_T - 1) / SCAN_T;
  int64_t need = 2 * npt + 4 + 2 * nblk;
  if (need > ctx->scratch_cap) {
    if (ctx->d_scratch) cudaFree(ctx->d_scratch);
    ctx->d_scratch = nullptr;
    ctx->scratch_cap = 0;
    if (cudaMalloc(&ctx->d_scratch, sizeof(int64_t) * need) != cudaSuccess) return RR_EALLOC;
    ctx->scratch_cap = need;
  }
  int64_t *seg_start = ctx->d_scratch, *tile_off = seg_start + npt, *out = tile_off + npt;
  int64_t *blk_count = out + 4, *blk_off = blk_count + nblk;
  RR_CUDA(cudaMemsetAsync(out, 0, sizeof(int64_t) * 4, st));
  rr_k4_heads_count<<<(unsigned)nblk, SCAN_T, 0, st>>>(ctx->d_lc_index, npt, ctx->nlc, blk_count, out);
  RR_LAUNCH_CHECK(ctx);
  rr_k4_heads_scan<<<1, SCAN_T, 0, st>>>(nblk, blk_count, blk_off, out);
  RR_LAUNCH_CHECK(ctx);
  rr_k4_heads_scatter<<<(unsigned)nblk, SCAN_T, 0, st>>>(ctx->d_lc_index, npt, ctx->nlc, blk_off,
                                                         seg_start);
  RR_LAUNCH_CHECK(ctx);
  int64_t h[4] = {0, 0, 0, 0};
  RR_CUDA(cudaMemcpyAsync(h, out, sizeof(int64_t) * 2, cudaMemcpyDeviceToHost, st));
  RR_CUDA(cudaStreamSynchronize(st));
  if (h[1]) return RR_EINDEX;
  int64_t nseg = h[0];
  rr_k4_tilecount<<<1, SCAN_T, 0, st>>>(ctx->d_lc_index, ctx->d_times, npt, ctx->d_lc, seg_start,
                                        tile_off, out);
  RR_LAUNCH_CHECK(ctx);
  RR_CUDA(cudaMemcpyAsync(h, out, sizeof(int64_t) * 3, cudaMemcpyDeviceToHost, st));
  RR_CUDA(cudaStreamSynchronize(st));
  int64_t ntiles = h[2];
  if (ntiles > ctx->tiles_cap) {
    if (ctx->d_tiles) cudaFree(ctx->d_tiles);
    ctx->d_tiles = nullptr;
    ctx->tiles_cap = 0;
    if (cudaMalloc(&ctx->d_tiles, sizeof(RRTile) * ntiles) != cudaSuccess) return RR_EALLOC;
    ctx->tiles_cap = ntiles;
  }
  rr_k4_tiles<<<(unsigned)((ntiles + 255) / 256), 256, 0, st>>>(
      ctx->d_lc_index, ctx->d_times, npt, ctx->d_lc, seg_start, tile_off, nseg, ntiles, ctx->d_tiles);
  RR_LAUNCH_CHECK(ctx);
  rr_k4_ranges<<<(unsigned)((ntiles * 32 + 255) / 256), 256, 0, st>>>(ctx->d_times, ntiles,
                                                                      ctx->d_tiles);
  RR_LAUNCH_CHECK(ctx);
  rr_k4_suboff<<<1, SCAN_T, 0, st>>>(ntiles, ctx->d_tiles, out);
  RR_LAUNCH_CHECK(ctx);
  RR_CUDA(cudaMemcpyAsync(h, out, sizeof(int64_t) * 4, cudaMemcpyDeviceToHost, st));
  RR_CUDA(cudaStreamSynchronize(st));
  ctx->ntiles = ntiles;
  ctx->nsub = h[3];
  return RR_OK;
}
