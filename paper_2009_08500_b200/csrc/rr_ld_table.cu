// rr_ld_table.cu - kernel 1: the per-call limb-darkening table.
//   T[row][n] = sum_j W[n][j] * ldp[row][j],   row = pv*npb + pb,  n = ik*ng + ig,  j < nz
//   Istar[row] = sum_j q[j] * ldp[row][j],     q[j] = pi (ze[j+1]^2 - ze[j]^2)    (reading R6)
// A "TN" matrix product C[M][N] = A[M][K] . B[N][K]^T with M = npv*npb, N = nk*ng (5000),
// K = nz (100..200), both operands K-contiguous.  fp64 FMA accumulation in k order for both ctx
// precisions (the fp32 mode only narrows the operand A on load and C on store).  It is a skinny
// product worth a few per cent of a step: a register-blocked DFMA kernel, 128x128
// block tile, 8x8 micro tile, operands staged k-major in shared memory with register prefetch of
// the next k slab.  B200's DMMA rate equals its DFMA rate, so tensor cores would buy nothing here.
#include "rr_common.cuh"

namespace {

constexpr int BM = 128, BN = 128, BK = 16, PAD = 2, NT = 256;

template <typename T> struct Vec2;
template <> struct Vec2<double> { using type = double2; };
template <> struct Vec2<float> { using type = float2; };

template <typename TA, typename TC>
__global__ void __launch_bounds__(NT, 1)
rr_ld_table_kernel(const TA *__restrict__ A, const double *__restrict__ B, TC *__restrict__ C,
                   int64_t M, int N, int K) {
  __shared__ __align__(16) double As[BK][BM + PAD];
  __shared__ __align__(16) double Bs[BK][BN + PAD];
  const int t = threadIdx.x;
  const int tx = t & 15, ty = t >> 4;
  const int64_t m0 = (int64_t)blockIdx.y * BM;
  const int n0 = blockIdx.x * BN;
  // loader mapping: thread -> (row r of the tile, k half h): 8 consecutive k of one row
  const int lr = t >> 1, lh = (t & 1) * 8;
  const int64_t am = m0 + lr;
  const int bn = n0 + lr;
  const bool a_ok = am < M, b_ok = bn < N;
  const TA *ap = A + (a_ok ? am : 0) * (int64_t)K;
  const double *bp = B + (int64_t)(b_ok ? bn : 0) * K;

  double acc[8][8];
#pragma unroll
  for (int i = 0; i < 8; ++i)
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[i][j] = 0.0;

  double ra[8], rb[8];
  auto gload = [&](int kb) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      int k = kb + lh + q;
      bool kin = k < K;
      ra[q] = (a_ok && kin) ? (double)ap[k] : 0.0;
      rb[q] = (b_ok && kin) ? bp[k] : 0.0;
    }
  };
  gload(0);
  for (int kb = 0; kb < K; kb += BK) {
#pragma unroll
    for (int q = 0; q < 8; ++q) {
      As[lh + q][lr] = ra[q];
      Bs[lh + q][lr] = rb[q];
    }
    __syncthreads();
    if (kb + BK < K) gload(kb + BK);
#pragma unroll
    for (int kk = 0; kk < BK; ++kk) {
      double a[8], b[8];
#pragma unroll
      for (int i = 0; i < 8; i += 2) {
        double2 v = *reinterpret_cast<const double2 *>(&As[kk][ty * 8 + i]);
        a[i] = v.x;
        a[i + 1] = v.y;
      }
#pragma unroll
      for (int c = 0; c < 4; ++c) {
        double2 v = *reinterpret_cast<const double2 *>(&Bs[kk][tx * 2 + 32 * c]);
        b[2 * c] = v.x;
        b[2 * c + 1] = v.y;
      }
#pragma unroll
      for (int i = 0; i < 8; ++i)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[i][j] = fma(a[i], b[j], acc[i][j]);
    }
    __syncthreads();
  }
  // epilogue: 16 lanes x 16 B contiguous per row
  const bool vec_ok = (N & 1) == 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    int64_t m = m0 + ty * 8 + i;
    if (m >= M) continue;
    TC *crow = C + m * (int64_t)N;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      int n = n0 + tx * 2 + 32 * c;
      if (vec_ok && n + 1 < N) {
        typename Vec2<TC>::type v;
        v.x = (TC)acc[i][2 * c];
        v.y = (TC)acc[i][2 * c + 1];
        *reinterpret_cast<typename Vec2<TC>::type *>(crow + n) = v;
      } else {
        if (n < N) crow[n] = (TC)acc[i][2 * c];
        if (n + 1 < N) crow[n + 1] = (TC)acc[i][2 * c + 1];
      }
    }
  }
}

// Istar: one warp per row.
template <typename TA, typename TC>
__global__ void rr_istar_kernel(const TA *__restrict__ A, const double *__restrict__ q,
                                const TC *__restrict__ given, TC *__restrict__ out, int64_t M,
                                int K) {
  int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (row >= M) return;
  if (given) {
    if (lane == 0) out[row] = given[row];
    return;
  }
  double s = 0.0;
  for (int j = lane; j < K; j += 32) s = fma(q[j], (double)A[row * K + j], s);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) out[row] = (TC)s;
}

// Lazy mode: Istar and the ctx-owned copy of the profile in ONE launch (a copy engine call and a
// kernel were two: small problems are bound by the length of the launch chain).  One warp per row.
template <typename T>
__global__ void rr_istar_copy_kernel(const T *__restrict__ A, const double *__restrict__ q,
                                     const T *__restrict__ given, T *__restrict__ out,
                                     T *__restrict__ copy, int64_t M, int K) {
  int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  int lane = threadIdx.x & 31;
  if (row >= M) return;
  double s = 0.0;
  for (int j = lane; j < K; j += 32) {
    const T a = A[row * K + j];
    copy[row * K + j] = a;
    s = fma(q[j], (double)a, s);
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) out[row] = given ? given[row] : (T)s;
}

// ---- named limb-darkening laws on the device --------------------
// ldp[row][j] = I(mu_j; ldc[row]) and the analytic disc integral Istar = 2 pi int_0^1 mu I dmu
// ("all integrated analytically over the stellar disk").  The paper names the laws
// and cites their sources without printing them; the forms are the textbook ones, stated in
// include/roadrunner.h.  One thread per (row, j); fp64 arithmetic, stored in the ctx precision.
__device__ double rr_law_value(int law, const double *c, int nc, double mu) {
  const double x = 1.0 - mu;
  switch (law) {
    case RR_LD_UNIFORM: return 1.0;
    case RR_LD_LINEAR: return 1.0 - c[0] * x;
    case RR_LD_QUADRATIC: return 1.0 - c[0] * x - c[1] * x * x;
    case RR_LD_QUADRATIC_TRI: {
      const double sq = sqrt(c[0]), u1 = 2.0 * sq * c[1], u2 = sq * (1.0 - 2.0 * c[1]);
      return 1.0 - u1 * x - u2 * x * x;
    }
    case RR_LD_GENERAL: {
      double s = 1.0, p = 1.0;
      for (int n = 0; n < nc; ++n) { p *= mu; s -= c[n] * (1.0 - p); }       // 1 - mu^(n+1)
      return s;
    }
    case RR_LD_NONLINEAR: {
      const double r = sqrt(mu);
      return 1.0 - c[0] * (1.0 - r) - c[1] * (1.0 - mu) - c[2] * (1.0 - mu * r) - c[3] * (1.0 - mu * mu);
    }
    case RR_LD_LOGARITHMIC: return 1.0 - c[0] * x - c[1] * (mu > 0.0 ? mu * log(mu) : 0.0);
    case RR_LD_EXPONENTIAL: return 1.0 - c[0] * x - c[1] / (1.0 - exp(mu));
    case RR_LD_POWER2: return 1.0 - c[0] * (1.0 - pow(mu, c[1]));
    case RR_LD_POWER2_PM: {
      const double cc = 1.0 - c[0] + c[1], al = log2(cc / c[1]);
      return 1.0 - cc * (1.0 - pow(mu, al));
    }
    default: return 1.0;
  }
}

// Istar / pi in closed form (every law but RR_LD_EXPONENTIAL, for which the host launcher asks for
// the discretised integral of reading R6 instead and this function is not called).
__device__ double rr_law_istar_over_pi(int law, const double *c, int nc) {
  switch (law) {
    case RR_LD_UNIFORM: return 1.0;
    case RR_LD_LINEAR: return 1.0 - c[0] / 3.0;
    case RR_LD_QUADRATIC: return 1.0 - c[0] / 3.0 - c[1] / 6.0;
    case RR_LD_QUADRATIC_TRI: {
      const double sq = sqrt(c[0]), u1 = 2.0 * sq * c[1], u2 = sq * (1.0 - 2.0 * c[1]);
      return 1.0 - u1 / 3.0 - u2 / 6.0;
    }
    case RR_LD_GENERAL: {
      double s = 1.0;
      for (int n = 0; n < nc; ++n) s -= c[n] * (double)(n + 1) / (double)(n + 3);
      return s;
    }
    case RR_LD_NONLINEAR:
      return 1.0 - c[0] / 5.0 - c[1] / 3.0 - 3.0 * c[2] / 7.0 - c[3] / 2.0;
    case RR_LD_LOGARITHMIC: return 1.0 - c[0] / 3.0 + 2.0 * c[1] / 9.0;
    case RR_LD_POWER2: return 1.0 - c[0] * c[1] / (c[1] + 2.0);
    case RR_LD_POWER2_PM: {
      const double cc = 1.0 - c[0] + c[1], al = log2(cc / c[1]);
      return 1.0 - cc * al / (al + 2.0);
    }
    default: return -1.0;
  }
}

template <typename TR>
__global__ void rr_ld_law_kernel(int law, const double *__restrict__ ldc, int nc,
                                 const double *__restrict__ mu, int64_t M, int nz,
                                 TR *__restrict__ ldp, TR *__restrict__ istar_or_null) {
  const int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= M * nz) return;
  const int64_t row = idx / nz;
  const int j = (int)(idx - row * nz);
  const double *c = ldc + row * nc;
  ldp[idx] = (TR)rr_law_value(law, c, nc, mu[j]);
  if (j == 0 && istar_or_null) istar_or_null[row] = (TR)(RR_PI * rr_law_istar_over_pi(law, c, nc));
}

// Lazy mode: the k-collapsed row of one (pv, passband),
//   ldw[ig] = (1 - ak) sum_j W[ik][ig][j] ldp[j] + ak sum_j W[ik+1][ig][j] ldp[j]
// for the pv's own k (ik, ak from the per-pv prep).  One block per (pv, passband); the profile sits
// in shared memory; one warp per g node, lanes over j (coalesced reads of W, which stays in L2:
// the two rows are 2 ng nz 8 B = 160 kB), shuffle sums.  fp64 accumulation in both precisions.
constexpr int RT = 256;
template <typename TR>
__global__ void __launch_bounds__(RT)
rr_ld_rows_kernel(const TR *__restrict__ ldp, const double *__restrict__ W,
                  const int2 *__restrict__ sup,
                  const RRPvBand *__restrict__ pvb, TR *__restrict__ rows, int npb, int nkpb,
                  int ng, int nz) {
  extern __shared__ double prof[];
  const int64_t row = blockIdx.x;                 // pv * npb + pb
  const int64_t v = row / npb;
  const int pb = (int)(row - v * npb);
  const RRPvBand &b = pvb[v * nkpb + (nkpb == 1 ? 0 : pb)];
  const int ik = b.ik;
  const double ak = b.ak;
  for (int j = threadIdx.x; j < nz; j += RT) prof[j] = (double)ldp[row * nz + j];
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double *W0 = W + (int64_t)ik * ng * nz;
  const double *W1 = W0 + (int64_t)ng * nz;
  // (gridDim.y blocks share a row's g nodes: with few rows every warp should have few nodes, each
  // is two dependent rounds of L2 loads - one row in one block took 13 us)
  for (int ig = blockIdx.y * (RT / 32) + warp; ig < ng; ig += (RT / 32) * gridDim.y) {
    const double *w0 = W0 + (int64_t)ig * nz, *w1 = W1 + (int64_t)ig * nz;
    // only the support of the two weight rows (rr_support_kernel): the rest is exactly zero; lanes
    // keep their j mod 32, so the sums are those of the full loop (1024 rows read 164 MB of W from
    // L2 otherwise: config 1's rows took as long as its flux kernel)
    const int2 a0 = sup[(int64_t)ik * ng + ig], a1 = sup[(int64_t)(ik + 1) * ng + ig];
    const int jl = min(a0.x, a1.x) & ~31, jh = max(a0.y, a1.y);
    double s0 = 0.0, s1 = 0.0;
    for (int j = jl + lane; j < jh; j += 32) {
      const double p = prof[j];
      s0 = fma(w0[j], p, s0);
      s1 = fma(w1[j], p, s1);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      s0 += __shfl_xor_sync(0xffffffffu, s0, o);
      s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    }
    if (lane == 0) rows[row * ng + ig] = (TR)fma(ak, s1 - s0, s0);
  }
}

// Lazy mode at scale: rows (pv, passband) are bucketed by their lower k row ik (counting sort:
// histogram, scan, scatter), and one block builds RB rows of ONE bucket, so that the two weight rows
// W[ik], W[ik+1] are read once per RB profiles (warp-uniform loads served by L1) instead of once per
// profile from L2 (2.6 GB of L2 reads at config 4 otherwise).  Lane = row, warp = g nodes.
constexpr int RB = 32;
#ifndef RR_ROWS_SMEM4_MAX
#define RR_ROWS_SMEM4_MAX (110 * 1024)   // NG = 4 while two blocks still fit an SM
#endif

__device__ __forceinline__ int rr_row_ik(const RRPvBand *__restrict__ pvb, int64_t row, int npb,
                                         int nkpb) {
  const int64_t v = row / npb;
  const int pb = (int)(row - v * npb);
  return pvb[v * nkpb + (nkpb == 1 ? 0 : pb)].ik;
}

__global__ void rr_rows_hist(const RRPvBand *__restrict__ pvb, int64_t M, int npb, int nkpb,
                             int *__restrict__ hist) {
  const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (row < M) atomicAdd(&hist[rr_row_ik(pvb, row, npb, nkpb)], 1);
}

// One block: exclusive scans of the bucket sizes and of their tile counts (nb <= 4096 buckets).
__global__ void rr_rows_scan(int nb, const int *__restrict__ hist, int *__restrict__ offs,
                             int *__restrict__ tileoff) {
  if (threadIdx.x == 0) {
    int o = 0, t = 0;
    for (int b = 0; b < nb; ++b) {
      offs[b] = o;
      tileoff[b] = t;
      o += hist[b];
      t += (hist[b] + RB - 1) / RB;
    }
    offs[nb] = o;
    tileoff[nb] = t;
  }
}

__global__ void rr_rows_scatter(const RRPvBand *__restrict__ pvb, int64_t M, int npb, int nkpb,
                                const int *__restrict__ offs, int *__restrict__ cursor,
                                int *__restrict__ list) {
  const int64_t row = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  if (row >= M) return;
  const int ik = rr_row_ik(pvb, row, npb, nkpb);
  list[offs[ik] + atomicAdd(&cursor[ik], 1)] = (int)row;
}

// Register tile: every warp takes NG g nodes (lane = row), so that one profile value feeds 2 NG FMAs,
// and the weights are read as 16-byte broadcasts (two j per load) when nz is even: per pair of j,
// 4 + 2 NG shared-memory wavefronts feed 4 NG FMAs (NG = 4: 0.75 per FMA; one lane = one row = one node
// needed 2 per FMA and was bound by the LSU at 1/4 of the FP64 pipe).  The sums run over j in order:
// bit-identical to the per-row builder.
template <typename TR, int NG>
__global__ void __launch_bounds__(256)
rr_ld_rows_bucket_kernel(const TR *__restrict__ ldp, const double *__restrict__ W,
                         const int2 *__restrict__ sup,
                         const RRPvBand *__restrict__ pvb, const int *__restrict__ list,
                         const int *__restrict__ offs, const int *__restrict__ tileoff, int nb,
                         TR *__restrict__ rows, int npb, int nkpb, int ng, int nz, int stride) {
  extern __shared__ __align__(16) double prof[];   // [RB][stride], stride odd: conflict-free
  __shared__ int rid[RB];
  __shared__ double akr[RB];
  constexpr int CH = 8 * NG;                       // g nodes per chunk: 8 warps x NG
  const int b = blockIdx.x;
  if (b >= tileoff[nb]) return;
  int lo = 0, hi = nb - 1;                         // last bucket whose first tile is <= b
  while (lo < hi) {
    const int mid = (lo + hi + 1) >> 1;
    if (tileoff[mid] <= b) lo = mid; else hi = mid - 1;
  }
  const int ik = lo;
  const int r0 = offs[ik] + (b - tileoff[ik]) * RB;
  const int nr = min(RB, offs[ik + 1] - r0);
  if (threadIdx.x < RB) {
    int row = -1;
    double ak = 0.0;
    if ((int)threadIdx.x < nr) {
      row = list[r0 + threadIdx.x];
      const int64_t v = row / npb;
      const int pb = (int)(row - v * npb);
      ak = pvb[v * nkpb + (nkpb == 1 ? 0 : pb)].ak;
    }
    rid[threadIdx.x] = row;
    akr[threadIdx.x] = ak;
  }
  __syncthreads();
  for (int idx = threadIdx.x; idx < RB * nz; idx += 256) {
    const int r = idx / nz, j = idx - r * nz;
    prof[r * stride + j] = (r < nr) ? (double)ldp[(int64_t)rid[r] * nz + j] : 0.0;
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const double *W0 = W + (int64_t)ik * ng * nz;
  const double *W1 = W0 + (int64_t)ng * nz;
  const double *pr = prof + lane * stride;
  const double ak = akr[lane];
  const int64_t orow = (int64_t)rid[lane] * ng;
  // The weight rows of CH g nodes at a time go through shared memory: all 256 threads load them
  // coalesced (deep memory-level parallelism), then every warp takes NG nodes, lane = row.  Only the
  // columns [ja, jb) in which some row of the chunk is non-zero are staged, and every warp sums over
  // the support of its own NG nodes (rr_support_kernel): a planet covers 2k of the stellar radius.
  __shared__ int jrange[2];
  double *wb0 = prof + RB * stride;                // 16-byte aligned; wb1 follows at an even offset
  const int2 *sup0 = sup + (int64_t)ik * ng, *sup1 = sup0 + ng;
  for (int c0 = 0; c0 < ng; c0 += CH) {
    const int nrow = min(CH, ng - c0);
    __syncthreads();                               // the previous chunk is consumed (first: profiles written)
    if (threadIdx.x == 0) { jrange[0] = nz; jrange[1] = 0; }
    __syncthreads();
    if ((int)threadIdx.x < 2 * nrow) {
      const int2 r = threadIdx.x < nrow ? sup0[c0 + threadIdx.x] : sup1[c0 + threadIdx.x - nrow];
      atomicMin(&jrange[0], r.x);
      atomicMax(&jrange[1], r.y);
    }
    __syncthreads();
    const int ja = jrange[0] & ~1, jb = min(nz, (jrange[1] + 1) & ~1);
    const int len = jb - ja, lenp = (len + 1) & ~1;  // row pitch in shared memory, even
    double *wb1 = wb0 + CH * lenp;
    for (int idx = threadIdx.x; idx < nrow * len; idx += 256) {
      const int q = idx / len, j = idx - q * len;
      wb0[q * lenp + j] = __ldg(W0 + (int64_t)(c0 + q) * nz + ja + j);
      wb1[q * lenp + j] = __ldg(W1 + (int64_t)(c0 + q) * nz + ja + j);
    }
    __syncthreads();
    const int g0 = warp * NG;
    if (g0 < nrow) {
      // support of this warp's nodes (both k rows), inside [ja, jb)
      int jl = nz, jh = 0;
#pragma unroll
      for (int q = 0; q < NG; ++q)
        if (g0 + q < nrow) {
          const int2 a = sup0[c0 + g0 + q], c = sup1[c0 + g0 + q];
          jl = min(jl, min(a.x, c.x));
          jh = max(jh, max(a.y, c.y));
        }
      const double *w0 = wb0 + g0 * lenp - ja, *w1 = wb1 + g0 * lenp - ja;   // indexed by j
      double s0[NG], s1[NG];
#pragma unroll
      for (int q = 0; q < NG; ++q) s0[q] = s1[q] = 0.0;
      if ((nz & 1) == 0) {                         // ja, lenp even: 16-byte aligned pairs
        jl &= ~1;                                  // stays >= ja (even)
        jh = min(jb, (jh + 1) & ~1);
#pragma unroll 2
        for (int j = jl; j < jh; j += 2) {
          const double p0 = pr[j], p1 = pr[j + 1];
#pragma unroll
          for (int q = 0; q < NG; ++q) {           // nodes past nrow read stale weights; never stored
            const double2 a = *reinterpret_cast<const double2 *>(w0 + q * lenp + j);
            const double2 c = *reinterpret_cast<const double2 *>(w1 + q * lenp + j);
            s0[q] = fma(a.y, p1, fma(a.x, p0, s0[q]));
            s1[q] = fma(c.y, p1, fma(c.x, p0, s1[q]));
          }
        }
      } else {
#pragma unroll 2
        for (int j = jl; j < jh; ++j) {
          const double p = pr[j];
#pragma unroll
          for (int q = 0; q < NG; ++q) {
            s0[q] = fma(w0[q * lenp + j], p, s0[q]);
            s1[q] = fma(w1[q * lenp + j], p, s1[q]);
          }
        }
      }
      if (lane < nr) {
#pragma unroll
        for (int q = 0; q < NG; ++q)
          if (g0 + q < nrow) rows[orow + c0 + g0 + q] = (TR)fma(ak, s1[q] - s0[q], s0[q]);
      }
    }
  }
}

template <typename TR>
int launch_typed(rr_ctx *ctx, RRWork *wk, const void *d_ldp, const void *d_istar, int64_t npv,
                 cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  int64_t M = npv * c.npb;
  int N = c.nk * c.ng, K = ctx->nz;
  dim3 grid((N + BN - 1) / BN, (unsigned)((M + BM - 1) / BM));
  rr_ld_table_kernel<TR, TR><<<grid, NT, 0, st>>>((const TR *)d_ldp, ctx->d_W, (TR *)wk->T, M,
                                                  N, K);
  RR_LAUNCH_CHECK(ctx);
  if (d_istar == wk->istar) return RR_OK;          // already in place (named law, closed form)
  int64_t threads = M * 32;
  rr_istar_kernel<TR, TR><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
      (const TR *)d_ldp, ctx->d_q, (const TR *)d_istar, (TR *)wk->istar, M, K);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

}  // namespace

// Grows wk->T / wk->istar as needed (cudaMalloc: synchronous, only when a larger npv arrives).
int rr_ld_table_launch(rr_ctx *ctx, RRWork *wk, const void *d_ldp, const void *d_istar,
                       int64_t npv, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t esz = c.precision != RR_FP64 ? 4 : 8;
  const int64_t needT = npv * c.npb * (int64_t)c.nk * c.ng * esz, needI = npv * c.npb * esz;
  if (needT > wk->T_cap) {
    if (wk->T) cudaFree(wk->T);
    wk->T = nullptr;
    wk->T_cap = 0;
    wk->table_npv = -1;
    if (cudaMalloc(&wk->T, needT) != cudaSuccess) { cudaGetLastError(); return RR_EALLOC; }
    wk->T_cap = needT;
  }
  if (needI > wk->istar_cap) {
    if (wk->istar) cudaFree(wk->istar);
    wk->istar = nullptr;
    wk->istar_cap = 0;
    wk->table_npv = -1;
    if (cudaMalloc(&wk->istar, needI) != cudaSuccess) { cudaGetLastError(); return RR_EALLOC; }
    wk->istar_cap = needI;
  }
  int rc = c.precision != RR_FP64 ? launch_typed<float>(ctx, wk, d_ldp, d_istar, npv, st)
                                  : launch_typed<double>(ctx, wk, d_ldp, d_istar, npv, st);
  wk->table_npv = rc == RR_OK ? npv : -1;
  wk->lazy = 0;
  wk->have_full = rc == RR_OK;
  wk->ldp_src = nullptr;
  return rc;
}

static int grow_buf(void **p, int64_t *cap, int64_t need) {
  if (need <= *cap) return RR_OK;
  if (*p) cudaFree(*p);
  *p = nullptr;
  *cap = 0;
  if (cudaMalloc(p, (size_t)need) != cudaSuccess) { cudaGetLastError(); return RR_EALLOC; }
  *cap = need;
  return RR_OK;
}

// Lazy mode, at rr_build_ld_table: keep the profile (copy = 1: into a buffer of ours; 0: the
// caller guarantees d_ldp lives until the evaluation, the host path's staging) and compute Istar.
int rr_ld_profile_launch(rr_ctx *ctx, RRWork *wk, const void *d_ldp, const void *d_istar,
                         int64_t npv, int copy, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t esz = c.precision != RR_FP64 ? 4 : 8;
  const int64_t M = npv * c.npb, needP = M * ctx->nz * esz, needI = M * esz;
  wk->table_npv = -1;
  int rc = grow_buf(&wk->istar, &wk->istar_cap, needI);
  if (rc == RR_OK && copy) rc = grow_buf(&wk->ldp, &wk->ldp_cap, needP);
  if (rc != RR_OK) return rc;
  wk->ldp_src = copy ? wk->ldp : d_ldp;
  const int64_t threads = M * 32;
  if (copy && d_ldp != wk->ldp) {
    if (c.precision != RR_FP64)
      rr_istar_copy_kernel<float><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
          (const float *)d_ldp, ctx->d_q, (const float *)d_istar, (float *)wk->istar,
          (float *)wk->ldp, M, ctx->nz);
    else
      rr_istar_copy_kernel<double><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
          (const double *)d_ldp, ctx->d_q, (const double *)d_istar, (double *)wk->istar,
          (double *)wk->ldp, M, ctx->nz);
    RR_LAUNCH_CHECK(ctx);
  } else if (d_istar == wk->istar) {
    // already in place (named law with a closed form)
  } else if (c.precision != RR_FP64) {
    rr_istar_kernel<float, float><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
        (const float *)d_ldp, ctx->d_q, (const float *)d_istar, (float *)wk->istar, M, ctx->nz);
    RR_LAUNCH_CHECK(ctx);
  } else {
    rr_istar_kernel<double, double><<<(unsigned)((threads + 255) / 256), 256, 0, st>>>(
        (const double *)d_ldp, ctx->d_q, (const double *)d_istar, (double *)wk->istar, M, ctx->nz);
    RR_LAUNCH_CHECK(ctx);
  }
  wk->table_npv = npv;
  wk->lazy = ctx->table_mode == RR_TABLE_DIRECT ? 2 : 1;
  wk->have_full = 0;
  return RR_OK;
}

// Lazy mode, at rr_evaluate (after the per-pv prep): the rows the flux kernel stages.
int rr_ld_rows_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t esz = c.precision != RR_FP64 ? 4 : 8;
  const int64_t M = npv * c.npb;
  if (M > 0x7fffffffLL) return RR_ESIZE;
  int rc = grow_buf(&wk->rows, &wk->rows_cap, M * c.ng * esz);
  if (rc != RR_OK) return rc;
  if (wk->lazy == 2) return rr_ld_rows_direct_launch(ctx, wk, npv, st);
  const int nb = c.nk - 1;                         // buckets: lower k row ik in [0, nk-2]
  const int stride = ctx->nz | 1;
  // profiles + 2 x (8 NG) weight rows; NG = 4 when that leaves two blocks per SM, else 2
  const size_t smem4 = sizeof(double) * (RB * stride + 2 * 32 * ctx->nz);
  const size_t smem2 = sizeof(double) * (RB * stride + 2 * 16 * ctx->nz);
  const int NGsel = smem4 <= RR_ROWS_SMEM4_MAX ? 4 : 2;
  const size_t smem_b = NGsel == 4 ? smem4 : smem2;
  if (M >= 2048 && nb <= 4096 && smem_b <= 200 * 1024) {
    // bucketed builder
    const int64_t need = sizeof(int32_t) * (4 * (int64_t)nb + 4 + M);
    rc = grow_buf((void **)&wk->bk, &wk->bk_cap, need);
    if (rc != RR_OK) return rc;
    int *hist = wk->bk, *cursor = hist + nb, *offs = cursor + nb, *tileoff = offs + nb + 1,
        *list = tileoff + nb + 1;
    RR_CUDA(cudaMemsetAsync(hist, 0, sizeof(int32_t) * 2 * nb, st));
    const unsigned gb = (unsigned)((M + 255) / 256);
    rr_rows_hist<<<gb, 256, 0, st>>>(wk->pvb, M, c.npb, c.nkpb, hist);
    RR_LAUNCH_CHECK(ctx);
    rr_rows_scan<<<1, 32, 0, st>>>(nb, hist, offs, tileoff);
    RR_LAUNCH_CHECK(ctx);
    rr_rows_scatter<<<gb, 256, 0, st>>>(wk->pvb, M, c.npb, c.nkpb, offs, cursor, list);
    RR_LAUNCH_CHECK(ctx);
    const unsigned tiles_max = (unsigned)((M + RB - 1) / RB + nb);
#define RR_BUCKET_LAUNCH(TR, NG)                                                                   \
    do {                                                                                           \
      if (smem_b > 48 * 1024)                                                                      \
        RR_CUDA(cudaFuncSetAttribute(rr_ld_rows_bucket_kernel<TR, NG>,                             \
                                     cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem_b));   \
      rr_ld_rows_bucket_kernel<TR, NG><<<tiles_max, 256, smem_b, st>>>(                            \
          (const TR *)wk->ldp_src, ctx->d_W, (const int2 *)ctx->d_Wsup, wk->pvb, list, offs,      \
          tileoff, nb, (TR *)wk->rows,                                                            \
          c.npb, c.nkpb, c.ng, ctx->nz, stride);                                                   \
    } while (0)
    if (c.precision != RR_FP64) {
      if (NGsel == 4) RR_BUCKET_LAUNCH(float, 4); else RR_BUCKET_LAUNCH(float, 2);
    } else {
      if (NGsel == 4) RR_BUCKET_LAUNCH(double, 4); else RR_BUCKET_LAUNCH(double, 2);
    }
#undef RR_BUCKET_LAUNCH
    RR_LAUNCH_CHECK(ctx);
    return RR_OK;
  }
  const size_t smem = sizeof(double) * ctx->nz;
  const int gy_max = (c.ng + RT / 32 - 1) / (RT / 32);
  const int gy = (int)std::max<int64_t>(1, std::min<int64_t>(gy_max, (2 * 8 * ctx->sm_count + M - 1) / M));
  const dim3 grid((unsigned)M, (unsigned)gy);
  if (c.precision != RR_FP64)
    rr_ld_rows_kernel<float><<<grid, RT, smem, st>>>(
        (const float *)wk->ldp_src, ctx->d_W, (const int2 *)ctx->d_Wsup, wk->pvb, (float *)wk->rows,
        c.npb, c.nkpb, c.ng, ctx->nz);
  else
    rr_ld_rows_kernel<double><<<grid, RT, smem, st>>>(
        (const double *)wk->ldp_src, ctx->d_W, (const int2 *)ctx->d_Wsup, wk->pvb, (double *)wk->rows,
        c.npb, c.nkpb, c.ng, ctx->nz);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

// Diagnostics in lazy mode: the full table of the kept profile, built on demand.
int rr_ld_full_from_profile(rr_ctx *ctx, RRWork *wk, cudaStream_t st) {
  if (wk->have_full) return RR_OK;
  if (wk->table_npv <= 0 || wk->ldp_src != wk->ldp || !wk->ldp) return RR_ESTATE;
  const rr_config &c = ctx->cfg;
  const int64_t esz = c.precision != RR_FP64 ? 4 : 8;
  const int64_t npv = wk->table_npv;
  int rc = grow_buf(&wk->T, &wk->T_cap, npv * c.npb * (int64_t)c.nk * c.ng * esz);
  if (rc != RR_OK) return rc;
  const int64_t M = npv * c.npb;
  const int N = c.nk * c.ng, K = ctx->nz;
  dim3 grid((N + BN - 1) / BN, (unsigned)((M + BM - 1) / BM));
  if (c.precision != RR_FP64)
    rr_ld_table_kernel<float, float><<<grid, NT, 0, st>>>((const float *)wk->ldp, ctx->d_W,
                                                          (float *)wk->T, M, N, K);
  else
    rr_ld_table_kernel<double, double><<<grid, NT, 0, st>>>((const double *)wk->ldp, ctx->d_W,
                                                            (double *)wk->T, M, N, K);
  RR_LAUNCH_CHECK(ctx);
  wk->have_full = 1;
  return RR_OK;
}


// Named law -> profile (into the ctx-owned copy) + analytic Istar, then as rr_build_ld_table.
// Asynchronous on st: whether the law has a closed-form disc integral is known on the host from the
// law alone (only RR_LD_EXPONENTIAL has none: reading R6 then), and the kernel writes Istar straight
// into the ctx-owned buffer; buffers grow (cudaMalloc) only when a larger npv arrives.
int rr_ld_law_launch(rr_ctx *ctx, RRWork *wk, int law, const double *d_ldc, int nc, int64_t npv,
                     cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t esz = c.precision != RR_FP64 ? 4 : 8;
  const int64_t M = npv * c.npb;
  const bool full = !(ctx->table_mode != RR_TABLE_FULL && ctx->nz <= 2000);
  wk->table_npv = -1;
  int rc = grow_buf(&wk->ldp, &wk->ldp_cap, M * ctx->nz * esz);
  if (rc == RR_OK) rc = grow_buf(&wk->istar, &wk->istar_cap, M * esz);
  if (rc != RR_OK) return rc;
  const bool closed = law != RR_LD_EXPONENTIAL;
  const int64_t n = M * ctx->nz;
  const unsigned grid = (unsigned)((n + 255) / 256);
  if (c.precision != RR_FP64)
    rr_ld_law_kernel<float><<<grid, 256, 0, st>>>(law, d_ldc, nc, ctx->d_mu, M, ctx->nz,
                                                  (float *)wk->ldp,
                                                  closed ? (float *)wk->istar : nullptr);
  else
    rr_ld_law_kernel<double><<<grid, 256, 0, st>>>(law, d_ldc, nc, ctx->d_mu, M, ctx->nz,
                                                   (double *)wk->ldp,
                                                   closed ? (double *)wk->istar : nullptr);
  RR_LAUNCH_CHECK(ctx);
  const void *ist = closed ? wk->istar : nullptr;  // no closed form: discretised integral (R6)
  if (!full)
    rc = rr_ld_profile_launch(ctx, wk, wk->ldp, ist, npv, 0, st);
  else
    rc = rr_ld_table_launch(ctx, wk, wk->ldp, ist, npv, st);
  if (rc == RR_OK && wk->lazy) wk->ldp_src = wk->ldp;
  return rc;
}
