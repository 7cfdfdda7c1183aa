// rr_geometry.cu - step a0 (model initialisation, once per rr_create): the z grid and the (k,g)
// geometry weight tensor W[nk][ng][nz], on the device, fp64.
//   z grid:   PAPER.md:83-90 (section 3.1.1): constant dz on [0,zcut], constant dmu on [zcut,1];
//             zm = mean of the bin edges (reading R1), mu = sqrt(1 - zm^2).
//   weights:  PAPER.md:59 and Fig. 1: w_j(c,k) = area of annulus j covered by the planet divided by
//             the whole covered area a(c,k); tabulated on k_ik x g_ig with
//             c = g (1+k).  Reading R5: the g = 1 node (a = 0) takes the limit, all weight in the
//             outermost annulus.
#include "rr_common.cuh"
#include "rr_math.cuh"

// Area common to two discs of radii r1, r2 with centres d apart (textbook lens; PAPER.md:57, :69
// "cheap to calculate analytically").  Partial overlap = two circular sectors minus the kite;
// the sector half-angles are taken with atan2 of (4 x triangle area, d^2 + r_a^2 - r_b^2), which
// stays accurate where the planet's limb touches a circle (reading R9).
__device__ double rr_lens_area(double r1, double r2, double d) {
  if (d >= r1 + r2) return 0.0;
  double rmin = fmin(r1, r2);
  if (d <= fabs(r1 - r2)) return RR_PI * rmin * rmin;
  double kite = sqrt((r1 + r2 - d) * (d + r1 - r2) * (d - r1 + r2) * (d + r1 + r2));
  double th1 = atan2(kite, (d - r2) * (d + r2) + r1 * r1);
  double th2 = atan2(kite, (d - r1) * (d + r1) + r2 * r2);
  return r1 * r1 * th1 + r2 * r2 * th2 - 0.5 * kite;
}

__global__ void rr_zgrid_kernel(double zcut, int nzin, int nzlimb, double *ze, double *zm,
                                double *mu, double *q) {
  int nz = nzin + nzlimb;
  int j = blockIdx.x * blockDim.x + threadIdx.x;
  if (j > nz) return;
  auto edge = [&](int i) -> double {
    if (i <= nzin) return (double)i * zcut / (double)nzin;
    if (i >= nz) return 1.0;
    // __dmul_rn / __dadd_rn: no FMA contraction, so that 1 - x^2 near the limb (where it is
    // ill-conditioned) rounds exactly as the plain formula does
    double mucut = sqrt(__dadd_rn(1.0, -__dmul_rn(zcut, zcut)));
    double mue = mucut * (1.0 - (double)(i - nzin) / (double)nzlimb);
    return sqrt(__dadd_rn(1.0, -__dmul_rn(mue, mue)));
  };
  double lo = edge(j);
  ze[j] = lo;
  if (j < nz) {
    double hi = edge(j + 1);
    double m = 0.5 * (lo + hi);
    zm[j] = m;
    mu[j] = sqrt(__dadd_rn(1.0, -__dmul_rn(m, m)));
    q[j] = RR_PI * (hi * hi - lo * lo);   // annulus area: Istar = sum_j q_j ldp_j (reading R6)
  }
}

// One thread per weight.  W[(ik*ng + ig)*nz + j].
__global__ void rr_weights_kernel(int nk, double k0, double k1, int ng, int nz,
                                  const double *__restrict__ ze, double *__restrict__ W) {
  int64_t idx = (int64_t)blockIdx.x * blockDim.x + threadIdx.x;
  int64_t total = (int64_t)nk * ng * nz;
  if (idx >= total) return;
  int j = (int)(idx % nz);
  int ig = (int)((idx / nz) % ng);
  int ik = (int)(idx / ((int64_t)nz * ng));
  double dk = (k1 - k0) / (double)(nk - 1);
  double k = k0 + ik * dk;
  double g = (ig == ng - 1) ? 1.0 : (double)ig / (double)(ng - 1);
  double c = g * (1.0 + k);
  double a = rr_lens_area(1.0, k, c);
  double w;
  if (!(a > 0.0)) {
    w = (j == nz - 1) ? 1.0 : 0.0;
  } else {
    double hi = rr_lens_area(ze[j + 1], k, c);
    double lo = (ze[j] > 0.0) ? rr_lens_area(ze[j], k, c) : 0.0;
    w = (hi - lo) / a;
  }
  W[idx] = w;
}

// The same area for the direct-model rows (evaluate-time path): the hot path's own sqrt and atan2.
__device__ __forceinline__ double rr_lens_area_fast(double r1, double r2, double d) {
  if (d >= r1 + r2) return 0.0;
  const double rmin = fmin(r1, r2);
  if (d <= fabs(r1 - r2)) return RR_PI * rmin * rmin;
  const double kite = rr_sqrt((r1 + r2 - d) * (d + r1 - r2) * (d - r1 + r2) * (d + r1 + r2));
  const double th1 = rr_atan2_pos(kite, fma(d - r2, d + r2, r1 * r1));
  const double th2 = rr_atan2_pos(kite, fma(d - r1, d + r1, r2 * r2));
  return fma(r1 * r1, th1, fma(r2 * r2, th2, -0.5 * kite));
}

// ---- direct model on the device -------------------------------
// The paper's default setting: no k grid.  For every (pv, passband) row the weights are computed at
// the pv's OWN k, `dg, w = calculate_weights(k, ze, ng)`, and contracted at once with the profile,
// `ldw = dot(w, ldp)`:
//   ldw[ig] = sum_j [A(ze[j+1]) - A(ze[j])] ldp[j] / a(c,k),   c = g_ig (1+k),  A(r) = lens(r, k, c)
//           = sum_{e=1..nz} A(ze[e]) D_e / a(c,k),   D_e = ldp[e-1] - ldp[e] (e < nz), D_nz = ldp[nz-1]
// (summation by parts: one lens area per annulus EDGE, no neighbour exchange).  ig = ng-1 takes the
// limit of reading R5.  One block per row, one warp per g node, lanes over edges; fp64 throughout.
// The result has the layout of the lazy rows, so the flux kernel is unchanged; there is no k
// interpolation error and no [k0, k1] limit.
template <typename TR>
__global__ void __launch_bounds__(256)
rr_ld_rows_direct_kernel(const TR *__restrict__ ldp, const double *__restrict__ ze,
                         const RRPvBand *__restrict__ pvb, TR *__restrict__ rows, int npb, int nkpb,
                         int ng, int nz) {
  extern __shared__ double sh[];                 // D[nz+1] (index = edge) | ze[nz+1] | a[ng]
  double *D = sh, *zes = sh + nz + 1, *area = sh + 2 * (nz + 1);
  const int64_t row = blockIdx.x;
  const int64_t v = row / npb;
  const int pb = (int)(row - v * npb);
  const double k = pvb[v * nkpb + (nkpb == 1 ? 0 : pb)].kw;   // the k the weights are taken at
  const TR *pr = ldp + row * nz;
  for (int e = threadIdx.x; e <= nz; e += 256) {
    zes[e] = ze[e];
    D[e] = (e == 0) ? 0.0 : (e < nz ? (double)pr[e - 1] - (double)pr[e] : (double)pr[nz - 1]);
  }
  // the whole occulted area a(c_ig, k) of every node: one thread per node, not one warp per node
  for (int ig = threadIdx.x; ig < ng - 1; ig += 256)
    area[ig] = rr_lens_area_fast(1.0, k, ((double)ig / (double)(ng - 1)) * (1.0 + k));
  __syncthreads();
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int ig = warp; ig < ng; ig += 8) {
    double out;
    if (ig == ng - 1) {
      out = (double)pr[nz - 1];                  // reading R5: all weight in the outermost annulus
    } else {
      const double c = ((double)ig / (double)(ng - 1)) * (1.0 + k);
      // edges are sorted: ze[e] <= c-k have A = 0; ze[e] >= c+k have A = pi k^2 and their D_e
      // telescope to ldp[e_hi - 1]; only the edges in between need a lens area
      int nlo = 0, nhi = 0;
      for (int e = 1 + lane; e <= nz; e += 32) {
        nlo += zes[e] <= c - k;
        nhi += zes[e] < c + k;
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        nlo += __shfl_xor_sync(0xffffffffu, nlo, o);
        nhi += __shfl_xor_sync(0xffffffffu, nhi, o);
      }
      const int e_lo = 1 + nlo, e_hi = 1 + nhi;          // partial edges: e_lo <= e < e_hi
      double s = 0.0;
      for (int e = e_lo + lane; e < e_hi; e += 32) s = fma(rr_lens_area_fast(zes[e], k, c), D[e], s);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
      if (e_hi <= nz) s = fma(RR_PI * k * k, (double)pr[e_hi - 1], s);
      out = s / area[ig];
    }
    if (lane == 0) rows[row * ng + ig] = (TR)out;
  }
}

int rr_ld_rows_direct_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t M = npv * c.npb;
  if (M > 0x7fffffffLL) return RR_ESIZE;
  const size_t smem = sizeof(double) * (2 * (ctx->nz + 1) + c.ng);   // <= 77 kB (nz <= 2000, ng <= 5600)
  if (smem > 48 * 1024) {
    RR_CUDA(cudaFuncSetAttribute(rr_ld_rows_direct_kernel<float>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    RR_CUDA(cudaFuncSetAttribute(rr_ld_rows_direct_kernel<double>,
                                 cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  }
  if (c.precision != RR_FP64)
    rr_ld_rows_direct_kernel<float><<<(unsigned)M, 256, smem, st>>>(
        (const float *)wk->ldp_src, ctx->d_ze, wk->pvb, (float *)wk->rows, c.npb, c.nkpb, c.ng,
        ctx->nz);
  else
    rr_ld_rows_direct_kernel<double><<<(unsigned)M, 256, smem, st>>>(
        (const double *)wk->ldp_src, ctx->d_ze, wk->pvb, (double *)wk->rows, c.npb, c.nkpb, c.ng,
        ctx->nz);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

// ---- small-planet approximation (reading R14) ---------------------
// Rows whose weight radius kw is <= the threshold take, at node g_ig, the profile's value at the
// planet's centre z = g_ig (1+kw): linear interpolation of ldp over the bin means zm, constant
// before the first and after the last node.  Runs after the row builder of the current mode and
// overwrites those rows (one warp per row, lanes over g nodes, binary search in zm).
template <typename TR>
__global__ void __launch_bounds__(256)
rr_ld_rows_small_kernel(const TR *__restrict__ ldp, const double *__restrict__ zm,
                        const RRPvBand *__restrict__ pvb, TR *__restrict__ rows, double k_small,
                        int64_t M, int npb, int nkpb, int ng, int nz) {
  const int64_t row = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (row >= M) return;
  const int64_t v = row / npb;
  const int pb = (int)(row - v * npb);
  const double k = pvb[v * nkpb + (nkpb == 1 ? 0 : pb)].kw;
  if (!(k <= k_small)) return;
  const TR *pr = ldp + row * nz;
  for (int ig = lane; ig < ng; ig += 32) {
    const double z = (ig == ng - 1) ? 1.0 + k : ((double)ig / (double)(ng - 1)) * (1.0 + k);
    double out;
    if (z <= zm[0]) {
      out = (double)pr[0];
    } else if (z >= zm[nz - 1]) {
      out = (double)pr[nz - 1];
    } else {
      int lo = 0, hi = nz - 1;                     // zm[lo] <= z < zm[hi]
      while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (zm[mid] <= z) lo = mid; else hi = mid;
      }
      const double a = (z - zm[lo]) / (zm[lo + 1] - zm[lo]);
      out = (1.0 - a) * (double)pr[lo] + a * (double)pr[lo + 1];
    }
    rows[row * ng + ig] = (TR)out;
  }
}

int rr_ld_rows_small_launch(rr_ctx *ctx, RRWork *wk, int64_t npv, cudaStream_t st) {
  const rr_config &c = ctx->cfg;
  const int64_t M = npv * c.npb;
  const unsigned grid = (unsigned)((M * 32 + 255) / 256);
  if (c.precision != RR_FP64)
    rr_ld_rows_small_kernel<float><<<grid, 256, 0, st>>>(
        (const float *)wk->ldp_src, ctx->d_zm, wk->pvb, (float *)wk->rows, ctx->k_small, M, c.npb,
        c.nkpb, c.ng, ctx->nz);
  else
    rr_ld_rows_small_kernel<double><<<grid, 256, 0, st>>>(
        (const double *)wk->ldp_src, ctx->d_zm, wk->pvb, (double *)wk->rows, ctx->k_small, M, c.npb,
        c.nkpb, c.ng, ctx->nz);
  RR_LAUNCH_CHECK(ctx);
  return RR_OK;
}

// Support of every weight row W[ik][ig][.]: the planet at separation g (1+k) covers only the annuli
// between c - k and c + k, so the row is zero outside [jlo, jhi).  The row builders of
// kernel 1 skip the zeros (adding w = 0 terms changes no sum).
__global__ void rr_support_kernel(const double *__restrict__ W, int nrows, int nz,
                                  int2 *__restrict__ sup) {
  const int r = blockIdx.x * blockDim.x + threadIdx.x;
  if (r >= nrows) return;
  const double *w = W + (int64_t)r * nz;
  int lo = nz, hi = 0;
  for (int j = 0; j < nz; ++j)
    if (w[j] != 0.0) {
      lo = min(lo, j);
      hi = j + 1;
    }
  if (lo >= hi) { lo = 0; hi = nz; }               // (cannot happen: the weights sum to 1)
  sup[r] = make_int2(lo, hi);
}

int rr_geometry_build(rr_ctx *ctx) {
  const rr_config &c = ctx->cfg;
  int nz = ctx->nz;
  RR_CUDA(cudaMalloc(&ctx->d_ze, sizeof(double) * (nz + 1)));
  RR_CUDA(cudaMalloc(&ctx->d_zm, sizeof(double) * nz));
  RR_CUDA(cudaMalloc(&ctx->d_mu, sizeof(double) * nz));
  RR_CUDA(cudaMalloc(&ctx->d_q, sizeof(double) * nz));
  int64_t nW = (int64_t)c.nk * c.ng * nz;
  RR_CUDA(cudaMalloc(&ctx->d_W, sizeof(double) * nW));
  rr_zgrid_kernel<<<(nz + 1 + 127) / 128, 128>>>(c.zcut, c.nzin, c.nzlimb, ctx->d_ze, ctx->d_zm,
                                                  ctx->d_mu, ctx->d_q);
  RR_LAUNCH_CHECK(ctx);
  rr_weights_kernel<<<(unsigned)((nW + 255) / 256), 256>>>(c.nk, c.k0, c.k1, c.ng, nz, ctx->d_ze,
                                                           ctx->d_W);
  RR_LAUNCH_CHECK(ctx);
  RR_CUDA(cudaMalloc(&ctx->d_Wsup, sizeof(int2) * (size_t)c.nk * c.ng));
  rr_support_kernel<<<(c.nk * c.ng + 127) / 128, 128>>>(ctx->d_W, c.nk * c.ng, nz,
                                                        (int2 *)ctx->d_Wsup);
  RR_LAUNCH_CHECK(ctx);
  ctx->h_ze.resize(nz + 1);
  ctx->h_mu.resize(nz);
  RR_CUDA(cudaMemcpy(ctx->h_ze.data(), ctx->d_ze, sizeof(double) * (nz + 1),
                     cudaMemcpyDeviceToHost));
  RR_CUDA(cudaMemcpy(ctx->h_mu.data(), ctx->d_mu, sizeof(double) * nz, cudaMemcpyDeviceToHost));
  return RR_OK;
}
