// rr_geometry.cu - step a0 (model initialisation, once per rr_create): the z grid and the (k,g)
// geometry weight tensor W[nk][ng][nz], on the device, fp64.
//   z grid:   PAPER.md:83-90 (section 3.1.1): constant dz on [0,zcut], constant dmu on [zcut,1];
//             zm = mean of the bin edges (reading R1), mu = sqrt(1 - zm^2).
//   weights:  PAPER.md:59 and Fig. 1: w_j(c,k) = area of annulus j covered by the planet divided by
//             the whole covered area a(c,k); tabulated on k_ik x g_ig with
//             c = g (1+k).  Reading R5: the g = 1 node (a = 0) takes the limit, all weight in the
//             outermost annulus.
#include "rr_common.cuh"

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
  ctx->h_ze.resize(nz + 1);
  ctx->h_mu.resize(nz);
  RR_CUDA(cudaMemcpy(ctx->h_ze.data(), ctx->d_ze, sizeof(double) * (nz + 1),
                     cudaMemcpyDeviceToHost));
  RR_CUDA(cudaMemcpy(ctx->h_mu.data(), ctx->d_mu, sizeof(double) * nz, cudaMemcpyDeviceToHost));
  return RR_OK;
}
