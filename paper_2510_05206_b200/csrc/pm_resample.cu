// pm_resample.cu -- NEXT-4: sheet-based particle resampling, trilinear variant ("increasing the
// number of particles in the density computation by introducing artificial particles, whose locations are
// determined by interpolating the displacement of the original particles in Lagrangian space"; Table 5
// n_resample :411 "copies of each particle per dim."; reading R21 in DESIGN.md).
//
// Input: N = n_p^3 positions in Lagrangian (C) order, particle (i,j,k) started at q = (i,j,k) L/n_p.  Output:
// (r n_p)^3 positions X' = q' + trilinear interpolation of Psi = minimum-image(X - q) between the 8 Lagrangian
// neighbours of q' = (i',j',k') L/(r n_p), wrapped into [0, L), C order.  A structured gather: no binning.
// HBM-bound on the 12 r^3 N bytes written (the 8 neighbours of a refined cell are shared by r^3 outputs).
#include "pm_internal.cuh"

namespace pmf {

namespace {

__global__ void __launch_bounds__(256) k_sheet_resample(const float* __restrict__ pos, int n_p, int r, double box,
                                                        float* __restrict__ out) {
  const int nf = n_p * r;
  const int64_t total = (int64_t)nf * nf * nf;
  const double dq = box / n_p, dqf = box / nf, rinv = 1.0 / r;
  for (int64_t o = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; o < total; o += (int64_t)gridDim.x * blockDim.x) {
    const int kf = (int)(o % nf), jf = (int)((o / nf) % nf), jf0 = (int)(o / ((int64_t)nf * nf));
    const int fi[3] = {jf0, jf, kf};
    int i0[3];
    double t[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      i0[a] = fi[a] / r;
      t[a] = (fi[a] - i0[a] * r) * rinv;
    }
    double acc[3] = {0.0, 0.0, 0.0};
#pragma unroll
    for (int dx = 0; dx < 2; ++dx)
#pragma unroll
      for (int dy = 0; dy < 2; ++dy)
#pragma unroll
        for (int dz = 0; dz < 2; ++dz) {
          int ii[3] = {i0[0] + dx, i0[1] + dy, i0[2] + dz};
          const double w = (dx ? t[0] : 1.0 - t[0]) * (dy ? t[1] : 1.0 - t[1]) * (dz ? t[2] : 1.0 - t[2]);
          if (w == 0.0) continue;
#pragma unroll
          for (int a = 0; a < 3; ++a) ii[a] -= ii[a] >= n_p ? n_p : 0;
          const float* p = pos + 3 * (((int64_t)ii[0] * n_p + ii[1]) * n_p + ii[2]);
#pragma unroll
          for (int a = 0; a < 3; ++a) {
            double psi = (double)__ldg(p + a) - ii[a] * dq;
            psi -= box * rint(psi / box);  // minimum image
            acc[a] += w * psi;
          }
        }
#pragma unroll
    for (int a = 0; a < 3; ++a) {
      double x = fi[a] * dqf + acc[a];
      x -= box * floor(x / box);
      float xf = (float)x;
      if (xf >= (float)box || xf < 0.f) xf = 0.f;  // rounded up to L
      out[3 * o + a] = xf;
    }
  }
}

}  // namespace

int launch_sheet_resample(Ctx* c, const float* pos, int n_p, int r, float* out, cudaStream_t st) {
  const int64_t total = (int64_t)n_p * r * n_p * r * n_p * r;
  int64_t grid = (total + 255) / 256;
  const int64_t cap = (int64_t)c->num_sms * 16;
  if (grid > cap) grid = cap;
  k_sheet_resample<<<(unsigned)grid, 256, 0, st>>>(pos, n_p, r, c->p.box, out);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
