// pm_power.cu -- NEXT-4: shell-binned (cross-)power spectrum of the interlaced, deconvolved PM density
// ("(cross-)power spectrum routine"; readings R20 in DESIGN.md):
//   delta_hat = 1/2 [d1 + e^{-ik.s} d2] (two-grid interlacing, R1 / R9) / W~(n) (ONE power of the assignment window:
//   one assignment, no gather), P(bin) = V <Re(deltaA_hat conj deltaB_hat)> / G^2 over the modes of the FULL Fourier
//   cube with b + 1/2 <= |n| < b + 3/2.  The spectra are cuFFT's 3-D R2C transforms of the particle-count meshes;
//   delta = (G/N) rho - 1 differs from rho only in n = 0 (never binned) and by the factor G/N applied at the end.
#include "pm_internal.cuh"

namespace pmf {

namespace {

constexpr int PB = 256;

struct PTabs {
  const double *win1, *pc, *ps;  // W~ per axis (one power), interlace phase
  int m, hz;
};

__device__ __forceinline__ double2 cmuld(double2 a, double2 b) {
  return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// acc: [3][nbins] = {n_modes, sum |n|, sum Re(A conj B)} (weights: multiplicity of the stored half)
__global__ void __launch_bounds__(PB) k_power_bins(PTabs t, const float2* __restrict__ a1,
                                                   const float2* __restrict__ a2, const float2* __restrict__ b1,
                                                   const float2* __restrict__ b2, int deconvolve, int nbins,
                                                   double* __restrict__ acc) {
  extern __shared__ double s_bin[];  // [3 * nbins]
  for (int j = threadIdx.x; j < 3 * nbins; j += PB) s_bin[j] = 0.0;
  __syncthreads();
  const int m = t.m, hz = t.hz;
  const int64_t rows = (int64_t)m * m;
  for (int64_t row = blockIdx.x; row < rows; row += gridDim.x) {
    const int ix = (int)(row / m), iy = (int)(row - (int64_t)ix * m);
    const int nx = ix < (m + 1) / 2 ? ix : ix - m, ny = iy < (m + 1) / 2 ? iy : iy - m;
    const double wxy = t.win1[ix] * t.win1[iy];
    const double2 pxy = cmuld(make_double2(t.pc[ix], t.ps[ix]), make_double2(t.pc[iy], t.ps[iy]));
    const size_t base = (size_t)row * hz;
    for (int iz = threadIdx.x; iz < hz; iz += PB) {
      const double kn = sqrt((double)nx * nx + (double)ny * ny + (double)iz * iz);
      const int b = (int)floor(kn - 0.5);
      if (b < 0 || b >= nbins) continue;
      const double mult = (iz == 0 || 2 * iz == m) ? 1.0 : 2.0;
      const double2 pz = make_double2(t.pc[iz], t.ps[iz]);
      const double2 ph = cmuld(pxy, pz);
      float2 v = a1[base + iz];
      double2 A = make_double2(v.x, v.y);
      if (a2) {
        v = a2[base + iz];
        const double2 q = cmuld(ph, make_double2(v.x, v.y));
        A = make_double2(0.5 * (A.x + q.x), 0.5 * (A.y + q.y));
      }
      double2 B = A;
      if (b1) {
        v = b1[base + iz];
        B = make_double2(v.x, v.y);
        if (b2) {
          v = b2[base + iz];
          const double2 q = cmuld(ph, make_double2(v.x, v.y));
          B = make_double2(0.5 * (B.x + q.x), 0.5 * (B.y + q.y));
        }
      }
      double pw = A.x * B.x + A.y * B.y;
      if (deconvolve) {
        const double w = wxy * t.win1[iz];
        pw /= w * w;
      }
      atomicAdd(&s_bin[b], mult);
      atomicAdd(&s_bin[nbins + b], mult * kn);
      atomicAdd(&s_bin[2 * nbins + b], mult * pw);
    }
  }
  __syncthreads();
  for (int j = threadIdx.x; j < 3 * nbins; j += PB)
    if (s_bin[j] != 0.0) atomicAdd(&acc[j], s_bin[j]);
}

__global__ void k_power_finish(int nbins, const double* __restrict__ acc, double kf, double pnorm,
                               double* __restrict__ k_mean, double* __restrict__ power, double* __restrict__ n_modes) {
  const int b = blockIdx.x * blockDim.x + threadIdx.x;
  if (b >= nbins) return;
  const double cnt = acc[b];
  const double safe = cnt > 0.0 ? cnt : 1.0;
  n_modes[b] = cnt;
  k_mean[b] = kf * acc[nbins + b] / safe;
  power[b] = pnorm * acc[2 * nbins + b] / safe;
}

}  // namespace

int launch_power_bins(Ctx* c, const float2* a1, const float2* a2, const float2* b1, const float2* b2, bool deconvolve,
                      int nbins, double* acc, cudaStream_t st) {
  PTabs t;
  t.win1 = c->tab_win1;
  t.pc = c->tab_cos;
  t.ps = c->tab_sin;
  t.m = c->mg;
  t.hz = c->mg / 2 + 1;
  const size_t smem = sizeof(double) * 3 * (size_t)nbins;
  int occ = 0;
  PM_TRY(kernel_occupancy(c, (const void*)k_power_bins, PB, smem, &occ));
  int64_t grid = (int64_t)c->num_sms * (occ > 4 ? 4 : occ);
  if (grid > (int64_t)c->mg * c->mg) grid = (int64_t)c->mg * c->mg;
  k_power_bins<<<(unsigned)grid, PB, smem, st>>>(t, a1, a2, b1, b2, deconvolve ? 1 : 0, nbins, acc);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

int launch_power_finish(Ctx* c, int nbins, const double* acc, double kf, double pnorm, double* k_mean, double* power,
                        double* n_modes, cudaStream_t st) {
  k_power_finish<<<(nbins + 127) / 128, 128, 0, st>>>(nbins, acc, kf, pnorm, k_mean, power, n_modes);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
