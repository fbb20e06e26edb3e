// pm_kspace.cu -- a3 / a7 / a10: the Fourier-space kernel (K3, K6) and its transpose.
//
// forward : ghat_a(n) = S_a(n) dhat(n),  S_a = -i D_a(n_a) * green(n),
//           green(n) = coeff_eff / (Lap(n) * win(n_x) win(n_y) win(n_z)),  green(0) = 0 (R7),
//           dhat = 1/2 [d1 + e^{-ik.s} d2] when a second (interlaced) spectrum is given (R1, R9).
//   PM    (Tables 1-2): D = Table 2 gradient symbol / Delta, Lap = sum_a l(theta_a)/Delta^2,
//           win = sinc^p(n/m)^deconv_pow.
//   NUFFT: D = k_a, Lap = -|k|^2, win = phi_hat(n_a)^2, win = 0 marks a dropped mode (R8).
// transpose: q(n) = sum_a conj(S_a) gbar_hat_a(n).
// The per-axis tables are fp64 (computed on the host at pm_create); the multiplier is formed in fp64 and
// applied to the fp32 spectrum.  HBM-bound: 8 B read + 24 B written per half-complex mode (forward).
#include "pm_internal.cuh"

namespace pmf {

struct KTabs {
  const double *grad, *lap, *win, *pc, *ps;
  int m, hz;
};

constexpr int KS_BLOCK = 128;
constexpr int KS_ROWS = 4;  // (ix, iy .. iy+3) rows per CTA: 4 independent loads in flight per thread, one table read

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// per-row (ix, iy) factors of the multiplier
struct RowFac {
  double lxy, wxy, dxv, dyv;
  float2 pxy;
};
__device__ __forceinline__ RowFac row_factors(const KTabs& t, int ix, int iy, bool phase, float sgn) {
  RowFac r;
  r.lxy = t.lap[ix] + t.lap[iy];
  r.wxy = t.win[ix] * t.win[iy];
  r.dxv = t.grad[ix];
  r.dyv = t.grad[iy];
  r.pxy = make_float2(1.f, 0.f);
  if (phase) {
    const double cr = t.pc[ix] * t.pc[iy] - t.ps[ix] * t.ps[iy];
    const double ci = t.pc[ix] * t.ps[iy] + t.ps[ix] * t.pc[iy];
    r.pxy = make_float2((float)cr, sgn * (float)ci);
  }
  return r;
}

// One CTA per KS_ROWS consecutive (ix, iy) rows of the half-complex grid (m is a multiple of 4, so the rows of
// a CTA share ix); threads run along iz.
__global__ void __launch_bounds__(KS_BLOCK) k_kspace_fwd(KTabs t, const float2* __restrict__ d1,
                                                         const float2* __restrict__ d2,
                                                         float2* __restrict__ g0, float2* __restrict__ g1,
                                                         float2* __restrict__ g2, double coeff_eff) {
  const int row0 = blockIdx.x * KS_ROWS;
  const int ix = row0 / t.m, iy0 = row0 - ix * t.m;
  RowFac rf[KS_ROWS];
#pragma unroll
  for (int r = 0; r < KS_ROWS; ++r) rf[r] = row_factors(t, ix, iy0 + r, d2 != nullptr, 1.f);
  const size_t base = (size_t)row0 * t.hz;
  for (int iz = threadIdx.x; iz < t.hz; iz += KS_BLOCK) {
    float2 d[KS_ROWS], e[KS_ROWS];
#pragma unroll
    for (int r = 0; r < KS_ROWS; ++r) d[r] = __ldcs(d1 + base + (size_t)r * t.hz + iz);
    if (d2) {
#pragma unroll
      for (int r = 0; r < KS_ROWS; ++r) e[r] = __ldcs(d2 + base + (size_t)r * t.hz + iz);
    }
    const double lz = t.lap[iz], wz = t.win[iz], gz = t.grad[iz];
    float2 pz = make_float2(1.f, 0.f);
    if (d2) pz = make_float2((float)t.pc[iz], (float)t.ps[iz]);
#pragma unroll
    for (int r = 0; r < KS_ROWS; ++r) {
      const double den = (rf[r].lxy + lz) * (rf[r].wxy * wz);
      const double green = (den != 0.0) ? coeff_eff / den : 0.0;  // n = 0 and dropped modes -> 0
      float2 v = d[r];
      if (d2) {
        const float2 q = cmul(cmul(rf[r].pxy, pz), e[r]);
        v = make_float2(0.5f * (v.x + q.x), 0.5f * (v.y + q.y));
      }
      // -i D green (re + i im) = D green (im - i re)
      const float mx = (float)(rf[r].dxv * green), my = (float)(rf[r].dyv * green), mz = (float)(gz * green);
      const size_t o = base + (size_t)r * t.hz + iz;
      g0[o] = make_float2(mx * v.y, -mx * v.x);
      g1[o] = make_float2(my * v.y, -my * v.x);
      g2[o] = make_float2(mz * v.y, -mz * v.x);
    }
  }
}

__global__ void __launch_bounds__(KS_BLOCK) k_kspace_tr(KTabs t, const float2* __restrict__ g0,
                                                        const float2* __restrict__ g1,
                                                        const float2* __restrict__ g2, float2* __restrict__ q1,
                                                        float2* __restrict__ q2, double coeff_eff) {
  const int row0 = blockIdx.x * KS_ROWS;
  const int ix = row0 / t.m, iy0 = row0 - ix * t.m;
  RowFac rf[KS_ROWS];
#pragma unroll
  for (int r = 0; r < KS_ROWS; ++r) rf[r] = row_factors(t, ix, iy0 + r, q2 != nullptr, -1.f);  // conj of the phase
  const size_t base = (size_t)row0 * t.hz;
  for (int iz = threadIdx.x; iz < t.hz; iz += KS_BLOCK) {
    float2 a[KS_ROWS], b[KS_ROWS], c[KS_ROWS];
#pragma unroll
    for (int r = 0; r < KS_ROWS; ++r) {
      const size_t o = base + (size_t)r * t.hz + iz;
      a[r] = __ldcs(g0 + o);
      b[r] = __ldcs(g1 + o);
      c[r] = __ldcs(g2 + o);
    }
    const double lz = t.lap[iz], wz = t.win[iz], gz = t.grad[iz];
    float2 pz = make_float2(1.f, 0.f);
    if (q2) pz = make_float2((float)t.pc[iz], (float)-t.ps[iz]);
#pragma unroll
    for (int r = 0; r < KS_ROWS; ++r) {
      const double den = (rf[r].lxy + lz) * (rf[r].wxy * wz);
      const double green = (den != 0.0) ? coeff_eff / den : 0.0;
      const float mx = (float)(rf[r].dxv * green), my = (float)(rf[r].dyv * green), mz = (float)(gz * green);
      // conj(S_a) = +i D_a green:  q = i * sum_a m_a (re_a + i im_a)
      float2 q = make_float2(-(mx * a[r].y + my * b[r].y + mz * c[r].y), mx * a[r].x + my * b[r].x + mz * c[r].x);
      const size_t o = base + (size_t)r * t.hz + iz;
      if (q2) {
        q.x *= 0.5f;
        q.y *= 0.5f;
        q2[o] = cmul(cmul(rf[r].pxy, pz), q);
      }
      q1[o] = q;
    }
  }
}

// Potential variant (no gradient symbol; PM_FLAG_GRAD_REAL / PM_FLAG_KERNEL_GRAD):
//   q = green * (d2 ? 1/2 [d1 + e^{-ik.s} d2] : d1)
__global__ void __launch_bounds__(KS_BLOCK) k_kspace_scalar(KTabs t, const float2* __restrict__ d1,
                                                            const float2* __restrict__ d2, float2* __restrict__ q1,
                                                            double coeff_eff) {
  const int row0 = blockIdx.x * KS_ROWS;
  const int ix = row0 / t.m, iy0 = row0 - ix * t.m;
  RowFac rf[KS_ROWS];
#pragma unroll
  for (int r = 0; r < KS_ROWS; ++r) rf[r] = row_factors(t, ix, iy0 + r, d2 != nullptr, 1.f);
  const size_t base = (size_t)row0 * t.hz;
  for (int iz = threadIdx.x; iz < t.hz; iz += KS_BLOCK) {
    const double lz = t.lap[iz], wz = t.win[iz];
    float2 pz = make_float2(1.f, 0.f);
    if (d2) pz = make_float2((float)t.pc[iz], (float)t.ps[iz]);
#pragma unroll
    for (int r = 0; r < KS_ROWS; ++r) {
      const size_t o = base + (size_t)r * t.hz + iz;
      const double den = (rf[r].lxy + lz) * (rf[r].wxy * wz);
      const float green = (float)((den != 0.0) ? coeff_eff / den : 0.0);
      float2 v = __ldcs(d1 + o);
      if (d2) {
        const float2 q = cmul(cmul(rf[r].pxy, pz), __ldcs(d2 + o));
        v = make_float2(0.5f * (v.x + q.x), 0.5f * (v.y + q.y));
      }
      q1[o] = make_float2(green * v.x, green * v.y);
    }
  }
}

static KTabs tabs_of(const Ctx* c) {
  KTabs t;
  t.grad = c->tab_grad;
  t.lap = c->tab_lap;
  t.win = c->tab_win;
  t.pc = c->tab_cos;
  t.ps = c->tab_sin;
  t.m = c->mg;
  t.hz = c->mg / 2 + 1;
  return t;
}

int launch_kspace_forward(Ctx* c, const float2* d1, const float2* d2, float2* const ghat[3], double coeff_eff,
                          cudaStream_t st) {
  k_kspace_fwd<<<c->mg * c->mg / KS_ROWS, KS_BLOCK, 0, st>>>(tabs_of(c), d1, d2, ghat[0], ghat[1], ghat[2], coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

int launch_kspace_transpose(Ctx* c, const float2* const gh[3], float2* q1, float2* q2, double coeff_eff,
                            cudaStream_t st) {
  k_kspace_tr<<<c->mg * c->mg / KS_ROWS, KS_BLOCK, 0, st>>>(tabs_of(c), gh[0], gh[1], gh[2], q1, q2, coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

int launch_kspace_scalar(Ctx* c, const float2* d1, const float2* d2, float2* q1, double coeff_eff, cudaStream_t st) {
  k_kspace_scalar<<<c->mg * c->mg / KS_ROWS, KS_BLOCK, 0, st>>>(tabs_of(c), d1, d2, q1, coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
