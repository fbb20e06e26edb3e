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

__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}

// One CTA per (ix, iy) row of the half-complex grid; threads run along iz.
__global__ void __launch_bounds__(KS_BLOCK) k_kspace_fwd(KTabs t, const float2* __restrict__ d1,
                                                         const float2* __restrict__ d2,
                                                         float2* __restrict__ g0, float2* __restrict__ g1,
                                                         float2* __restrict__ g2, double coeff_eff) {
  const int row = blockIdx.x;
  const int ix = row / t.m, iy = row - ix * t.m;
  const double lxy = t.lap[ix] + t.lap[iy];
  const double wxy = t.win[ix] * t.win[iy];
  const double dxv = t.grad[ix], dyv = t.grad[iy];
  float2 pxy = make_float2(1.f, 0.f);
  if (d2) {
    const double cr = t.pc[ix] * t.pc[iy] - t.ps[ix] * t.ps[iy];
    const double ci = t.pc[ix] * t.ps[iy] + t.ps[ix] * t.pc[iy];
    pxy = make_float2((float)cr, (float)ci);
  }
  const size_t base = (size_t)row * t.hz;
  for (int iz = threadIdx.x; iz < t.hz; iz += KS_BLOCK) {
    const double den = (lxy + t.lap[iz]) * (wxy * t.win[iz]);
    const double green = (den != 0.0) ? coeff_eff / den : 0.0;  // n = 0 and dropped modes -> 0
    float2 d = d1[base + iz];
    if (d2) {
      const float2 pz = make_float2((float)t.pc[iz], (float)t.ps[iz]);
      const float2 e = cmul(cmul(pxy, pz), d2[base + iz]);
      d = make_float2(0.5f * (d.x + e.x), 0.5f * (d.y + e.y));
    }
    // -i D green (re + i im) = D green (im - i re)
    const float mx = (float)(dxv * green), my = (float)(dyv * green), mz = (float)(t.grad[iz] * green);
    g0[base + iz] = make_float2(mx * d.y, -mx * d.x);
    g1[base + iz] = make_float2(my * d.y, -my * d.x);
    g2[base + iz] = make_float2(mz * d.y, -mz * d.x);
  }
}

__global__ void __launch_bounds__(KS_BLOCK) k_kspace_tr(KTabs t, const float2* __restrict__ g0,
                                                        const float2* __restrict__ g1,
                                                        const float2* __restrict__ g2, float2* __restrict__ q1,
                                                        float2* __restrict__ q2, double coeff_eff) {
  const int row = blockIdx.x;
  const int ix = row / t.m, iy = row - ix * t.m;
  const double lxy = t.lap[ix] + t.lap[iy];
  const double wxy = t.win[ix] * t.win[iy];
  const double dxv = t.grad[ix], dyv = t.grad[iy];
  float2 pxy = make_float2(1.f, 0.f);
  if (q2) {  // conj of the interlace phase
    const double cr = t.pc[ix] * t.pc[iy] - t.ps[ix] * t.ps[iy];
    const double ci = t.pc[ix] * t.ps[iy] + t.ps[ix] * t.pc[iy];
    pxy = make_float2((float)cr, (float)-ci);
  }
  const size_t base = (size_t)row * t.hz;
  for (int iz = threadIdx.x; iz < t.hz; iz += KS_BLOCK) {
    const double den = (lxy + t.lap[iz]) * (wxy * t.win[iz]);
    const double green = (den != 0.0) ? coeff_eff / den : 0.0;
    const float mx = (float)(dxv * green), my = (float)(dyv * green), mz = (float)(t.grad[iz] * green);
    const float2 a = g0[base + iz], b = g1[base + iz], c = g2[base + iz];
    // conj(S_a) = +i D_a green:  q = i * sum_a m_a (re_a + i im_a)
    float2 q = make_float2(-(mx * a.y + my * b.y + mz * c.y), mx * a.x + my * b.x + mz * c.x);
    if (q2) {
      q.x *= 0.5f;
      q.y *= 0.5f;
      const float2 pz = make_float2((float)t.pc[iz], (float)-t.ps[iz]);
      q2[base + iz] = cmul(cmul(pxy, pz), q);
    }
    q1[base + iz] = q;
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
  k_kspace_fwd<<<c->mg * c->mg, KS_BLOCK, 0, st>>>(tabs_of(c), d1, d2, ghat[0], ghat[1], ghat[2], coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

int launch_kspace_transpose(Ctx* c, const float2* const gh[3], float2* q1, float2* q2, double coeff_eff,
                            cudaStream_t st) {
  k_kspace_tr<<<c->mg * c->mg, KS_BLOCK, 0, st>>>(tabs_of(c), gh[0], gh[1], gh[2], q1, q2, coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
