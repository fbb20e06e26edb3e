// pm_stencil.cu -- PM_FLAG_GRAD_REAL: the finite-difference gradient of Table 2 applied as its real-space stencil
// ("Real" column: 1/2 [-1 0 1], 1/12 [1 -8 0 8 -1], 1/60 [-1 9 -45 0 45 -9 1]; the "Fourier"
// column is the DFT of these stencils, so IFFT(-i D(theta)/Delta phi_hat) == -stencil(IFFT(phi_hat))).
//
//   k_fd_gradient  : phi -> g_a = -(1/Delta) sum_s c_s (phi[j + s e_a] - phi[j - s e_a]),  a = x, y, z
//
// One inverse FFT instead of three for the force: the Fourier-space kernel writes 4G instead of 12G bytes, two C2R
// transforms disappear, and this pass moves 4G + 12G.
//
// Forward evaluations only (pm_force, pm_dkd_step, pm_poisson_force).  The stencil differences a potential that is
// dominated by low k and much larger than Delta |grad phi|, so g carries WHITE rounding noise eps |phi| / Delta: 1e-6 of
// the force, but the reverse-mode calls gather g with grad W, i.e. difference it once more between neighbouring nodes,
// which amplifies exactly that noise (VJP parity 4e-6 at 64^3, 1.85e-5 at 512^3).  They keep the three-inverse-FFT
// meshes and the Fourier-space transposed operator (pm_api.cu forward_meshes).
#include "pm_internal.cuh"

namespace pmf {

namespace {

constexpr int SB = 256;      // threads per CTA
constexpr int ZV = 32;       // float4 groups along z per CTA row (128 nodes)
constexpr int YB = SB / ZV;  // y rows per CTA

// c_s / denominator of the stencil with R offsets per side, s = 1..R (Table 2, "Real" column)
__host__ __device__ constexpr float fd_coef(int R, int s) {
  return R == 1 ? 0.5f
                : R == 2 ? (s == 1 ? 8.f / 12.f : -1.f / 12.f)
                         : (s == 1 ? 45.f / 60.f : (s == 2 ? -9.f / 60.f : 1.f / 60.f));
}

__device__ __forceinline__ int wrapi(int v, int m) {  // v in [-m, 2m)
  v += v < 0 ? m : 0;
  v -= v >= m ? m : 0;
  return v;
}
__device__ __forceinline__ float4 ld4(const float* p) { return __ldg(reinterpret_cast<const float4*>(p)); }
__device__ __forceinline__ float4 sub4(float4 a, float4 b) {
  return make_float4(a.x - b.x, a.y - b.y, a.z - b.z, a.w - b.w);
}
__device__ __forceinline__ float4 fma4(float s, float4 a, float4 acc) {
  return make_float4(fmaf(s, a.x, acc.x), fmaf(s, a.y, acc.y), fmaf(s, a.z, acc.z), fmaf(s, a.w, acc.w));
}

// sum_s c_s (f[z + s] - f[z - s]) for the 4 nodes of a z group; lo / mid / hi = the groups z-4.., z.., z+4..
template <int R>
__device__ __forceinline__ float4 zdiff(float4 lo, float4 mid, float4 hi) {
  const float v[12] = {lo.x, lo.y, lo.z, lo.w, mid.x, mid.y, mid.z, mid.w, hi.x, hi.y, hi.z, hi.w};
  float o[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    float acc = 0.f;
#pragma unroll
    for (int s = 1; s <= R; ++s) acc = fmaf(fd_coef(R, s), v[4 + k + s] - v[4 + k - s], acc);
    o[k] = acc;
  }
  return make_float4(o[0], o[1], o[2], o[3]);
}

// grid: (m/(4 ZV) rounded up, m / YB rounded up, m);  m is a multiple of 4
template <int R>
__global__ void __launch_bounds__(SB) k_fd_gradient(const float* __restrict__ phi, float* __restrict__ gx,
                                                    float* __restrict__ gy, float* __restrict__ gz, int m,
                                                    float neg_inv_delta) {
  const int z = (blockIdx.x * ZV + (threadIdx.x % ZV)) * 4;
  const int y = blockIdx.y * YB + threadIdx.x / ZV;
  const int x = blockIdx.z;
  if (z >= m || y >= m) return;
  const size_t mm = (size_t)m * m;
  const float* row = phi + (size_t)x * mm + (size_t)y * m;
  const float4 mid = ld4(row + z);
  const float4 lo = ld4(row + wrapi(z - 4, m)), hi = ld4(row + wrapi(z + 4, m));
  float4 ax = make_float4(0.f, 0.f, 0.f, 0.f), ay = ax;
#pragma unroll
  for (int s = 1; s <= R; ++s) {
    const float c = fd_coef(R, s);
    ax = fma4(c, sub4(ld4(phi + (size_t)wrapi(x + s, m) * mm + (size_t)y * m + z),
                      ld4(phi + (size_t)wrapi(x - s, m) * mm + (size_t)y * m + z)), ax);
    ay = fma4(c, sub4(ld4(phi + (size_t)x * mm + (size_t)wrapi(y + s, m) * m + z),
                      ld4(phi + (size_t)x * mm + (size_t)wrapi(y - s, m) * m + z)), ay);
  }
  const float4 az = zdiff<R>(lo, mid, hi);
  const size_t o = (size_t)x * mm + (size_t)y * m + z;
  const float k = neg_inv_delta;
  __stcs(reinterpret_cast<float4*>(gx + o), make_float4(k * ax.x, k * ax.y, k * ax.z, k * ax.w));
  __stcs(reinterpret_cast<float4*>(gy + o), make_float4(k * ay.x, k * ay.y, k * ay.z, k * ay.w));
  __stcs(reinterpret_cast<float4*>(gz + o), make_float4(k * az.x, k * az.y, k * az.z, k * az.w));
}

dim3 stencil_grid(int m) { return dim3((m / 4 + ZV - 1) / ZV, (m + YB - 1) / YB, m); }

}  // namespace

// g_a = -grad_a phi with the stencil of c->p.grad_order (2, 4, 6).  phi, g[a]: dense fp32 [m]^3, 16-byte aligned.
int launch_fd_gradient(Ctx* c, const float* phi, float* const g[3], cudaStream_t st) {
  const int m = c->mg;
  const float k = (float)(-(double)m / c->p.box);
  switch (c->p.grad_order) {
    case 2: k_fd_gradient<1><<<stencil_grid(m), SB, 0, st>>>(phi, g[0], g[1], g[2], m, k); break;
    case 4: k_fd_gradient<2><<<stencil_grid(m), SB, 0, st>>>(phi, g[0], g[1], g[2], m, k); break;
    case 6: k_fd_gradient<3><<<stencil_grid(m), SB, 0, st>>>(phi, g[0], g[1], g[2], m, k); break;
    default: return fail(c, PM_ESTATE, "real-space gradient needs grad_order 2, 4 or 6");
  }
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
