// pm_step.cu -- the per-particle updates of the drift-kick-drift step (Eq. 2.14a-c, :179-183) and of its
// backward-in-time adjoint step (Table 3, :344-358) that are not fused into the gather:
//
//   drift            X <- X + tau V                                         (2.14a; Table 3 "Primal drift" with -tau)
//   adjoint drift    V* <- a V* + b X*                                      (Table 3: a = 1, b = tau_2 before the kick;
//                                                                             a = alpha ("rescale"), b = tau_1 after it)
//   scalar adjoint   dot += sum_i X*_i . V_i                                (tau_2* = X*^n . V^n,  tau_1* = X*^{n-1} . V^{n-1})
//
// one pass over the arrays per call (HBM-bound: 36N bytes for a drift, 84N with the adjoint part).  The kick,
// the second drift of the forward step and the alpha*, beta* reductions ride on the gather (GatherDev).
// Drifts are evaluated in fp32, operation by operation as DESIGN.md reading R18 specifies, so
// that the force is evaluated at the same fp32 positions on both sides.
#include "pm_internal.cuh"

namespace pmf {

namespace {

constexpr int STB = 256;

// n3 = 3N scalars, VEC of them per thread and iteration (VEC = 4: 16-byte accesses).  xs == NULL: drift only.
template <int VEC>
__global__ void __launch_bounds__(STB) k_step_update(float* __restrict__ x, const float* __restrict__ v,
                                                     const float* __restrict__ xs, float* __restrict__ vs, int64_t n3,
                                                     float tau_x, float a, float b, float box,
                                                     double* __restrict__ dot) {
  __shared__ double s_part[STB / 32];
  double acc = 0.0;
  const int64_t stride = (int64_t)gridDim.x * STB * VEC;
  for (int64_t i = ((int64_t)blockIdx.x * STB + threadIdx.x) * VEC; i < n3; i += stride) {
    float xv[VEC], vv[VEC], xsv[VEC], vsv[VEC];
    if (VEC == 4) {
      *reinterpret_cast<float4*>(xv) = __ldcs(reinterpret_cast<const float4*>(x + i));
      *reinterpret_cast<float4*>(vv) = __ldcs(reinterpret_cast<const float4*>(v + i));
      if (xs) {
        *reinterpret_cast<float4*>(xsv) = __ldcs(reinterpret_cast<const float4*>(xs + i));
        *reinterpret_cast<float4*>(vsv) = __ldcs(reinterpret_cast<const float4*>(vs + i));
      }
    } else {
      xv[0] = x[i], vv[0] = v[i];
      if (xs) xsv[0] = xs[i], vsv[0] = vs[i];
    }
#pragma unroll
    for (int k = 0; k < VEC; ++k) {
      xv[k] = drift_fp32(xv[k], vv[k], tau_x, box);
      if (xs) {
        vsv[k] = fmaf(b, xsv[k], a * vsv[k]);
        acc += (double)xsv[k] * (double)vv[k];
      }
    }
    if (VEC == 4) {
      *reinterpret_cast<float4*>(x + i) = *reinterpret_cast<float4*>(xv);
      if (xs) *reinterpret_cast<float4*>(vs + i) = *reinterpret_cast<float4*>(vsv);
    } else {
      x[i] = xv[0];
      if (xs) vs[i] = vsv[0];
    }
  }
  if (xs && dot) {
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, d);
    if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
      double t = 0.0;
      for (int w = 0; w < STB / 32; ++w) t += s_part[w];
      atomicAdd(dot, t);
    }
  }
}

}  // namespace

int launch_step_update(Ctx* c, float* x, const float* v, const float* xs, float* vs, int64_t n, float tau_x, float a,
                       float b, double* dot, cudaStream_t st) {
  const int64_t n3 = 3 * n;
  if (n3 == 0) return PM_OK;
  const uintptr_t al = reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(v) |
                       reinterpret_cast<uintptr_t>(xs) | reinterpret_cast<uintptr_t>(vs);
  const bool vec = (n3 % 4 == 0) && (al & 15u) == 0;
  const int64_t work = vec ? n3 / 4 : n3;
  int64_t grid = (work + STB - 1) / STB;
  const int64_t cap = (int64_t)c->num_sms * 8;
  if (grid > cap) grid = cap;
  if (vec)
    k_step_update<4><<<(unsigned)grid, STB, 0, st>>>(x, v, xs, vs, n3, tau_x, a, b, (float)c->p.box, dot);
  else
    k_step_update<1><<<(unsigned)grid, STB, 0, st>>>(x, v, xs, vs, n3, tau_x, a, b, (float)c->p.box, dot);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
