// pm_microbench.cu -- measured ceilings of the shared-memory pipe, for the NUFFT stages ("measure a
// shared-atomic microbenchmark on the box and use it as that stage's ceiling").  Spreading with the ES kernel does
// w^3 shared-memory integer atomics per particle, interpolation 3 w^3 shared-memory loads; neither is HBM-bound.
// Every lane of a warp touches its own bank (conflict-free), 16 independent operations in flight per thread,
// 2048 resident threads per SM: the number is what the LSU pipe delivers at its best.
#include "pm_internal.cuh"

namespace pmf {

namespace {

constexpr int MB_BLOCK = 256;
constexpr int MB_WORDS = 32 * 32;  // per warp: 32 rows of 32 banks

template <int KIND>  // 0: ld.shared.f32, 1: atom.shared.add.u32, 2: ld.shared.v4.f32 (counted as 4 lane-words)
__global__ void __launch_bounds__(MB_BLOCK) k_smem_peak(int iters, float* __restrict__ sink) {
  __shared__ __align__(16) unsigned s[(MB_BLOCK / 32) * MB_WORDS];
  const unsigned lane = threadIdx.x & 31u;
  unsigned* w = s + (threadIdx.x >> 5) * MB_WORDS;
  for (int j = lane; j < MB_WORDS; j += 32) w[j] = j;
  __syncwarp();
  float acc = 0.f;
  unsigned row = lane;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      const unsigned r = (row + u) & 31u;  // the row changes, the bank (= lane) does not: conflict-free
      if (KIND == 0) {
        acc += __uint_as_float(*(volatile unsigned*)(w + r * 32 + lane));
      } else if (KIND == 1) {
        atomicAdd(w + r * 32 + lane, row + 3u);  // a data-dependent addend: ATOMS.ADD, as in the spreading kernel
      } else {
        uint4 v;  // a quarter-warp covers all 32 banks
        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                     : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                     : "r"((unsigned)__cvta_generic_to_shared(w + r * 32 + 4 * (lane & 7u))));
        acc += __uint_as_float(v.x ^ v.y ^ v.z ^ v.w);
      }
    }
    row += 5;
  }
  if (acc == 1.2345f) sink[0] = acc + (float)w[lane];  // never true
}

template <int KIND>
int run_peak(Ctx* c, double* out, cudaStream_t st) {
  const int iters = 4096;
  const int grid = c->num_sms * 8;
  float* sink = nullptr;
  PM_CUDA(c, cudaMalloc((void**)&sink, sizeof(float)));
  cudaEvent_t e0, e1;
  PM_CUDA(c, cudaEventCreate(&e0));
  PM_CUDA(c, cudaEventCreate(&e1));
  k_smem_peak<KIND><<<grid, MB_BLOCK, 0, st>>>(iters, sink);  // warm-up
  float best = 1e30f;
  for (int rep = 0; rep < 3; ++rep) {
    cudaEventRecord(e0, st);
    k_smem_peak<KIND><<<grid, MB_BLOCK, 0, st>>>(iters, sink);
    cudaEventRecord(e1, st);
    cudaEventSynchronize(e1);
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    if (ms < best) best = ms;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(sink);
  PM_CUDA(c, cudaGetLastError());
  const double ops = (double)grid * MB_BLOCK * (double)iters * 16.0 * (KIND == 2 ? 4.0 : 1.0);
  *out = ops / ((double)best * 1e-3);
  return PM_OK;
}

}  // namespace

}  // namespace pmf

extern "C" int pm_smem_peak(pm_ctx* ctx, int kind, double* lane_ops_per_s_host, void* stream) {
  using namespace pmf;
  Ctx* c = C(ctx);
  if (!c || !lane_ops_per_s_host) return PM_EINVAL;
  PM_TRY(enter_device(c));
  switch (kind) {
    case 0: return run_peak<0>(c, lane_ops_per_s_host, (cudaStream_t)stream);
    case 1: return run_peak<1>(c, lane_ops_per_s_host, (cudaStream_t)stream);
    case 2: return run_peak<2>(c, lane_ops_per_s_host, (cudaStream_t)stream);
  }
  return fail(c, PM_EINVAL, "kind must be 0 (loads), 1 (integer atomics) or 2 (128-bit loads)");
}
