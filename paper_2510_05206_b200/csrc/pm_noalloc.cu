// pm_noalloc.cu -- pm_mesh_power_noalloc: the shell binning of the (cross-)power spectrum (DESIGN.md
// reading R20; the k_power_bins step of pm_power_spectrum) for callers that cannot allocate: code under CUDA graph
// capture, tight serving loops, harnesses that forbid cudaMalloc.  No ctx, no cudaMalloc / cudaFree, no library
// routine that allocates: the caller passes the half-complex spectra and the three output arrays, and the scratch
// of the kernel -- the [3][nbins] fp64 accumulators {n_modes, sum |n|, sum Re(A conj B)} that pm_power_spectrum keeps
// in a cudaMalloc'ed buffer of its ctx -- lives in a file-scope __device__ array of PM_NOALLOC_MAX_BINS bins
// (24 KB, held by every GPU that loads the library until the process exits).
//
// The array is shared by every call on a device and keeps the last call's contents: each call clears the part it
// uses first, in stream order.  Calls that overlap on the GPU (different streams, no dependency) race on it.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "pm_internal.cuh"

namespace pmf {

namespace {

constexpr int NB = 256;                              // threads per CTA
constexpr int MAX_BINS = PM_NOALLOC_MAX_BINS;        // include/pmforce.h
constexpr int MAX_DEVICES = 64;

// scratch: acc[0..nbins) mode counts, acc[nbins..2 nbins) sum |n|, acc[2 nbins..3 nbins) sum Re(A conj B)
static __device__ __align__(256) double g_power_scratch[3 * MAX_BINS];

// In host code `g_power_scratch` is a host-side stand-in, not a device address: the address the kernels get comes from
// cudaGetSymbolAddress, looked up once per device with that device current.
struct DeviceSetup {
  double* scratch = nullptr;
  int num_sms = 0;
};
DeviceSetup g_setup[MAX_DEVICES];
std::mutex g_setup_mutex;

__global__ void __launch_bounds__(NB) k_mesh_power_bins(const float2* __restrict__ a, const float2* __restrict__ b,
                                                        int m, int nbins, double* __restrict__ acc) {
  extern __shared__ double s_bin[];  // [3 * nbins]
  for (int j = threadIdx.x; j < 3 * nbins; j += NB) s_bin[j] = 0.0;
  __syncthreads();
  const int hz = m / 2 + 1;
  const int64_t rows = (int64_t)m * m;
  for (int64_t row = blockIdx.x; row < rows; row += gridDim.x) {
    const int ix = (int)(row / m), iy = (int)(row - (int64_t)ix * m);
    const int nx = ix < (m + 1) / 2 ? ix : ix - m, ny = iy < (m + 1) / 2 ? iy : iy - m;
    const size_t base = (size_t)row * hz;
    for (int iz = threadIdx.x; iz < hz; iz += NB) {
      const double kn = sqrt((double)nx * nx + (double)ny * ny + (double)iz * iz);
      const int bin = (int)floor(kn - 0.5);  // b + 1/2 <= |n| < b + 3/2 (R20)
      if (bin < 0 || bin >= nbins) continue;
      const double mult = (iz == 0 || 2 * iz == m) ? 1.0 : 2.0;  // the stored half stands for both signs of n_z
      const float2 va = a[base + iz];
      const float2 vb = b ? b[base + iz] : va;
      const double pw = (double)va.x * (double)vb.x + (double)va.y * (double)vb.y;
      atomicAdd(&s_bin[bin], mult);
      atomicAdd(&s_bin[nbins + bin], mult * kn);
      atomicAdd(&s_bin[2 * nbins + bin], mult * pw);
    }
  }
  __syncthreads();
  for (int j = threadIdx.x; j < 3 * nbins; j += NB)
    if (s_bin[j] != 0.0) atomicAdd(&acc[j], s_bin[j]);
}

__global__ void k_mesh_power_finish(int nbins, const double* __restrict__ acc, double kf, double norm,
                                    double* __restrict__ k_mean, double* __restrict__ power,
                                    double* __restrict__ n_modes) {
  const int bin = blockIdx.x * blockDim.x + threadIdx.x;
  if (bin >= nbins) return;
  const double cnt = acc[bin];
  const double safe = cnt > 0.0 ? cnt : 1.0;
  n_modes[bin] = cnt;
  k_mean[bin] = kf * acc[nbins + bin] / safe;
  power[bin] = norm * acc[2 * nbins + bin] / safe;
}

int report(char* errbuf, int32_t errbuf_len, int code, const char* fmt, ...) {
  if (errbuf && errbuf_len > 0) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(errbuf, (size_t)errbuf_len, fmt, ap);
    va_end(ap);
  }
  return code;
}

}  // namespace

}  // namespace pmf

using namespace pmf;

extern "C" int pm_mesh_power_noalloc(const float* spec_a, const float* spec_b, int32_t m, double box, double norm,
                                     int32_t nbins, double* k_mean, double* power, double* n_modes, char* errbuf,
                                     int32_t errbuf_len, void* stream) {
  if (errbuf && errbuf_len > 0) errbuf[0] = '\0';
  if (!spec_a || !k_mean || !power || !n_modes) return report(errbuf, errbuf_len, PM_EINVAL, "NULL pointer");
  if (m < 2 || m > 4096) return report(errbuf, errbuf_len, PM_EINVAL, "m = %d outside [2, 4096]", (int)m);
  if (!(box > 0.0)) return report(errbuf, errbuf_len, PM_EINVAL, "box must be positive");
  if (nbins < 1)
    return report(errbuf, errbuf_len, PM_EINVAL, "nbins = %d: at least one bin", (int)nbins);
  if (nbins > MAX_BINS)
    return report(errbuf, errbuf_len, PM_EINVAL,
                  "nbins = %d exceeds PM_NOALLOC_MAX_BINS = %d (the static scratch array holds no more; "
                  "pm_power_spectrum has no such limit)", (int)nbins, MAX_BINS);
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return report(errbuf, errbuf_len, PM_ECUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
  if (dev < 0 || dev >= MAX_DEVICES)
    return report(errbuf, errbuf_len, PM_EINVAL, "device ordinal %d outside [0, %d)", dev, MAX_DEVICES);
  DeviceSetup su;
  {  // set-up, once per device, with that device current
    std::lock_guard<std::mutex> lock(g_setup_mutex);
    if (!g_setup[dev].scratch) {
      double* ptr = nullptr;
      e = cudaGetSymbolAddress((void**)&ptr, g_power_scratch);
      if (e != cudaSuccess || !ptr)
        return report(errbuf, errbuf_len, PM_ECUDA, "cudaGetSymbolAddress(g_power_scratch): %s", cudaGetErrorString(e));
      int sms = 0;
      e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
      if (e != cudaSuccess || sms < 1)
        return report(errbuf, errbuf_len, PM_ECUDA, "cudaDeviceGetAttribute: %s", cudaGetErrorString(e));
      g_setup[dev].num_sms = sms;
      g_setup[dev].scratch = ptr;
    }
    su = g_setup[dev];
  }
  cudaStream_t st = reinterpret_cast<cudaStream_t>(stream);
  // the array keeps the previous call's sums: clear what this call accumulates into
  e = cudaMemsetAsync(su.scratch, 0, sizeof(double) * 3 * (size_t)nbins, st);
  if (e != cudaSuccess) return report(errbuf, errbuf_len, PM_ECUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
  const size_t smem = sizeof(double) * 3 * (size_t)nbins;  // <= 24 KB: below the default dynamic limit
  int64_t grid = (int64_t)su.num_sms * 4;
  if (grid > (int64_t)m * m) grid = (int64_t)m * m;
  k_mesh_power_bins<<<(unsigned)grid, NB, smem, st>>>(reinterpret_cast<const float2*>(spec_a),
                                                      reinterpret_cast<const float2*>(spec_b), m, nbins, su.scratch);
  e = cudaGetLastError();
  if (e != cudaSuccess) return report(errbuf, errbuf_len, PM_ECUDA, "k_mesh_power_bins: %s", cudaGetErrorString(e));
  k_mesh_power_finish<<<(nbins + 127) / 128, 128, 0, st>>>(nbins, su.scratch, 2.0 * M_PI / box, norm, k_mean, power,
                                                           n_modes);
  e = cudaGetLastError();
  if (e != cudaSuccess) return report(errbuf, errbuf_len, PM_ECUDA, "k_mesh_power_finish: %s", cudaGetErrorString(e));
  return PM_OK;
}
