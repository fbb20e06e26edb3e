// pm_internal.cuh -- shared declarations of libpmforce (not part of the public ABI).
//
// Data layout in HBM:
//   * meshes: dense fp32 [m][m][m], z fastest; half-complex spectra [m][m][m/2+1] float2.
//   * sorted particle records: one uint4 per particle {ux, uy, uz, orig_index}; u* are tile-local cell
//     coordinates in unsigned fixed point, value = (u_local + REC_BIAS) * 2^REC_FRAC, computed once by the
//     binning pass with an error-free product (the plain fp32 product x*(m/L) would cost 1e-5 of force
//     accuracy).  Two other layouts were measured and rejected: four separate arrays (round 1: the scatter read
//     0.4 GB less, the permute pass took 1.29 ms instead of 0.69 ms) and word-transposed blocks of 32 records
//     (round 2: ux[32] uy[32] uz[32] index[32] per 512 bytes; the assign read 12 B/particle and went 0.72 ->
//     0.67 ms, but the binning pass, with four 4-byte stores per record, went 0.82 -> 1.21 ms at unchanged DRAM
//     bytes -- its stall is the round trip of the slot-claim atomics, which the extra stores lengthen).
//   * tiles of TX x TY x TZ cells in z-fastest order; tile_off[ntiles+1]; work items (tile, begin, end)
//     of at most ITEM_MAX particles.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <cufft.h>
#include <stdint.h>
#include <stdio.h>
#include <string.h>

#include "../../include/pmforce.h"

namespace pmf {

// ---- tile geometry ------------------------------------------------------------------------------
constexpr int TX = 8, TY = 8, TZ = 32;  // cells per tile: a warp's 32 consecutive (Lagrangian-order) records fill
                                        // one z row, so their shared-memory accesses fall in 32 different banks
constexpr int BLOCK = 256;              // threads per CTA of the scatter / gather kernels
constexpr int PPT = 8;                  // particles per thread and work item
constexpr int CHUNK = BLOCK * PPT;      // particles a CTA holds in registers at a time
constexpr int ITEM_MAX = 2 * CHUNK;     // max particles per work item: a tile is one item unless it is denser than
                                        // this (clustered inputs), then it is split evenly for load balance
constexpr int REC_FRAC = 26;            // fractional bits of a record coordinate
constexpr int REC_BIAS = 2;             // cells added so that shifted / half-added values stay >= 0
constexpr uint32_t REC_ONE = 1u << REC_FRAC;
constexpr uint32_t REC_MASK = REC_ONE - 1u;

struct WorkItem {
  uint32_t tile, begin, end;  // tile: bit 31 set = this item holds ALL particles of its tile (exclusive interior)
  uint32_t txyz;  // tile coordinates packed tx | ty << 10 | tz << 20 (written by k_items: no division in the hot kernels)
};

// Everything a scatter / gather kernel needs to know about the grid and the binned particles.
struct BinView {
  const uint4* rec;
  const WorkItem* items;
  const uint32_t* nitems;
  uint32_t* sched;  // [2]: next-item counter and finished-CTA counter of the dynamic tile schedule (zero between launches)
  int m, ntx, nty, ntz;
  int xbl;  // log2 of xb; tiles are numbered ((tx / xb * nty + ty) * xb + tx % xb) * ntz + tz, see tile_id()
};

// Tile numbering.  Work items are processed in tile order by ~1000 concurrently resident CTAs, so tiles
// that share a halo should be close in that order for the halo to be served from L2.  z-neighbours are
// adjacent, y-neighbours xb * ntz apart, x-neighbours ntz apart inside a block of xb tile columns.
__host__ __device__ __forceinline__ uint32_t tile_id(int tx, int ty, int tz, int nty, int ntz, int xbl) {
  return (uint32_t)((((((tx >> xbl) * nty + ty) << xbl) | (tx & ((1 << xbl) - 1))) * ntz) + tz);
}

enum { MAX_W = 16 };

// Periodic wrap of a drifted coordinate into [0, L) in fp32, operation by operation as DESIGN.md reading R18 specifies
// (one conditional add, then one conditional subtract; a particle moves less than one box length per drift).
__device__ __forceinline__ float wrap_box_fp32(float y, float L) {
  if (y < 0.0f) y = __fadd_rn(y, L);
  if (y >= L) y = __fsub_rn(y, L);
  return y;
}
__device__ __forceinline__ float drift_fp32(float x, float v, float tau, float L) {
  return wrap_box_fp32(__fadd_rn(x, __fmul_rn(tau, v)), L);
}


struct Ctx;

// ---- error helpers ------------------------------------------------------------------------------
int fail(Ctx* c, int code, const char* fmt, ...);
#define PM_CUDA(c, expr)                                                                     \
  do {                                                                                       \
    cudaError_t e__ = (expr);                                                                \
    if (e__ != cudaSuccess)                                                                  \
      return pmf::fail((c), e__ == cudaErrorMemoryAllocation ? PM_ENOMEM : PM_ECUDA,         \
                       "%s failed: %s (%s:%d)", #expr, cudaGetErrorString(e__), __FILE__,    \
                       __LINE__);                                                            \
  } while (0)
#define PM_CUFFT(c, expr)                                                                    \
  do {                                                                                       \
    cufftResult r__ = (expr);                                                                \
    if (r__ != CUFFT_SUCCESS)                                                                \
      return pmf::fail((c), r__ == CUFFT_ALLOC_FAILED ? PM_ENOMEM : PM_ECUFFT,               \
                       "%s failed: cufftResult %d (%s:%d)", #expr, (int)r__, __FILE__,       \
                       __LINE__);                                                            \
  } while (0)
#define PM_TRY(expr)             \
  do {                           \
    int rc__ = (expr);           \
    if (rc__ != PM_OK) return rc__; \
  } while (0)

// ---- the context --------------------------------------------------------------------------------
struct Ctx {
  pm_params p;
  int device;
  int num_sms;
  int mg;        // grid the particles are binned on: m (PM) or m_f (NUFFT)
  int m_modes;   // NUFFT: retained modes per dim (= p.m); PM: = m
  int64_t G;     // mg^3
  int64_t Gh;    // mg^2 (mg/2+1)
  int ntx, nty, ntz, ntiles, xbl;
  int bin_occ0, bin_occ;  // resident CTAs per SM of the two binning passes
  // zero-fill rider of the histogram pass (pm_bin.cu): pm_force asks ensure_bins to clear its assignment mesh
  void* zero_req;
  size_t zero_req_bytes;
  bool zero_done;  // rho[0] was cleared by the binning pass of this call
  bool scatter_mesh_zeroed;  // hint for the next scatter launch: its target mesh is all zero (pm_force's own meshes)
  int nufft_w;
  double nufft_beta;

  // symbol tables, fp64, length mg each (device)
  double* tab_grad;   // D(theta)/Delta         (PM)   | k_a               (NUFFT)
  double* tab_lap;    // l(theta)/Delta^2       (PM)   | k_a^2             (NUFFT)
  double* tab_win;    // W~(n)^deconv_pow       (PM)   | phi_hat(n)^2, 0 = mode dropped (NUFFT)
  double* tab_cos;    // interlace phase, real part (R9)
  double* tab_sin;    // interlace phase, imaginary part
  double* tab_win1;   // W~(n) to the FIRST power (power spectrum: one assignment, no gather); 1 for NUFFT

  // binning workspace
  int64_t cap;
  uint4* rec;
  uint32_t bin_capt;    // slots per tile bucket of the single-pass binning; 0 = two-pass (histogram + permute)
  uint32_t ov_base;     // first overflow record in rec: ntiles * bin_capt
  uint32_t* ov_count;   // [1] overflow list length
  uint4* ov_rec;        // [cap] overflow records, unsorted
  uint32_t* ov_tile;    // [cap] their tiles
  uint32_t* ov_cur;     // [ntiles] cursor of the overflow sort
  uint32_t* tile_cnt;   // [ntiles]   histogram, then reused as cursor
  uint32_t* tile_off;   // [ntiles+1]
  uint32_t* item_off;   // [ntiles+1]
  uint32_t* scan_tmp;   // [2 * nblocks_scan + 2]
  WorkItem* items;      // [max_items]
  uint32_t* nitems;     // device scalar
  uint32_t* sched;      // [2] dynamic-schedule counters, see BinView
  int64_t max_items;
  const float* bin_pos; // pointer the records were built from
  int64_t bin_n;
  bool bin_pinned;      // built by an explicit pm_bin
  bool bin_valid;

  // FFT
  cufftHandle plan_r2c, plan_c2r;
  bool plans_ok;
  void* fft_work;
  size_t fft_work_bytes;
  // fused x-FFT + k-space path (pm_xfft.cu): batched 2-D (y,z) plans, twiddles e^{-2 pi i k/m}
  bool xfused;
  bool plans2_ok;
  cufftHandle plan2_r2c, plan2_c2r;
  size_t fft2_work_bytes;
  float2* xtw;
  float4* xsym;  // fp32 {lap, win, grad, 0} per index
  float2* xph;   // fp32 interlace phase {cos, sin} per index

  // meshes owned by the ctx (pm_force path)
  float* rho[2];     // assignment targets (second: interlace = 1)
  float2* dhat[2];   // their spectra
  float2* ghat[3];   // force spectra
  float* g[3];       // force meshes
  float* gbar[3];    // VJP: scattered cotangents (lazy)
  bool vjp_ready;
  float* phi;        // potential mesh (lazy; PM_FLAG_GRAD_REAL, PM_FLAG_KERNEL_GRAD)
  bool g_valid;      // g[0..2] (or phi) hold the forward meshes of the PINNED records (pm_bin): pm_force_vjp reuses them
  double* step_dots; // [4] scalar adjoints of pm_dkd_step_adjoint when the caller passes none (lazy)
  double* ps_acc;    // [3 * ps_nbins] power-spectrum accumulators (lazy)
  int ps_nbins;

  // host staging for pm_force_host
  float* host_pos_dev;
  float* host_force_dev;

  // profiling
  bool profiling;
  cudaEvent_t ev[2][2 * PM_NUM_STAGES];  // [evaluation: interlace = 2 runs the stages twice][begin, end per stage]
  bool ev_used[2][PM_NUM_STAGES];
  int ev_slot;                           // evaluation the stages being recorded belong to
  bool ev_ok;
  int64_t launches;
  cudaStream_t prof_stream;

  // per-ctx launch state (never process-wide statics: a second ctx may live on another device)
  struct KernState {
    const void* fn;
    int occ;
  } kern[96];        // kernels whose shared-memory attribute is set and whose occupancy is known
  int nkern;
  struct TMapEntry {
    const float* base;
    int sx, sy, sz;
    CUtensorMap map;
  } tmaps[24];       // tensor maps of the meshes the gather has staged (a mesh pointer + box identifies one)
  int ntmaps, tmap_next;

  char err[512];
};

inline Ctx* C(pm_ctx* c) { return reinterpret_cast<Ctx*>(c); }
inline const Ctx* C(const pm_ctx* c) { return reinterpret_cast<const Ctx*>(c); }

struct ShiftSplit {
  int roll[3];       // integer cells
  uint32_t frac[3];  // fractional part in [0,1) as REC_FRAC fixed point
  bool shifted;      // any frac != 0
};
ShiftSplit split_shift(const Ctx* c, const double* shift);

// ---- stage entry points (host side, defined in the .cu files) ------------------------------------
int ensure_bins(Ctx* c, const float* pos, int64_t N, cudaStream_t st, bool pin);
BinView bin_view(const Ctx* c);
int bin_occupancy(int pass);

// Scatter ncomp (1..3) fields.  Weight of particle i, component a: wsrc ? wsrc[i*wstride + a] : 1.
int launch_scatter(Ctx* c, int order, const ShiftSplit& sh, int ncomp, const float* wsrc, int wstride,
                   float* const mesh[], cudaStream_t st);
// Gather.  mode GATHER_VALUES: v[i*ncomp + a] = sum_j mesh[a][j] W.
// GATHER_GRAD: v[i*3 + b] = sum_a coef_a(i) sum_j mesh[a][j] dW/dX^b, with
//   coef_a(i) = a < ncot ? cot[i*cstride + a] : const_coef * (wmul ? wmul[i] : 1).
// GATHER_JVP (Eq. C.13b): v[i*ncomp + a] = pos_tan_i . sum_j mesh[a][j] dW/dX  (+ sum_j mesh[ncomp + a][j] W when
//   has_mesh_tan: the tangent meshes follow the primal ones in `mesh`).
// out = alpha * v + out_scale * out (out_scale = 0: out is not read).
enum { GATHER_VALUES = 0, GATHER_GRAD = 1, GATHER_JVP = 2 };
struct GatherArgs {
  int ncomp = 0;
  const float* const* mesh = nullptr;
  int mode = GATHER_VALUES;
  const float* cot = nullptr;
  int cstride = 0, ncot = 0;
  float const_coef = 0.f;
  const float* wmul = nullptr;
  const float* pos_tan = nullptr;
  bool has_mesh_tan = false;
  float alpha = 1.f, out_scale = 0.f;
  float* out = nullptr;
  // fused tails of the DKD step and of its adjoint (ncomp = 3, GATHER_VALUES; see GatherDev in pm_mesh_kernels.cuh)
  float* drift_pos = nullptr;
  float drift_tau = 0.f;
  const float* dot_with = nullptr;
  double* dot_acc = nullptr;
  double* dot_out = nullptr;
  float dot_scale = 1.f;
};
inline GatherArgs gather_values(int ncomp, const float* const* mesh, float* out, float alpha = 1.f,
                                float out_scale = 0.f) {
  GatherArgs a;
  a.ncomp = ncomp;
  a.mesh = mesh;
  a.out = out;
  a.alpha = alpha;
  a.out_scale = out_scale;
  return a;
}
inline GatherArgs gather_grad(int ncomp, const float* const* mesh, const float* cot, int cstride, int ncot,
                              float const_coef, const float* wmul, float* out, float alpha = 1.f,
                              float out_scale = 0.f) {
  GatherArgs a = gather_values(ncomp, mesh, out, alpha, out_scale);
  a.mode = GATHER_GRAD;
  a.cot = cot;
  a.cstride = cstride;
  a.ncot = ncot;
  a.const_coef = const_coef;
  a.wmul = wmul;
  return a;
}
int launch_gather(Ctx* c, int order, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st);
// Sets cudaFuncAttributeMaxDynamicSharedMemorySize and returns the resident CTAs per SM of a kernel on this
// ctx's device; both are done once per (ctx, kernel).
int kernel_occupancy(Ctx* c, const void* fn, int block, size_t smem, int* occ);
// The calls of include/pmforce.h run on the device the ctx was created on.
int enter_device(Ctx* c);
// Tensor map of a dense fp32 [m][m][m] mesh (m = c->mg) with a box of sx * sy * sz elements, no swizzle,
// out-of-bounds elements zero-filled.  base must be 16-byte aligned (PM_EINVAL otherwise).
// Encoded once per (mesh pointer, box) and kept in the ctx.
int make_mesh_tmap(Ctx* c, const float* base, int sx, int sy, int sz, CUtensorMap* out);

// NUFFT spreading / interpolation with the ES kernel (same conventions).
int launch_es_scatter(Ctx* c, int ncomp, const float* wsrc, int wstride, float* const mesh[],
                      cudaStream_t st);
int launch_es_gather(Ctx* c, const GatherArgs& a, cudaStream_t st);

// k-space kernels.
int launch_kspace_forward(Ctx* c, const float2* d1, const float2* d2, float2* const ghat[3],
                          double coeff_eff, cudaStream_t st);
int launch_kspace_transpose(Ctx* c, const float2* const gh[3], float2* q1, float2* q2,
                            double coeff_eff, cudaStream_t st);
int fft_r2c(Ctx* c, const float* in, float2* out, cudaStream_t st);
int fft_c2r(Ctx* c, float2* in, float* out, cudaStream_t st);
// fused path: 2-D (y,z) transforms by cuFFT, x transforms + k-space kernel in one kernel (pm_xfft.cu)
int xfft_init(Ctx* c);
int fft2_r2c(Ctx* c, const float* in, float2* out, cudaStream_t st);
int fft2_c2r(Ctx* c, float2* in, float* out, cudaStream_t st);
int launch_xfft_forward(Ctx* c, const float2* d1, const float2* d2, float2* const gh[3], double coeff_eff,
                        cudaStream_t st);
int launch_xfft_transpose(Ctx* c, const float2* const gh[3], float2* q1, float2* q2, double coeff_eff,
                          cudaStream_t st);
// The whole spectral operator on real meshes (a2-a4 resp. a10), fused when the ctx supports it:
//   forward:   delta (, delta2) -> g[0..2];     transpose: gbar[0..2] -> delta_cot (, delta_cot2)
// dhat / ghat of the ctx are the scratch spectra.  stages = true records the bench's stage events.
int spectral_forward(Ctx* c, const float* d1, const float* d2, float* const g[3], double coeff_eff, bool stages,
                     cudaStream_t st);
int spectral_transpose(Ctx* c, const float* const gb[3], float* q1, float* q2, double coeff_eff, cudaStream_t st);

// potential-only spectral paths (PM_FLAG_GRAD_REAL, PM_FLAG_KERNEL_GRAD)
int ensure_phi(Ctx* c);
int spectral_potential_hat(Ctx* c, bool two, float2* out, double coeff_eff, cudaStream_t st);
int spectral_potential(Ctx* c, const float* d1, const float* d2, float* phi, double coeff_eff, bool stages,
                       cudaStream_t st);
int launch_xfft_potential(Ctx* c, const float2* d1, const float2* d2, float2* phi, double coeff_eff, cudaStream_t st);
int launch_kspace_scalar(Ctx* c, const float2* d1, const float2* d2, float2* q1, double coeff_eff, cudaStream_t st);
int launch_fd_gradient(Ctx* c, const float* phi, float* const g[3], cudaStream_t st);
// forward-mode scatter (pm_jvp.cu)
int launch_scatter_jvp(Ctx* c, int order, const ShiftSplit& sh, const float* w, const float* w_tan,
                       const float* pos_tan, float* mesh_tan, cudaStream_t st);
// drift / adjoint-drift kernels of the DKD step (pm_step.cu): X <- wrap(X + tau_x V) (fp32, R18);
// if xs: Vs <- a Vs + b Xs and *dot += sum Xs . V (V read before / after as Table 3 orders it: see pm_step.cu)
int launch_step_update(Ctx* c, float* x, const float* v, const float* xs, float* vs, int64_t n, float tau_x,
                       float a, float b, double* dot, cudaStream_t st);
// power spectrum binning (pm_power.cu)
int launch_power_bins(Ctx* c, const float2* d1a, const float2* d1b, const float2* d2a, const float2* d2b,
                      bool deconvolve, int nbins, double* acc, cudaStream_t st);
int launch_power_finish(Ctx* c, int nbins, const double* acc, double kf, double pnorm, double* k_mean,
                        double* power, double* n_modes, cudaStream_t st);
// sheet resampling (pm_resample.cu)
int launch_sheet_resample(Ctx* c, const float* pos, int n_p, int r, float* out, cudaStream_t st);

// profiling helpers
void stage_begin(Ctx* c, int stage, cudaStream_t st);
void stage_end(Ctx* c, int stage, cudaStream_t st);
inline void count_launch(Ctx* c, int n = 1) { c->launches += n; }

}  // namespace pmf
