// pm_ctx.cu -- context lifetime, parameter validation, fp64 symbol tables, cuFFT plans, profiling.
#include <math.h>
#include <stdarg.h>
#include <stdlib.h>

#include <new>
#include <vector>

#include "pm_internal.cuh"

namespace pmf {

int fail(Ctx* c, int code, const char* fmt, ...) {
  if (c) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(c->err, sizeof(c->err), fmt, ap);
    va_end(ap);
  }
  return code;
}

ShiftSplit split_shift(const Ctx* c, const double* shift) {
  ShiftSplit s;
  s.shifted = false;
  for (int a = 0; a < 3; ++a) {
    double cells = shift ? shift[a] * ((double)c->mg / c->p.box) : 0.0;
    double k = floor(cells);
    double f = cells - k;
    uint32_t fx = (uint32_t)llrint(f * (double)REC_ONE);
    if (fx >= REC_ONE) {  // rounded up to a whole cell
      fx = 0;
      k += 1.0;
    }
    long long kk = (long long)k % c->mg;
    s.roll[a] = (int)kk;
    s.frac[a] = fx;
    if (fx) s.shifted = true;
  }
  return s;
}

// ---- TMA tensor maps -----------------------------------------------------------------------------------
// cuTensorMapEncodeTiled is a driver-API call; it is fetched through the runtime so that the library does
// not link against libcuda directly.
typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static EncodeTiledFn g_encode_tiled = nullptr;

int make_mesh_tmap(Ctx* c, const float* base, int sx, int sy, int sz, CUtensorMap* out) {
  for (int i = 0; i < c->ntmaps; ++i) {
    const Ctx::TMapEntry& e = c->tmaps[i];
    if (e.base == base && e.sx == sx && e.sy == sy && e.sz == sz) {
      *out = e.map;
      return PM_OK;
    }
  }
  if (!g_encode_tiled) {
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    PM_CUDA(c, cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres));
    if (!fn || qres != cudaDriverEntryPointSuccess) return fail(c, PM_ECUDA, "cuTensorMapEncodeTiled not available");
    g_encode_tiled = (EncodeTiledFn)fn;
  }
  if (!base || (reinterpret_cast<uintptr_t>(base) & 15u))
    return fail(c, PM_EINVAL, "mesh pointers must be non-NULL and 16-byte aligned");
  const cuuint64_t m = (cuuint64_t)c->mg;
  const cuuint64_t dims[3] = {m, m, m};                                       // innermost (z) first
  const cuuint64_t strides[2] = {m * sizeof(float), m * m * sizeof(float)};   // bytes, dims 1 and 2
  const cuuint32_t box[3] = {(cuuint32_t)sz, (cuuint32_t)sy, (cuuint32_t)sx};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = g_encode_tiled(out, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, const_cast<float*>(base), dims, strides,
                                    box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(c, PM_ECUDA, "cuTensorMapEncodeTiled failed: CUresult %d (box %d x %d x %d)", (int)r, sx, sy, sz);
  constexpr int NT = (int)(sizeof(c->tmaps) / sizeof(c->tmaps[0]));
  const int slot = c->ntmaps < NT ? c->ntmaps++ : (c->tmap_next++ % NT);  // full: overwrite round-robin
  c->tmaps[slot].base = base;
  c->tmaps[slot].sx = sx;
  c->tmaps[slot].sy = sy;
  c->tmaps[slot].sz = sz;
  c->tmaps[slot].map = *out;
  return PM_OK;
}

int kernel_occupancy(Ctx* c, const void* fn, int block, size_t smem, int* occ) {
  for (int i = 0; i < c->nkern; ++i)
    if (c->kern[i].fn == fn) {
      *occ = c->kern[i].occ;
      return PM_OK;
    }
  int o = 0;
  PM_CUDA(c, cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
  PM_CUDA(c, cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, fn, block, smem));
  if (o < 1) return fail(c, PM_ECUDA, "kernel does not fit on an SM (%zu bytes of shared memory)", smem);
  constexpr int NK = (int)(sizeof(c->kern) / sizeof(c->kern[0]));
  if (c->nkern < NK) {
    c->kern[c->nkern].fn = fn;
    c->kern[c->nkern].occ = o;
    ++c->nkern;
  }
  *occ = o;
  return PM_OK;
}

int enter_device(Ctx* c) {
  int dev = -1;
  PM_CUDA(c, cudaGetDevice(&dev));
  if (dev != c->device) PM_CUDA(c, cudaSetDevice(c->device));
  return PM_OK;
}

// ---- symbol tables (Table 1 Fourier column, Table 2; readings R4-R6, R9) ---------------------------
static double sinc_pi(double x) {  // sin(pi x)/(pi x)
  if (x == 0.0) return 1.0;
  double a = M_PI * x;
  return sin(a) / a;
}

static void pm_tables(const pm_params& p, int m, std::vector<double>& grad, std::vector<double>& lap,
                      std::vector<double>& win, std::vector<double>& pc, std::vector<double>& ps) {
  const double delta = p.box / m;
  for (int i = 0; i < m; ++i) {
    const int n = (i < (m + 1) / 2) ? i : i - m;  // FFT order; n = -m/2 at i = m/2 (even m)
    const double th = 2.0 * M_PI * (double)n / (double)m;
    const bool nyq = (m % 2 == 0) && (i == m / 2);
    double D, l;
    switch (p.grad_order) {  // Table 2 gradient rows, theta = pi k
      case 0: D = nyq ? 0.0 : th; break;  // R5
      case 2: D = sin(th); break;
      case 4: D = (8.0 * sin(th) - sin(2.0 * th)) / 6.0; break;
      default: D = (45.0 * sin(th) - 9.0 * sin(2.0 * th) + sin(3.0 * th)) / 30.0; break;
    }
    switch (p.lap_order) {  // Table 2 Laplacian rows; order 2 sign per R4
      case 0: l = -th * th; break;
      case 2: l = 2.0 * cos(th) - 2.0; break;
      case 4: l = -(cos(2.0 * th) - 16.0 * cos(th) + 15.0) / 6.0; break;
      default: l = -(-2.0 * cos(3.0 * th) + 27.0 * cos(2.0 * th) - 270.0 * cos(th) + 245.0) / 90.0; break;
    }
    grad[i] = D / delta;
    lap[i] = l / (delta * delta);
    win[i] = pow(sinc_pi((double)n / (double)m), (double)(p.worder * p.deconv_pow));
    // e^{-i k.s}, s = Delta/2 per axis: exp(-i pi n / m); real part only on the Nyquist index (R9)
    pc[i] = nyq ? 0.0 : cos(M_PI * (double)n / (double)m);
    ps[i] = nyq ? 0.0 : -sin(M_PI * (double)n / (double)m);
  }
}

// Gauss-Legendre nodes / weights on [-1, 1] by Newton iteration on P_n.
static void gauss_legendre(int n, std::vector<double>& x, std::vector<double>& w) {
  x.resize(n);
  w.resize(n);
  for (int i = 0; i < (n + 1) / 2; ++i) {
    double z = cos(M_PI * (i + 0.75) / (n + 0.5));
    double pp = 1.0;
    for (int it = 0; it < 100; ++it) {
      double p1 = 1.0, p2 = 0.0;
      for (int j = 1; j <= n; ++j) {
        double p3 = p2;
        p2 = p1;
        p1 = ((2.0 * j - 1.0) * z * p2 - (j - 1.0) * p3) / j;
      }
      pp = n * (z * p1 - p2) / (z * z - 1.0);
      double dz = p1 / pp;
      z -= dz;
      if (fabs(dz) < 1e-15) break;
    }
    x[i] = -z;
    x[n - 1 - i] = z;
    w[i] = w[n - 1 - i] = 2.0 / ((1.0 - z * z) * pp * pp);
  }
}

// NUFFT tables on the fine grid (readings R8, R10): k, k^2, phi_hat(n)^2 (0 = dropped).
static void nufft_tables(const pm_params& p, int mf, int w, double beta, std::vector<double>& kk,
                         std::vector<double>& k2, std::vector<double>& ph2) {
  std::vector<double> xg, wg;
  gauss_legendre(256, xg, wg);
  for (int i = 0; i < mf; ++i) {
    const int n = (i < (mf + 1) / 2) ? i : i - mf;
    const double k = 2.0 * M_PI * (double)n / p.box;
    kk[i] = k;
    k2[i] = -k * k;  // Lap = -|k|^2, so that S_a = -i k_a C / Lap = i k_a C / |k|^2
    if (2 * abs(n) < p.m) {  // |n| < m/2: below the particle Nyquist (R8)
      // phi_hat(n) = int_{-w/2}^{w/2} phi(2x/w) cos(2 pi n x / m_f) dx
      double acc = 0.0;
      for (size_t q = 0; q < xg.size(); ++q) {
        const double z = xg[q];
        const double phi = exp(beta * (sqrt(fmax(0.0, 1.0 - z * z)) - 1.0));
        acc += wg[q] * (0.5 * w) * phi * cos(2.0 * M_PI * (double)n * (0.5 * w * z) / (double)mf);
      }
      ph2[i] = acc * acc;
    } else {
      ph2[i] = 0.0;
    }
  }
}

static int validate(const pm_params& p, char* why, size_t n) {
#define BAD(msg)                \
  do {                          \
    snprintf(why, n, "%s", msg); \
    return PM_EINVAL;           \
  } while (0)
  if (p.m < 8 || p.m % 4 != 0) BAD("m must be a multiple of 4 and >= 8");
  if (p.m > 4096) BAD("m > 4096 not supported");
  if (!(p.box > 0.0) || !isfinite(p.box)) BAD("box must be finite and > 0");
  if (!isfinite(p.coeff)) BAD("coeff must be finite");
  if (p.max_particles < 1 || p.max_particles > 0x7fffffffLL) BAD("max_particles must be in [1, 2^31)");
  if (p.method != 0 && p.method != 1) BAD("method must be 0 (PM) or 1 (NUFFT)");
  if (p.method == 0) {
    if (p.worder < 2 || p.worder > 4) BAD("worder must be 2, 3 or 4");
    if (p.interlace < 0 || p.interlace > 2) BAD("interlace must be 0, 1 or 2");
    if (p.deconv_pow < 0 || p.deconv_pow > 2) BAD("deconv_pow must be 0, 1 or 2");
    if (p.grad_order != 0 && p.grad_order != 2 && p.grad_order != 4 && p.grad_order != 6)
      BAD("grad_order must be 0, 2, 4 or 6");
    if (p.lap_order != 0 && p.lap_order != 2 && p.lap_order != 4 && p.lap_order != 6)
      BAD("lap_order must be 0, 2, 4 or 6");
  } else {
    if (!(p.nufft_sigma >= 1.0) || p.nufft_sigma > 4.0) BAD("nufft_sigma must be in [1, 4]");
    if (p.nufft_width != 0 && (p.nufft_width < 2 || p.nufft_width > MAX_W))
      BAD("nufft_width must be 0 or in [2, 16]");
    if (p.nufft_width == 0 && !(p.nufft_eps > 0.0 && p.nufft_eps < 1.0))
      BAD("nufft_eps must be in (0, 1) when nufft_width = 0");
    if (p.interlace != 0) BAD("interlace is not defined for the NUFFT path");
  }
  if (p.reserved != 0) BAD("reserved must be 0");
  if (p.flags & ~(PM_FLAG_BIN_TWOPASS | PM_FLAG_NO_XFUSE | PM_FLAG_GRAD_REAL | PM_FLAG_KERNEL_GRAD))
    BAD("unknown bit in flags");
  if ((p.flags & PM_FLAG_GRAD_REAL) && (p.method != 0 || p.grad_order == 0))
    BAD("PM_FLAG_GRAD_REAL needs method = 0 and grad_order 2, 4 or 6 (a finite-difference stencil of Table 2)");
  if ((p.flags & PM_FLAG_KERNEL_GRAD) && p.method != 1) BAD("PM_FLAG_KERNEL_GRAD needs method = 1");
#undef BAD
  return PM_OK;
}

static int upload(Ctx* c, double** dst, const std::vector<double>& src) {
  PM_CUDA(c, cudaMalloc((void**)dst, src.size() * sizeof(double)));
  PM_CUDA(c, cudaMemcpy(*dst, src.data(), src.size() * sizeof(double), cudaMemcpyHostToDevice));
  return PM_OK;
}

static int build(Ctx* c) {
  const pm_params& p = c->p;
  PM_CUDA(c, cudaGetDevice(&c->device));
  cudaDeviceProp prop;
  PM_CUDA(c, cudaGetDeviceProperties(&prop, c->device));
  c->num_sms = prop.multiProcessorCount;
  if (prop.major < 10)
    return fail(c, PM_ECUDA, "libpmforce is built for sm_100a; device is sm_%d%d", prop.major, prop.minor);

  if (p.method == 0) {
    c->mg = p.m;
    c->m_modes = p.m;
  } else {
    int mf = (int)llrint(p.nufft_sigma * p.m);
    if (mf % 4 != 0 || mf < p.m) return fail(c, PM_EINVAL, "round(nufft_sigma*m) = %d must be a multiple of 4", mf);
    c->mg = mf;
    c->m_modes = p.m;
    // R10: w = ceil(log10(1/eps)) + 1; beta = 2.30 w at sigma = 2, else 0.97 pi w (1 - 1/(2 sigma))
    int w = p.nufft_width ? p.nufft_width : (int)ceil(log10(1.0 / p.nufft_eps) - 1e-12) + 1;
    if (w < 2) w = 2;
    if (w < 4 || w > 8) return fail(c, PM_EINVAL, "ES kernel width %d is not built (built: 4..8)", w);
    c->nufft_w = w;
    c->nufft_beta = (fabs(p.nufft_sigma - 2.0) < 1e-12) ? 2.30 * w
                                                         : 0.97 * M_PI * w * (1.0 - 1.0 / (2.0 * p.nufft_sigma));
  }
  const int mg = c->mg;
  c->G = (int64_t)mg * mg * mg;
  c->Gh = (int64_t)mg * mg * (mg / 2 + 1);
  c->ntx = (mg + TX - 1) / TX;
  c->nty = (mg + TY - 1) / TY;
  c->ntz = (mg + TZ - 1) / TZ;
  c->ntiles = c->ntx * c->nty * c->ntz;
  c->bin_occ0 = bin_occupancy(0);
  c->bin_occ = bin_occupancy(1);
  c->xbl = (c->ntx % 8 == 0) ? 3 : (c->ntx % 4 == 0) ? 2 : (c->ntx % 2 == 0) ? 1 : 0;

  // tables
  std::vector<double> a(mg), b(mg), w(mg), pc(mg, 1.0), ps(mg, 0.0);
  if (p.method == 0)
    pm_tables(p, mg, a, b, w, pc, ps);
  else
    nufft_tables(p, mg, c->nufft_w, c->nufft_beta, a, b, w);
  PM_TRY(upload(c, &c->tab_grad, a));
  PM_TRY(upload(c, &c->tab_lap, b));
  PM_TRY(upload(c, &c->tab_win, w));
  PM_TRY(upload(c, &c->tab_cos, pc));
  PM_TRY(upload(c, &c->tab_sin, ps));
  {  // W~(n) to the first power (pm_power_spectrum)
    std::vector<double> w1(mg, 1.0);
    if (p.method == 0)
      for (int i = 0; i < mg; ++i) {
        const int n = (i < (mg + 1) / 2) ? i : i - mg;
        w1[i] = pow(sinc_pi((double)n / (double)mg), (double)p.worder);
      }
    PM_TRY(upload(c, &c->tab_win1, w1));
  }

  // binning workspace
  c->cap = p.max_particles;
  c->max_items = 2 * (int64_t)c->ntiles + c->cap / ITEM_MAX + 2;
  {  // single-pass binning: a bucket of twice the mean tile load per tile, overflow sorted behind the buckets
    const int64_t mean = (c->cap + c->ntiles - 1) / c->ntiles;
    int64_t capt = (2 * mean + 31) / 32 * 32;
    if (capt < 64) capt = 64;
    const int64_t total = (int64_t)c->ntiles * capt + c->cap;
    c->bin_capt = ((p.flags & PM_FLAG_BIN_TWOPASS) || total >= (int64_t)0xffffffff) ? 0u : (uint32_t)capt;
    c->ov_base = (uint32_t)((int64_t)c->ntiles * c->bin_capt);
  }
  const int scan_blocks = (c->ntiles + 4095) / 4096;
  PM_CUDA(c, cudaMalloc((void**)&c->rec, sizeof(uint4) * ((size_t)c->ov_base + (size_t)c->cap)));
  if (c->bin_capt) {
    PM_CUDA(c, cudaMalloc((void**)&c->ov_count, sizeof(uint32_t)));
    // + reserved-but-unused list space (holes): < 32 of every 1024-entry chunk, and one open chunk per resident
    // binning warp at the end of the pass
    const size_t ov_len = (size_t)c->cap + (size_t)c->cap / 16 + ((size_t)c->num_sms * c->bin_occ * 8 + 1) * 1024;
    PM_CUDA(c, cudaMalloc((void**)&c->ov_rec, sizeof(uint4) * ov_len));
    PM_CUDA(c, cudaMalloc((void**)&c->ov_tile, sizeof(uint32_t) * ov_len));
    PM_CUDA(c, cudaMalloc((void**)&c->ov_cur, sizeof(uint32_t) * (size_t)c->ntiles));
  }
  PM_CUDA(c, cudaMalloc((void**)&c->tile_cnt, sizeof(uint32_t) * (size_t)c->ntiles));
  PM_CUDA(c, cudaMalloc((void**)&c->tile_off, sizeof(uint32_t) * (size_t)(c->ntiles + 1)));
  PM_CUDA(c, cudaMalloc((void**)&c->item_off, sizeof(uint32_t) * (size_t)(c->ntiles + 1)));
  PM_CUDA(c, cudaMalloc((void**)&c->scan_tmp, sizeof(uint32_t) * (size_t)(2 * scan_blocks + 2)));
  PM_CUDA(c, cudaMalloc((void**)&c->items, sizeof(WorkItem) * (size_t)c->max_items));
  PM_CUDA(c, cudaMalloc((void**)&c->nitems, sizeof(uint32_t)));
  PM_CUDA(c, cudaMemset(c->nitems, 0, sizeof(uint32_t)));
  PM_CUDA(c, cudaMalloc((void**)&c->sched, 2 * sizeof(uint32_t)));
  PM_CUDA(c, cudaMemset(c->sched, 0, 2 * sizeof(uint32_t)));

  // cuFFT plans (library call, reported as its own line; north_star "may call cuFFT")
  size_t ws1 = 0, ws2 = 0;
  PM_CUFFT(c, cufftCreate(&c->plan_r2c));
  PM_CUFFT(c, cufftCreate(&c->plan_c2r));
  c->plans_ok = true;
  PM_CUFFT(c, cufftSetAutoAllocation(c->plan_r2c, 0));
  PM_CUFFT(c, cufftSetAutoAllocation(c->plan_c2r, 0));
  PM_CUFFT(c, cufftMakePlan3d(c->plan_r2c, mg, mg, mg, CUFFT_R2C, &ws1));
  PM_CUFFT(c, cufftMakePlan3d(c->plan_c2r, mg, mg, mg, CUFFT_C2R, &ws2));
  c->fft_work_bytes = ws1 > ws2 ? ws1 : ws2;
  PM_TRY(xfft_init(c));  // 2-D plans + twiddles of the fused x-FFT path, when m allows it
  if (c->xfused && c->fft2_work_bytes > c->fft_work_bytes) c->fft_work_bytes = c->fft2_work_bytes;
  if (c->fft_work_bytes) {  // one work area: the plans never run concurrently (one stream per ctx)
    PM_CUDA(c, cudaMalloc(&c->fft_work, c->fft_work_bytes));
    PM_CUFFT(c, cufftSetWorkArea(c->plan_r2c, c->fft_work));
    PM_CUFFT(c, cufftSetWorkArea(c->plan_c2r, c->fft_work));
    if (c->xfused) {
      PM_CUFFT(c, cufftSetWorkArea(c->plan2_r2c, c->fft_work));
      PM_CUFFT(c, cufftSetWorkArea(c->plan2_c2r, c->fft_work));
    }
  }

  // meshes of the fused path
  const int ngrids = (p.method == 0 && p.interlace == 1) ? 2 : 1;
  for (int i = 0; i < ngrids; ++i) {
    PM_CUDA(c, cudaMalloc((void**)&c->rho[i], sizeof(float) * (size_t)c->G));
    PM_CUDA(c, cudaMalloc((void**)&c->dhat[i], sizeof(float2) * (size_t)c->Gh));
  }
  for (int a3 = 0; a3 < 3; ++a3) {
    PM_CUDA(c, cudaMalloc((void**)&c->ghat[a3], sizeof(float2) * (size_t)c->Gh));
    PM_CUDA(c, cudaMalloc((void**)&c->g[a3], sizeof(float) * (size_t)c->G));
  }
  for (int i = 0; i < 2 * 2 * PM_NUM_STAGES; ++i) PM_CUDA(c, cudaEventCreate(&c->ev[0][0] + i));
  c->ev_ok = true;
  PM_CUDA(c, cudaDeviceSynchronize());
  return PM_OK;
}

static void teardown(Ctx* c) {
  if (!c) return;
  cudaDeviceSynchronize();
  if (c->plans_ok) {
    cufftDestroy(c->plan_r2c);
    cufftDestroy(c->plan_c2r);
  }
  if (c->plans2_ok) {
    cufftDestroy(c->plan2_r2c);
    cufftDestroy(c->plan2_c2r);
  }
  void* ptrs[] = {c->tab_grad, c->tab_lap, c->tab_win, c->tab_cos, c->tab_sin, c->tab_win1, c->phi, c->step_dots,
                  c->ps_acc, c->rec, c->tile_cnt,
                  c->tile_off, c->item_off, c->scan_tmp, c->items, c->nitems, c->sched, c->fft_work, c->rho[0],
                  c->rho[1], c->dhat[0], c->dhat[1], c->ghat[0], c->ghat[1], c->ghat[2], c->g[0],
                  c->g[1], c->g[2], c->gbar[0], c->gbar[1], c->gbar[2], c->xtw, c->xsym, c->xph, c->ov_count, c->ov_rec, c->ov_tile, c->ov_cur,
                  c->host_pos_dev,
                  c->host_force_dev};
  for (void* q : ptrs)
    if (q) cudaFree(q);
  if (c->ev_ok)
    for (int i = 0; i < 2 * 2 * PM_NUM_STAGES; ++i) cudaEventDestroy((&c->ev[0][0])[i]);
  free(c);
}

int ensure_phi(Ctx* c) {
  if (c->phi) return PM_OK;
  PM_CUDA(c, cudaMalloc((void**)&c->phi, sizeof(float) * (size_t)c->G));
  return PM_OK;
}

void stage_begin(Ctx* c, int stage, cudaStream_t st) {
  if (!c->profiling) return;
  cudaEventRecord(c->ev[c->ev_slot][2 * stage], st);
  c->ev_used[c->ev_slot][stage] = true;
  c->prof_stream = st;
}
void stage_end(Ctx* c, int stage, cudaStream_t st) {
  if (!c->profiling) return;
  cudaEventRecord(c->ev[c->ev_slot][2 * stage + 1], st);
}

int fft_r2c(Ctx* c, const float* in, float2* out, cudaStream_t st) {
  PM_CUFFT(c, cufftSetStream(c->plan_r2c, st));
  PM_CUFFT(c, cufftExecR2C(c->plan_r2c, const_cast<float*>(in), reinterpret_cast<cufftComplex*>(out)));
  return PM_OK;
}
int fft_c2r(Ctx* c, float2* in, float* out, cudaStream_t st) {
  PM_CUFFT(c, cufftSetStream(c->plan_c2r, st));
  PM_CUFFT(c, cufftExecC2R(c->plan_c2r, reinterpret_cast<cufftComplex*>(in), out));
  return PM_OK;
}

}  // namespace pmf

using namespace pmf;

static thread_local char g_create_err[512] = "";

extern "C" {

int pm_create(pm_ctx** out, const pm_params* p) {
  if (!out || !p) return PM_EINVAL;
  Ctx* c = (Ctx*)calloc(1, sizeof(Ctx));
  if (!c) return PM_ENOMEM;
  c->p = *p;
  int rc = validate(*p, c->err, sizeof(c->err));
  if (rc == PM_OK) rc = build(c);
  if (rc != PM_OK) {
    snprintf(g_create_err, sizeof(g_create_err), "%s", c->err);
    teardown(c);
    cudaGetLastError();
    return rc;
  }
  *out = reinterpret_cast<pm_ctx*>(c);
  return PM_OK;
}

int pm_destroy(pm_ctx* ctx) {
  teardown(C(ctx));
  return PM_OK;
}

const char* pm_strerror(int code) {
  switch (code) {
    case PM_OK: return "ok";
    case PM_EINVAL: return "invalid argument";
    case PM_ENOMEM: return "out of memory";
    case PM_ECUDA: return "CUDA error";
    case PM_ECUFFT: return "cuFFT error";
    case PM_ESTATE: return "call not valid in this state";
    default: return "unknown error";
  }
}

const char* pm_last_error(const pm_ctx* ctx) { return ctx ? C(ctx)->err : g_create_err; }
int32_t pm_mesh_dim(const pm_ctx* ctx) { return ctx ? C(ctx)->p.m : 0; }
int32_t pm_fine_dim(const pm_ctx* ctx) { return (ctx && C(ctx)->p.method == 1) ? C(ctx)->mg : 0; }
int32_t pm_nufft_width(const pm_ctx* ctx) { return ctx ? C(ctx)->nufft_w : 0; }
double pm_nufft_beta(const pm_ctx* ctx) { return ctx ? C(ctx)->nufft_beta : 0.0; }

int pm_set_profiling(pm_ctx* ctx, int enable) {
  if (!ctx) return PM_EINVAL;
  C(ctx)->profiling = enable != 0;
  return PM_OK;
}

int pm_get_stage_ms(pm_ctx* ctx, float* ms_host, int n, int64_t* launches_host) {
  Ctx* c = C(ctx);
  if (!c || !ms_host || n < 0 || n > PM_NUM_STAGES) return PM_EINVAL;
  PM_CUDA(c, cudaStreamSynchronize(c->prof_stream));
  for (int s = 0; s < n; ++s) {
    ms_host[s] = 0.f;
    for (int e = 0; e < 2; ++e)  // the two evaluations of interlace = 2 add up
      if (c->ev_used[e][s]) {
        float t = 0.f;
        PM_CUDA(c, cudaEventElapsedTime(&t, c->ev[e][2 * s], c->ev[e][2 * s + 1]));
        ms_host[s] += t;
      }
  }
  if (launches_host) *launches_host = c->launches;
  return PM_OK;
}

}  // extern "C"
