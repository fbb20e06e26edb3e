/* pmforce.h -- C ABI of the B200-native particle-mesh force path of DISCO-DJ II (arXiv 2510.05206).
 *
 * Citations are "PAPER.md:<line>" plus the section / equation / table the line falls in; R<n> are the
 * readings of the paper listed in DESIGN.md.
 *
 * Conventions (all calls)
 *  - Every array pointer is a DEVICE pointer owned by the caller unless its name ends in `_host`.  The
 *    library allocates only ctx-internal workspace (pm_create, and lazily on the first VJP / NUFFT call)
 *    and frees it in pm_destroy.  Nothing is returned that the caller must free.
 *  - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls enqueue work and
 *    return; there is no hidden synchronisation except in pm_create / pm_destroy / pm_force_host /
 *    pm_get_stage_ms and the first call that has to allocate lazily.
 *  - Return value: 0 (PM_OK) or a negative pm_status.  Nothing aborts, throws or prints.  Asynchronous
 *    CUDA faults surface on the next call that checks cudaGetLastError.
 *  - Positions: fp32 [N,3] row-major (x,y,z per particle), any finite value (wrapped periodically into
 *    [0, box), Eq. 2.1 "periodic").  Non-finite positions are the caller's responsibility.
 *  - Meshes: fp32 [m][m][m] row-major, z fastest, dense (no padding); node j sits at r_j = j * box/m
 *    (reading R3).  `m` is the PM mesh for pm_* calls and the fine grid
 *    m_f = round(nufft_sigma * m) for nufft_* calls.  m and m_f must be multiples of 4 and >= 8.
 *  - `shift`: host pointer to 3 doubles in length units (NULL = 0): the operator is evaluated with
 *    W(r_j - X_i + s), i.e. particles displaced by -s (used for interlaced grids).
 */
#ifndef PMFORCE_H
#define PMFORCE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct pm_ctx pm_ctx; /* opaque: cuFFT plans, workspace, bin buffers, symbol tables */

typedef enum pm_status {
  PM_OK = 0,
  PM_EINVAL = -1, /* bad parameter, NULL pointer, N > max_particles, unsupported option */
  PM_ENOMEM = -2, /* device or host allocation failed */
  PM_ECUDA = -3,  /* a CUDA runtime call or an earlier asynchronous kernel failed */
  PM_ECUFFT = -4, /* a cuFFT call failed */
  PM_ESTATE = -5  /* call not valid for this ctx (e.g. nufft_* on a ctx created with method = 0) */
} pm_status;

/* Plain-old-data, copied at pm_create.  Names follow Table 5. */
typedef struct pm_params {
  int32_t m;           /* mesh cells per dimension ("res_pm"); NUFFT: number of retained modes per dim   */
  int32_t worder;      /* 2 CIC, 3 TSC, 4 PCS ("worder", Table 1)                        */
  int32_t interlace;   /* 0 none; 1 two-grid Fourier-space combination; 2 two-grid force average (R1)     */
  int32_t deconv_pow;  /* 0 none, 1 or 2: divide by W~(k)^deconv_pow ("deconvolve" = 2)      */
  int32_t grad_order;  /* 0 exact i k; 2, 4, 6 finite-difference symbol (Table 2)        */
  int32_t lap_order;   /* 0 exact -k^2; 2, 4, 6 finite-difference symbol (Table 2)                        */
  int32_t method;      /* 0 PM (Sec. 2.5); 1 NUFFT                     */
  int32_t nufft_width; /* ES-kernel width w in fine cells, 4..8 (the widths built); 0 = from nufft_eps (R10)  */
  double box;          /* box size L > 0                                                                   */
  double coeff;        /* C in Lap(phi) = C * delta, g = -grad(phi) (Eq. 2.1-2.2, R11)      */
  double nufft_sigma;  /* upsampling factor sigma (5/4; BASELINE config 3: 2)                */
  double nufft_eps;    /* requested NUFFT tolerance                                         */
  int64_t max_particles; /* capacity of the binning workspace; N of every call must be <= this.  The ctx       */
                         /* allocates about 68 bytes per particle for it (tile buckets of twice the mean load,  */
                         /* overflow segment and list: DESIGN.md section 6); PM_FLAG_BIN_TWOPASS selects the    */
                         /* 16 bytes per particle two-pass sort instead                                         */
  int32_t flags;         /* PM_FLAG_* bits, 0 = defaults                                                        */
  int32_t reserved;      /* must be 0                                                                           */
} pm_params;

/* pm_params.flags.  No environment variable steers the library. */
#define PM_FLAG_BIN_TWOPASS 1 /* a0: histogram + permute counting sort (two reads of the positions, 16 B/particle of
                                 workspace) instead of the single-pass bucketed sort */
#define PM_FLAG_NO_XFUSE 2    /* a2-a4: 3-D cuFFT + pointwise Fourier-space kernel instead of the fused x-FFT kernel */
#define PM_FLAG_GRAD_REAL 4   /* a3-a4, method 0, grad_order 2/4/6: apply the gradient as the real-space stencil of
                                 Table 2 ("Real" column; its DFT IS the Fourier symbol) to the
                                 potential mesh: ONE inverse FFT instead of three.  Same operator, other rounding.
                                 Forward evaluations only (pm_force, pm_dkd_step, pm_poisson_force): the reverse-mode
                                 calls always use the Fourier-space operator. */
#define PM_FLAG_KERNEL_GRAD 8 /* method 1: force from the gradient of the ES kernel ("SPH-like"):
                                 the potential is interpolated with grad(phi_ES) instead of multiplying by i k.
                                 pm_force only (its VJP would need second derivatives of the kernel: PM_ESTATE). */

/* ---- lifetime ------------------------------------------------------------------------------------- */
/* Validates p, builds cuFFT plans, symbol tables and workspace on the current CUDA device.  *out is set
 * only on success.  Synchronises the device. */
int pm_create(pm_ctx** out, const pm_params* p);
int pm_destroy(pm_ctx* ctx); /* NULL is allowed */
const char* pm_strerror(int code);
const char* pm_last_error(const pm_ctx* ctx); /* detail of the last failure on this ctx ("" if none);
                                                  NULL: why the last pm_create on this thread failed */

/* Geometry the caller needs to allocate tensors. */
int32_t pm_mesh_dim(const pm_ctx* ctx);        /* m   */
int32_t pm_fine_dim(const pm_ctx* ctx);        /* m_f (0 unless method = 1) */
int32_t pm_nufft_width(const pm_ctx* ctx);     /* w actually used (0 unless method = 1) */
double pm_nufft_beta(const pm_ctx* ctx);       /* ES-kernel beta actually used */

/* ---- a0: binning (the build's own step; north_star "sorted into cell tiles") ------------------------ */
/* Sorts the N particles into mesh tiles (counting sort) and keeps the sorted records in the ctx.  After
 * pm_bin, every call on this ctx that is given the SAME `pos` pointer and N reuses the records, so the
 * caller must not change the positions at that address until the next pm_bin.  Calls given another
 * pointer / N (or made without a prior pm_bin) bin internally first and drop the pinned records.
 * For a method = 1 ctx the tiles are those of the fine grid. */
int pm_bin(pm_ctx* ctx, const float* pos, int64_t N, void* stream);

/* ---- a1: mass assignment, Eq. C.1, Table 1 kernels ----------------------------------- */
/* mesh[j] += sum_i w_i W(r_j - X_i + s).  ACCUMULATES onto `mesh`: the caller zeroes it.
 * w: [N] or NULL (all ones, "M_i = 1" PAPER.md:256). */
int pm_assign(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift,
              float* mesh, void* stream);
/* VJP of pm_assign (rule table): given mesh_cot [m^3],
 *   pos_cot[i,b] = w_i sum_j mesh_cot[j] dW_j(X_i)/dX_i^b   (Eq. C.6, grad-W gather)  -- [N,3] or NULL
 *   w_cot[i]     =     sum_j mesh_cot[j] W_j(X_i)           (Eq. C.8, scalar gather)  -- [N]   or NULL
 * Both are overwritten.  (The cotangent of the input mesh is mesh_cot itself, Eq. C.4.) */
int pm_assign_vjp(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift,
                  const float* mesh_cot, float* pos_cot, float* w_cot, void* stream);

/* ---- a2-a4: FFT, Fourier-space kernel, inverse FFTs (Tables 1-2) ------------ */
/* force_mesh[a] = IFFT( S_a * FFT(delta) ), S_a(n) = -Grad_a(n) coeff / Lap(n) / W~(n)^deconv_pow,
 * S_a(0) = 0 (R7).  delta_mesh2 (grid shifted by half a cell) must be non-NULL iff interlace = 1; the
 * spectra are then combined as 1/2 [d1 + e^{-ik.s} d2] (R1, R9).  force_mesh: host array of 3 device
 * pointers, overwritten.  The inputs are not modified. */
int pm_poisson_force(pm_ctx* ctx, const float* delta_mesh, const float* delta_mesh2,
                     float* const force_mesh[3], void* stream);
/* Transpose of pm_poisson_force: delta_cot = IFFT( sum_a conj(S_a) FFT(force_cot[a]) ) (overwritten);
 * delta_cot2 receives the cotangent of the second grid iff interlace = 1 (else must be NULL). */
int pm_poisson_force_vjp(pm_ctx* ctx, const float* const force_cot[3], float* delta_cot,
                         float* delta_cot2, void* stream);

/* ---- a5: gather, Eq. C.2 ------------------------------------------------------------- */
/* out[i,a] = sum_j mesh[a][j] W(r_j - X_i + s), a < ncomp (1..3).  mesh: host array of ncomp device
 * pointers.  out: [N,ncomp], overwritten, in the caller's particle order. */
int pm_interp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N,
              const double* shift, float* out, void* stream);
/* VJP of pm_interp: given out_cot [N,ncomp],
 *   mesh_cot[a][j] += sum_i out_cot[i,a] W_j(X_i)                         (Eq. C.10; ACCUMULATES) or NULL
 *   pos_cot[i,b]    = sum_a out_cot[i,a] sum_j mesh[a][j] dW_j(X_i)/dX_i^b (Eq. C.12; overwritten) or NULL */
int pm_interp_vjp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N,
                  const double* shift, const float* out_cot, float* const mesh_cot[], float* pos_cot,
                  void* stream);

/* ---- NEXT-2: forward-mode rules, Eq. C.13, rule table :956-960 (method 0) ---------- */
/* Tangent of pm_assign, Eq. C.13a:
 *   mesh_tan[j] += sum_i [ w_tan[i] W_j(X_i) + w_i pos_tan[i,:] . dW_j(X_i)/dX_i ]     (-grad W_j = dW_j/dX_i, :860)
 * ACCUMULATES onto mesh_tan, which the caller initialises with the tangent of the input mesh (Eq. C.4) or zero.
 * w: [N] or NULL (ones); pos_tan: [N,3] or NULL (0); w_tan: [N] or NULL (0). */
int pm_assign_jvp(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift,
                  const float* pos_tan, const float* w_tan, float* mesh_tan, void* stream);
/* Tangent of pm_interp, Eq. C.13b (ncomp = 1 or 3):
 *   out_tan[i,a] = sum_j [ mesh_tan[a][j] W_j(X_i) + mesh[a][j] pos_tan[i,:] . dW_j(X_i)/dX_i ]
 * mesh_tan: host array of ncomp device pointers or NULL (0); pos_tan: [N,3] or NULL (0); out_tan: [N,ncomp],
 * overwritten. */
int pm_interp_jvp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N,
                  const double* shift, const float* pos_tan, const float* const mesh_tan[], float* out_tan,
                  void* stream);

/* ---- a6-a8, a12: NUFFT path (method = 1), exponential-of-semicircle kernel ------- */
/* fine[j] += sum_i c_i prod_a phi(2 (j_a - u_a)/w), u = X / (box/m_f); phi(z) = exp(beta (sqrt(1-z^2)-1)).
 * ACCUMULATES.  c: [N] or NULL (ones). */
int nufft_spread(pm_ctx* ctx, const float* pos, const float* c, int64_t N, float* fine, void* stream);
int nufft_spread_vjp(pm_ctx* ctx, const float* pos, const float* c, int64_t N, const float* fine_cot,
                     float* pos_cot, float* c_cot, void* stream);
/* Spread grid -> three fine force grids: FFT, keep |n_a| < m/2 (R8), divide by phi_hat twice (R10,
 * PAPER.md:262), Poisson + i k gradient, (coeff / n_particles) normalisation, zero-pad, inverse FFTs. */
int nufft_poisson_force(pm_ctx* ctx, const float* fine, int64_t n_particles, float* const force_fine[3],
                        void* stream);
int nufft_poisson_force_vjp(pm_ctx* ctx, const float* const force_cot[3], int64_t n_particles,
                            float* fine_cot, void* stream);
/* out[i,a] = sum_j fine[a][j] prod_b phi(2 (j_b - u_b)/w)  (Eq. 2.19 through the grid). */
int nufft_interp(pm_ctx* ctx, const float* const fine[], int ncomp, const float* pos, int64_t N,
                 float* out, void* stream);
int nufft_interp_vjp(pm_ctx* ctx, const float* const fine[], int ncomp, const float* pos, int64_t N,
                     const float* out_cot, float* const fine_cot[], float* pos_cot, void* stream);

/* ---- whole path ------------------------------------------------------------------------------------- */
/* force[i,:] = A(X_i): a0-a5 (method 0: bin, assign (x2 if interlaced), R2C, k-space, 3 C2R, gather; the
 * density contrast delta = (m^3/N) rho - 1 of Eq. 2.3 PAPER.md:92 is folded into the k-space kernel) or
 * a0, a6-a8 (method 1).  force: [N,3], overwritten. */
int pm_force(pm_ctx* ctx, const float* pos, int64_t N, float* force, void* stream);
/* pos_cot = force_cot^T dA/dX (a9-a11; App. C).  force_cot: [N,3]; pos_cot: [N,3],
 * overwritten.  The forward meshes are recomputed, unless the records are pinned (pm_bin) and the last pm_force
 * on this ctx ran on the pinned (pos, N): then its force meshes are reused (interlace 0 or 1). */
int pm_force_vjp(pm_ctx* ctx, const float* pos, int64_t N, const float* force_cot, float* pos_cot,
                 void* stream);
/* ---- NEXT-1: drift-kick-drift step (Eq. 2.14a-c) and its backward-in-time adjoint ----- */
/* One step, in place:  X <- X + tau1 V;  V <- alpha V + beta A(X);  X <- X + tau2 V   (A = pm_force of this ctx).
 * pos, vel: [N,3] device arrays, both overwritten.  Positions are kept in [0, box): every drift wraps, in fp32
 * arithmetic that is specified operation by operation (reading R18) so that a CPU reference evaluates
 * the force at bitwise the same positions.  The kick and the second drift run in the epilogue of the gather; no
 * force array is written.  alpha, beta, tau1, tau2 are plain scalars (Eq. 2.15-2.17 are the caller's business).
 * Drops any pm_bin pin (the positions change).  PM_ESTATE for a ctx with PM_FLAG_KERNEL_GRAD. */
int pm_dkd_step(pm_ctx* ctx, float* pos, float* vel, int64_t N, double tau1, double tau2, double alpha,
                double beta, void* stream);
/* The backward-in-time step of Table 3, rows in the table's order, in place:
 *   in : (X^n, V^n, X*^n, V*^n)        out: (X^{n-1}, V^{n-1}, X*^{n-1}, V*^{n-1})
 * with the same (tau1, tau2, alpha, beta) the forward step n-1 -> n used.  The acceleration A(X^{n-1/2}) and
 * its VJP with V*^{n-1/2} share ONE set of forward meshes.  scalar_adj: device pointer to 4
 * doubles or NULL; receives the adjoints of the temporal coefficients of this step {tau1*, tau2*, alpha*,
 * beta*} (overwritten; alpha* = V*^{n-1/2} . V^{n-1}: DESIGN.md reading R19). */
int pm_dkd_step_adjoint(pm_ctx* ctx, float* pos, float* vel, float* pos_adj, float* vel_adj, int64_t N,
                        double tau1, double tau2, double alpha, double beta, double* scalar_adj, void* stream);

/* ---- NEXT-4: analysis ------------------------------------------------------------------------------- */
/* Shell-averaged (cross-)power spectrum of the density of `pos` (x `pos2`; NULL = auto spectrum).
 * The density is assigned with the ctx's worder and, if interlace = 1, combined from two interlaced grids;
 * deconvolve != 0 divides by ONE power of the assignment window (reading R20).  Bin b (0 <= b < nbins,
 * nbins <= m) holds the modes of the full Fourier cube with b + 1/2 <= |n| < b + 3/2, k = 2 pi n / box.
 * Outputs: device arrays of nbins doubles: mean |k| of the bin, P = box^3 <Re(dA conj dB)> / m^6 (no shot-noise
 * subtraction), number of modes; empty bins give 0.  method 0 only. */
int pm_power_spectrum(pm_ctx* ctx, const float* pos, int64_t N, const float* pos2, int64_t N2, int deconvolve,
                      int nbins, double* k_mean, double* power, double* n_modes, void* stream);
/* The shell binning of pm_power_spectrum on spectra the CALLER holds, for callers that cannot allocate (CUDA graph
 * capture, serving loops, harnesses that forbid cudaMalloc): no ctx, and the call makes no cudaMalloc / cudaFree
 * and calls no allocating library routine.  Runs on the CURRENT device.
 *   spec_a, spec_b : device arrays of m * m * (m/2 + 1) complex (interleaved re, im; the half-complex layout of a
 *                    3-D R2C transform of a real [m][m][m] mesh, z fastest); spec_b NULL = auto spectrum.
 *   outputs        : device arrays of nbins doubles, overwritten:  n_modes(b) = number of modes of the full
 *                    Fourier cube with b + 1/2 <= |n| < b + 3/2 (reading R20),  k_mean(b) = (2 pi / box) <|n|>,
 *                    power(b) = norm * <Re(A conj B)>  (norm = box^3 / (N_A N_B) for particle-count meshes
 *                    reproduces pm_power_spectrum without interlacing and deconvolution).  Empty bins give 0.
 *   errbuf         : host buffer of errbuf_len bytes (or NULL) that receives a message when the status is not PM_OK.
 * The kernel's scratch (3 * nbins fp64 accumulators) is a static __device__ array of PM_NOALLOC_MAX_BINS bins
 * (24 KB on every GPU that loads the library, until exit): nbins beyond it is rejected with PM_EINVAL.  Every call
 * on a device shares that array and clears it first, in stream order; calls that OVERLAP on the GPU (different
 * streams without a dependency) race on it.  The first call on a device looks the array's address up
 * (cudaGetSymbolAddress): make it outside graph capture. */
#define PM_NOALLOC_MAX_BINS 1024
int pm_mesh_power_noalloc(const float* spec_a, const float* spec_b, int32_t m, double box, double norm,
                          int32_t nbins, double* k_mean, double* power, double* n_modes, char* errbuf,
                          int32_t errbuf_len, void* stream);
/* Sheet-based resampling, trilinear variant (Table 5 n_resample :411; reading R21).
 * pos: [n_p^3, 3] in Lagrangian (C) order (particle (i,j,k) started at (i,j,k) box/n_p); pos_out:
 * [(r n_p)^3, 3], the refined sheet X' = q' + trilinear interpolation of the displacement, wrapped into
 * [0, box); feed it to pm_assign with weights r^-3.  Any ctx with the right box serves (m is not used). */
int pm_sheet_resample(pm_ctx* ctx, const float* pos, int32_t n_p, int32_t r, float* pos_out, void* stream);

/* Same as pm_force with HOST buffers: copies pos_host to the device, runs pm_force, copies the forces
 * back and synchronises.  Pinned host memory gives asynchronous copies; pageable memory also works. */
int pm_force_host(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream);
/* The same without the final synchronisation: the three steps are enqueued on `stream` and the call returns.  The
 * host buffers must stay valid -- and must be pinned for the copies to be asynchronous -- until the caller has
 * synchronised the stream.  One evaluation cannot overlap its own two copies (every force depends on every
 * position), but two evaluations in flight can: with two ctx on two streams the device-to-host copy of one
 * overlaps the host-to-device copy of the next and both directions of the host link stay busy (bench.py, e2e).
 * The first call on a ctx allocates its staging buffers (and synchronises the device once). */
int pm_force_host_async(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream);

/* ---- measurement ------------------------------------------------------------------------------------ */
/* When enabled, pm_force / pm_force_vjp record CUDA events around each stage on the caller's stream. */
int pm_set_profiling(pm_ctx* ctx, int enable);
#define PM_STAGE_BIN 0
#define PM_STAGE_ASSIGN 1
#define PM_STAGE_FFT_FWD 2
#define PM_STAGE_KSPACE 3
#define PM_STAGE_FFT_INV 4
#define PM_STAGE_INTERP 5
#define PM_STAGE_VJP_SCATTER 6
#define PM_STAGE_VJP_KSPACE 7 /* 3 R2C + transposed kernel + C2R */
#define PM_STAGE_VJP_GATHER 8
#define PM_STAGE_GRADIENT 9 /* real-space stencil of PM_FLAG_GRAD_REAL */
#define PM_STAGE_STEP 10    /* drift / adjoint-drift kernels of pm_dkd_step(_adjoint) */
#define PM_NUM_STAGES 11
/* Synchronises on the last profiled call and writes the duration in ms of each stage (0 if it did not
 * run) to ms_host[0..n-1], n <= PM_NUM_STAGES.  launches_host (or NULL) receives how many kernels of
 * this library (cuFFT's excluded) that call launched. */
int pm_get_stage_ms(pm_ctx* ctx, float* ms_host, int n, int64_t* launches_host);
/* Measured ceiling of the shared-memory pipe on this device, in lane operations per second (the roofline of the NUFFT
 * spreading / interpolation kernels, which are bound by shared-memory atomics and loads, not by HBM):
 * kind 0 = conflict-free 32-bit loads, 1 = conflict-free 32-bit integer atomic adds, 2 = 128-bit loads (counted as
 * 4 words).  Runs a micro-kernel for a few milliseconds and synchronises. */
int pm_smem_peak(pm_ctx* ctx, int kind, double* lane_ops_per_s_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* PMFORCE_H */
