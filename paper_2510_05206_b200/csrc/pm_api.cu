// pm_api.cu -- the extern "C" entry points of include/pmforce.h: argument checks, stage composition.
#include <math.h>

#include "pm_internal.cuh"

using namespace pmf;

namespace {

inline cudaStream_t S(void* s) { return (cudaStream_t)s; }

int need_method(Ctx* c, int method, const char* who) {
  if (!c) return PM_EINVAL;
  if (c->p.method != method)
    return fail(c, PM_ESTATE, "%s needs a ctx created with method = %d", who, method);
  return enter_device(c);
}

ShiftSplit half_cell(const Ctx* c) {
  const double h = 0.5 * c->p.box / c->mg;
  const double s[3] = {h, h, h};
  return split_shift(c, s);
}

int ensure_vjp_buffers(Ctx* c) {
  if (c->vjp_ready) return PM_OK;
  float* t[3] = {nullptr, nullptr, nullptr};
  for (int a = 0; a < 3; ++a) {
    const cudaError_t e = cudaMalloc((void**)&t[a], sizeof(float) * (size_t)c->G);
    if (e != cudaSuccess) {  // all or nothing: a partial set would leak on the next attempt
      for (int k = 0; k < a; ++k) cudaFree(t[k]);
      return fail(c, PM_ENOMEM, "cudaMalloc of the VJP meshes failed: %s", cudaGetErrorString(e));
    }
  }
  for (int a = 0; a < 3; ++a) c->gbar[a] = t[a];
  c->vjp_ready = true;
  return PM_OK;
}

bool kernel_grad(const Ctx* c) { return c->p.method == 1 && (c->p.flags & PM_FLAG_KERNEL_GRAD); }

// a1: assignment of unit-mass particles onto the ctx meshes (interlace 1: also the half-cell shifted grid)
int assign_ctx_meshes(Ctx* c, const ShiftSplit& sh, bool second_grid, cudaStream_t st) {
  stage_begin(c, PM_STAGE_ASSIGN, st);
  if (!c->zero_done) PM_CUDA(c, cudaMemsetAsync(c->rho[0], 0, sizeof(float) * (size_t)c->G, st));
  c->zero_done = false;  // consumed: a second evaluation in the same call clears the mesh itself
  if (c->p.method == 0) {
    c->scatter_mesh_zeroed = true;  // the ctx meshes were just cleared: exclusive tile interiors may be stored
    int rc = launch_scatter(c, c->p.worder, sh, 1, nullptr, 0, &c->rho[0], st);
    if (rc == PM_OK && second_grid) {
      rc = (cudaMemsetAsync(c->rho[1], 0, sizeof(float) * (size_t)c->G, st) == cudaSuccess) ? PM_OK : PM_ECUDA;
      if (rc == PM_OK) rc = launch_scatter(c, c->p.worder, half_cell(c), 1, nullptr, 0, &c->rho[1], st);
    }
    c->scatter_mesh_zeroed = false;
    PM_TRY(rc);
  } else {
    PM_TRY(launch_es_scatter(c, 1, nullptr, 0, &c->rho[0], st));
  }
  stage_end(c, PM_STAGE_ASSIGN, st);
  return PM_OK;
}

int gather_any(Ctx* c, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  return c->p.method == 0 ? launch_gather(c, c->p.worder, sh, a, st) : launch_es_gather(c, a, st);
}

// a1-a4 on the grid shifted by `sh`: the binned particles -> force meshes g[0..2] (or, for the NUFFT
// kernel-gradient option, the potential mesh phi).  coeff_eff carries every scalar: coeff, the density-contrast
// factor m^3/N of Eq. 2.3 and cuFFT's missing 1/m^3.
// for_vjp: the meshes feed grad-W gathers (the direct term of the VJP, Eq. C.12), which difference g between
// neighbouring nodes.  The real-space stencil of PM_FLAG_GRAD_REAL leaves white rounding noise eps |phi| / Delta on g
// (phi is dominated by low k and much larger than Delta |grad phi|): harmless for the force itself (1e-6), amplified
// by that second difference (measured 1.85e-5 on the VJP at 512^3, 4e-6 at 64^3).  Reverse-mode calls therefore
// always take the three-inverse-FFT meshes, whatever the flag says.
int forward_meshes(Ctx* c, int64_t N, const ShiftSplit& sh, bool second_grid, bool for_vjp, cudaStream_t st) {
  c->g_valid = false;
  PM_TRY(assign_ctx_meshes(c, sh, second_grid, st));
  const double coeff_eff = c->p.coeff / (double)N;
  if (kernel_grad(c)) {
    PM_TRY(ensure_phi(c));
    return spectral_potential(c, c->rho[0], nullptr, c->phi, coeff_eff, true, st);
  }
  const int32_t flags = c->p.flags;
  if (for_vjp) c->p.flags &= ~PM_FLAG_GRAD_REAL;
  const int rc = spectral_forward(c, c->rho[0], second_grid ? c->rho[1] : nullptr, c->g, coeff_eff, true, st);
  c->p.flags = flags;
  return rc;
}

// a5: per-particle values of the force meshes with the epilogue of `ga` (out = alpha * A + out_scale * out, ...)
int gather_force(Ctx* c, const ShiftSplit& sh, GatherArgs ga, cudaStream_t st) {
  stage_begin(c, PM_STAGE_INTERP, st);
  const float* gm[3] = {c->g[0], c->g[1], c->g[2]};
  const float* ph[1] = {c->phi};
  if (kernel_grad(c)) {  // A = -grad of the ES interpolant of phi
    GatherArgs gg = gather_grad(1, ph, nullptr, 0, 0, 1.0f, nullptr, ga.out, -ga.alpha, ga.out_scale);
    PM_TRY(gather_any(c, sh, gg, st));
  } else {
    ga.ncomp = 3;
    ga.mesh = gm;
    PM_TRY(gather_any(c, sh, ga, st));
  }
  stage_end(c, PM_STAGE_INTERP, st);
  return PM_OK;
}

// a9-a11 on the grid shifted by `sh`, given the forward meshes g[0..2] of the same grid:
// pos_cot = alpha * lam^T dF/dX + out_scale * pos_cot.
int vjp_from_meshes(Ctx* c, int64_t N, const ShiftSplit& sh, bool second_grid, const float* lam, float alpha,
                    float out_scale, float* pos_cot, cudaStream_t st) {
  PM_TRY(ensure_vjp_buffers(c));
  const double coeff_eff = c->p.coeff / (double)N;
  // (ii) gbar_a = scatter(lam_a)  (Eq. C.10)
  stage_begin(c, PM_STAGE_VJP_SCATTER, st);
  for (int a = 0; a < 3; ++a) PM_CUDA(c, cudaMemsetAsync(c->gbar[a], 0, sizeof(float) * (size_t)c->G, st));
  if (c->p.method == 0)
    PM_TRY(launch_scatter(c, c->p.worder, sh, 3, lam, 3, c->gbar, st));
  else
    PM_TRY(launch_es_scatter(c, 3, lam, 3, c->gbar, st));
  stage_end(c, PM_STAGE_VJP_SCATTER, st);
  // (iii) rho_bar = IFFT( sum_a conj(S_a) FFT(gbar_a) ), with the m^3/N of the density contrast folded in
  stage_begin(c, PM_STAGE_VJP_KSPACE, st);
  PM_TRY(spectral_transpose(c, c->gbar, c->rho[0], second_grid ? c->rho[1] : nullptr, coeff_eff, st));
  stage_end(c, PM_STAGE_VJP_KSPACE, st);
  // (i) + (iv): grad-W gathers (Eq. C.12 weighted by lam, Eq. C.6 with w_i = 1)
  stage_begin(c, PM_STAGE_VJP_GATHER, st);
  const float* m4[4] = {c->g[0], c->g[1], c->g[2], c->rho[0]};
  int rc = gather_any(c, sh, gather_grad(4, m4, lam, 3, 3, 1.0f, nullptr, pos_cot, alpha, out_scale), st);
  if (rc == PM_EINVAL && c->p.method == 1) {  // ES kernel too wide for 4 staged meshes: 3 + 1
    PM_TRY(gather_any(c, sh, gather_grad(3, m4, lam, 3, 3, 0.0f, nullptr, pos_cot, alpha, out_scale), st));
    rc = gather_any(c, sh, gather_grad(1, m4 + 3, nullptr, 0, 0, 1.0f, nullptr, pos_cot, alpha, 1.0f), st);
  }
  PM_TRY(rc);
  if (second_grid) {
    const float* m1[1] = {c->rho[1]};
    PM_TRY(launch_gather(c, c->p.worder, half_cell(c), gather_grad(1, m1, nullptr, 0, 0, 1.0f, nullptr, pos_cot, alpha, 1.0f), st));
  }
  stage_end(c, PM_STAGE_VJP_GATHER, st);
  return PM_OK;
}

// The evaluations one force call is made of (R1): one, or two half-weighted ones for interlace = 2.
struct Evals {
  int n;
  ShiftSplit sh[2];
  bool second_grid;
  float weight;
};
Evals evals_of(const Ctx* c) {
  Evals e;
  e.sh[0] = split_shift(c, nullptr);
  e.sh[1] = half_cell(c);
  const bool two = c->p.method == 0 && c->p.interlace == 2;
  e.n = two ? 2 : 1;
  e.weight = two ? 0.5f : 1.0f;
  e.second_grid = c->p.method == 0 && c->p.interlace == 1;
  return e;
}

// binning of a whole-path call, with the zero-fill rider for the assignment mesh
int bin_for_path(Ctx* c, const float* pos, int64_t N, cudaStream_t st) {
  stage_begin(c, PM_STAGE_BIN, st);
  c->zero_done = false;
  c->zero_req = c->rho[0];  // cleared by the binning pass when it runs (pm_bin.cu, zero-fill rider)
  c->zero_req_bytes = sizeof(float) * (size_t)c->G;
  const int brc = ensure_bins(c, pos, N, st, false);
  c->zero_req = nullptr;
  PM_TRY(brc);
  stage_end(c, PM_STAGE_BIN, st);
  return PM_OK;
}

void reset_profile(Ctx* c) {
  c->launches = 0;
  c->ev_slot = 0;
  for (int e = 0; e < 2; ++e)
    for (int s = 0; s < PM_NUM_STAGES; ++s) c->ev_used[e][s] = false;
}

}  // namespace

extern "C" {

int pm_assign(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift, float* mesh,
              void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_assign"));
  if (!mesh) return fail(c, PM_EINVAL, "mesh is NULL");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  return launch_scatter(c, c->p.worder, split_shift(c, shift), 1, w, 1, &mesh, S(stream));
}

int pm_assign_vjp(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift,
                  const float* mesh_cot, float* pos_cot, float* w_cot, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_assign_vjp"));
  if (!mesh_cot) return fail(c, PM_EINVAL, "mesh_cot is NULL");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  const ShiftSplit sh = split_shift(c, shift);
  const float* m1[1] = {mesh_cot};
  if (pos_cot)
    PM_TRY(launch_gather(c, c->p.worder, sh, gather_grad(1, m1, nullptr, 0, 0, 1.0f, w, pos_cot), S(stream)));
  if (w_cot) PM_TRY(launch_gather(c, c->p.worder, sh, gather_values(1, m1, w_cot), S(stream)));
  return PM_OK;
}

int pm_poisson_force(pm_ctx* ctx, const float* delta_mesh, const float* delta_mesh2, float* const force_mesh[3],
                     void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_poisson_force"));
  const bool two = c->p.interlace == 1;
  if (!delta_mesh || !force_mesh || !force_mesh[0] || !force_mesh[1] || !force_mesh[2])
    return fail(c, PM_EINVAL, "NULL mesh pointer");
  if (two != (delta_mesh2 != nullptr))
    return fail(c, PM_EINVAL, "delta_mesh2 must be given iff interlace = 1");
  cudaStream_t st = S(stream);
  return spectral_forward(c, delta_mesh, two ? delta_mesh2 : nullptr, force_mesh, c->p.coeff / (double)c->G, false, st);
}

int pm_poisson_force_vjp(pm_ctx* ctx, const float* const force_cot[3], float* delta_cot, float* delta_cot2,
                         void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_poisson_force_vjp"));
  const bool two = c->p.interlace == 1;
  if (!delta_cot || !force_cot || !force_cot[0] || !force_cot[1] || !force_cot[2])
    return fail(c, PM_EINVAL, "NULL mesh pointer");
  if (two != (delta_cot2 != nullptr))
    return fail(c, PM_EINVAL, "delta_cot2 must be given iff interlace = 1");
  cudaStream_t st = S(stream);
  return spectral_transpose(c, force_cot, delta_cot, two ? delta_cot2 : nullptr, c->p.coeff / (double)c->G, st);
}

int pm_interp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N, const double* shift,
              float* out, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_interp"));
  if (!mesh || !out || ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "bad mesh / out / ncomp");
  for (int a = 0; a < ncomp; ++a)
    if (!mesh[a]) return fail(c, PM_EINVAL, "mesh[%d] is NULL", a);
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  return launch_gather(c, c->p.worder, split_shift(c, shift), gather_values(ncomp, mesh, out), S(stream));
}

int pm_interp_vjp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N,
                  const double* shift, const float* out_cot, float* const mesh_cot[], float* pos_cot, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_interp_vjp"));
  if (!out_cot || ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "bad out_cot / ncomp");
  if (pos_cot && !mesh) return fail(c, PM_EINVAL, "pos_cot needs the primal meshes");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  const ShiftSplit sh = split_shift(c, shift);
  if (mesh_cot) PM_TRY(launch_scatter(c, c->p.worder, sh, ncomp, out_cot, ncomp, mesh_cot, S(stream)));
  if (pos_cot)
    PM_TRY(launch_gather(c, c->p.worder, sh, gather_grad(ncomp, mesh, out_cot, ncomp, ncomp, 0.0f, nullptr, pos_cot),
                         S(stream)));
  return PM_OK;
}

// ---- NUFFT stages ------------------------------------------------------------------------------------
int nufft_spread(pm_ctx* ctx, const float* pos, const float* cw, int64_t N, float* fine, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_spread"));
  if (!fine) return fail(c, PM_EINVAL, "fine is NULL");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  return launch_es_scatter(c, 1, cw, 1, &fine, S(stream));
}

int nufft_spread_vjp(pm_ctx* ctx, const float* pos, const float* cw, int64_t N, const float* fine_cot,
                     float* pos_cot, float* c_cot, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_spread_vjp"));
  if (!fine_cot) return fail(c, PM_EINVAL, "fine_cot is NULL");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  const float* m1[1] = {fine_cot};
  if (pos_cot) PM_TRY(launch_es_gather(c, gather_grad(1, m1, nullptr, 0, 0, 1.0f, cw, pos_cot), S(stream)));
  if (c_cot) PM_TRY(launch_es_gather(c, gather_values(1, m1, c_cot), S(stream)));
  return PM_OK;
}

int nufft_poisson_force(pm_ctx* ctx, const float* fine, int64_t n_particles, float* const force_fine[3],
                        void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_poisson_force"));
  if (!fine || !force_fine || !force_fine[0] || !force_fine[1] || !force_fine[2] || n_particles < 1)
    return fail(c, PM_EINVAL, "NULL mesh pointer or n_particles < 1");
  cudaStream_t st = S(stream);
  return spectral_forward(c, fine, nullptr, force_fine, c->p.coeff / (double)n_particles, false, st);
}

int nufft_poisson_force_vjp(pm_ctx* ctx, const float* const force_cot[3], int64_t n_particles, float* fine_cot,
                            void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_poisson_force_vjp"));
  if (!fine_cot || !force_cot || !force_cot[0] || !force_cot[1] || !force_cot[2] || n_particles < 1)
    return fail(c, PM_EINVAL, "NULL mesh pointer or n_particles < 1");
  cudaStream_t st = S(stream);
  return spectral_transpose(c, force_cot, fine_cot, nullptr, c->p.coeff / (double)n_particles, st);
}

int nufft_interp(pm_ctx* ctx, const float* const fine[], int ncomp, const float* pos, int64_t N, float* out,
                 void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_interp"));
  if (!fine || !out || ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "bad fine / out / ncomp");
  for (int a = 0; a < ncomp; ++a)
    if (!fine[a]) return fail(c, PM_EINVAL, "fine[%d] is NULL", a);
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  return launch_es_gather(c, gather_values(ncomp, fine, out), S(stream));
}

int nufft_interp_vjp(pm_ctx* ctx, const float* const fine[], int ncomp, const float* pos, int64_t N,
                     const float* out_cot, float* const fine_cot[], float* pos_cot, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 1, "nufft_interp_vjp"));
  if (!out_cot || ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "bad out_cot / ncomp");
  if (pos_cot && !fine) return fail(c, PM_EINVAL, "pos_cot needs the primal grids");
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  if (fine_cot) PM_TRY(launch_es_scatter(c, ncomp, out_cot, ncomp, fine_cot, S(stream)));
  if (pos_cot)
    PM_TRY(launch_es_gather(c, gather_grad(ncomp, fine, out_cot, ncomp, ncomp, 0.0f, nullptr, pos_cot), S(stream)));
  return PM_OK;
}

// ---- whole path --------------------------------------------------------------------------------------
int pm_force(pm_ctx* ctx, const float* pos, int64_t N, float* force, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!force) return fail(c, PM_EINVAL, "force is NULL");
  if (N < 1) return fail(c, PM_EINVAL, "N must be >= 1");
  cudaStream_t st = S(stream);
  reset_profile(c);
  PM_TRY(bin_for_path(c, pos, N, st));
  const Evals ev = evals_of(c);
  for (int e = 0; e < ev.n; ++e) {
    c->ev_slot = e;
    PM_TRY(forward_meshes(c, N, ev.sh[e], ev.second_grid, false, st));
    PM_TRY(gather_force(c, ev.sh[e], gather_values(3, nullptr, force, ev.weight, e == 0 ? 0.0f : 1.0f), st));
  }
  // the meshes stay valid for a pm_force_vjp on the same pinned records (a single evaluation, Fourier-space gradient)
  c->g_valid = ev.n == 1 && c->bin_pinned && !kernel_grad(c) && !(c->p.flags & PM_FLAG_GRAD_REAL);
  return PM_OK;
}

int pm_force_vjp(pm_ctx* ctx, const float* pos, int64_t N, const float* force_cot, float* pos_cot, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!force_cot || !pos_cot) return fail(c, PM_EINVAL, "force_cot / pos_cot is NULL");
  if (N < 1) return fail(c, PM_EINVAL, "N must be >= 1");
  if (kernel_grad(c))
    return fail(c, PM_ESTATE, "pm_force_vjp is not built for PM_FLAG_KERNEL_GRAD (needs second derivatives of the kernel)");
  cudaStream_t st = S(stream);
  reset_profile(c);
  const bool reuse = c->g_valid && c->bin_valid && c->bin_pinned && c->bin_pos == pos && c->bin_n == N;
  PM_TRY(bin_for_path(c, pos, N, st));  // returns at once when the pinned records are those of (pos, N)
  const Evals ev = evals_of(c);
  for (int e = 0; e < ev.n; ++e) {
    c->ev_slot = e;
    if (!reuse) PM_TRY(forward_meshes(c, N, ev.sh[e], ev.second_grid, true, st));
    PM_TRY(vjp_from_meshes(c, N, ev.sh[e], ev.second_grid, force_cot, ev.weight, e == 0 ? 0.0f : 1.0f, pos_cot, st));
  }
  c->g_valid = reuse || (ev.n == 1 && c->bin_pinned);
  return PM_OK;
}

// ---- NEXT-1: drift-kick-drift step and its adjoint -----------------------------------------------------
int pm_dkd_step(pm_ctx* ctx, float* pos, float* vel, int64_t N, double tau1, double tau2, double alpha, double beta,
                void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!pos || !vel) return fail(c, PM_EINVAL, "pos / vel is NULL");
  if (N < 1 || N > c->cap) return fail(c, PM_EINVAL, "N outside [1, max_particles]");
  if (kernel_grad(c)) return fail(c, PM_ESTATE, "pm_dkd_step is not built for PM_FLAG_KERNEL_GRAD");
  cudaStream_t st = S(stream);
  reset_profile(c);
  c->bin_valid = false;  // the positions change
  c->g_valid = false;
  stage_begin(c, PM_STAGE_STEP, st);
  PM_TRY(launch_step_update(c, pos, vel, nullptr, nullptr, N, (float)tau1, 0.f, 0.f, nullptr, st));  // (2.14a)
  stage_end(c, PM_STAGE_STEP, st);
  PM_TRY(bin_for_path(c, pos, N, st));
  const Evals ev = evals_of(c);
  for (int e = 0; e < ev.n; ++e) {
    c->ev_slot = e;
    PM_TRY(forward_meshes(c, N, ev.sh[e], ev.second_grid, false, st));
    // (2.14b) V <- alpha V + beta A in the gather epilogue; after the last evaluation (2.14c) X <- X + tau2 V
    GatherArgs ga = gather_values(3, nullptr, vel, (float)beta * ev.weight, e == 0 ? (float)alpha : 1.0f);
    if (e == ev.n - 1) {
      ga.drift_pos = pos;
      ga.drift_tau = (float)tau2;
    }
    PM_TRY(gather_force(c, ev.sh[e], ga, st));
  }
  c->bin_valid = false;  // the records describe X^{n+1/2}, pos now holds X^{n+1}
  return PM_OK;
}

int pm_dkd_step_adjoint(pm_ctx* ctx, float* pos, float* vel, float* pos_adj, float* vel_adj, int64_t N, double tau1,
                        double tau2, double alpha, double beta, double* scalar_adj, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!pos || !vel || !pos_adj || !vel_adj) return fail(c, PM_EINVAL, "NULL state pointer");
  if (N < 1 || N > c->cap) return fail(c, PM_EINVAL, "N outside [1, max_particles]");
  if (alpha == 0.0) return fail(c, PM_EINVAL, "alpha = 0: the kick cannot be undone");
  if (kernel_grad(c)) return fail(c, PM_ESTATE, "pm_dkd_step_adjoint is not built for PM_FLAG_KERNEL_GRAD");
  cudaStream_t st = S(stream);
  reset_profile(c);
  if (!scalar_adj) {
    if (!c->step_dots) PM_CUDA(c, cudaMalloc((void**)&c->step_dots, 4 * sizeof(double)));
    scalar_adj = c->step_dots;
  }
  double* d_tau1 = scalar_adj, *d_tau2 = scalar_adj + 1, *d_alpha = scalar_adj + 2, *d_beta = scalar_adj + 3;
  PM_CUDA(c, cudaMemsetAsync(scalar_adj, 0, 4 * sizeof(double), st));
  c->bin_valid = false;
  c->g_valid = false;
  // Table 3: primal drift X^{n-1/2} = X^n - tau2 V^n; adjoint drift V*^{n-1/2} = V*^n + tau2 X*^n; tau2* = X*^n . V^n
  stage_begin(c, PM_STAGE_STEP, st);
  PM_TRY(launch_step_update(c, pos, vel, pos_adj, vel_adj, N, (float)-tau2, 1.0f, (float)tau2, d_tau2, st));
  stage_end(c, PM_STAGE_STEP, st);
  PM_TRY(bin_for_path(c, pos, N, st));
  const Evals ev = evals_of(c);
  for (int e = 0; e < ev.n; ++e) {
    c->ev_slot = e;
    PM_TRY(forward_meshes(c, N, ev.sh[e], ev.second_grid, true, st));
    // primal kick V^{n-1} = (V^n - beta A) / alpha, with beta* = V*^{n-1/2} . A and (after the last evaluation)
    // alpha* = V*^{n-1/2} . V^{n-1} reduced in the same pass
    GatherArgs ga = gather_values(3, nullptr, vel, (float)(-beta / alpha) * ev.weight, e == 0 ? (float)(1.0 / alpha) : 1.0f);
    ga.dot_with = vel_adj;
    ga.dot_acc = d_beta;
    ga.dot_scale = ev.weight;
    ga.dot_out = e == ev.n - 1 ? d_alpha : nullptr;
    PM_TRY(gather_force(c, ev.sh[e], ga, st));
    // adjoint kick X*^{n-1} = X*^n + beta V*^{n-1/2} . grad_X A(X^{n-1/2}): the VJP on the same meshes (:338)
    PM_TRY(vjp_from_meshes(c, N, ev.sh[e], ev.second_grid, vel_adj, (float)beta * ev.weight, 1.0f, pos_adj, st));
  }
  // rescale V*^K = alpha V*^{n-1/2}; primal drift X^{n-1} = X^{n-1/2} - tau1 V^{n-1}; adjoint drift
  // V*^{n-1} = V*^K + tau1 X*^{n-1}; tau1* = X*^{n-1} . V^{n-1}
  PM_TRY(launch_step_update(c, pos, vel, pos_adj, vel_adj, N, (float)-tau1, (float)alpha, (float)tau1, d_tau1, st));
  c->bin_valid = false;
  return PM_OK;
}

// ---- NEXT-2: forward-mode rules ------------------------------------------------------------------------
int pm_assign_jvp(pm_ctx* ctx, const float* pos, const float* w, int64_t N, const double* shift, const float* pos_tan,
                  const float* w_tan, float* mesh_tan, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_assign_jvp"));
  if (!mesh_tan) return fail(c, PM_EINVAL, "mesh_tan is NULL");
  if (!pos_tan && !w_tan) return PM_OK;  // zero tangents: mesh_tan keeps the tangent of the input mesh (Eq. C.4)
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  return launch_scatter_jvp(c, c->p.worder, split_shift(c, shift), w, w_tan, pos_tan, mesh_tan, S(stream));
}

int pm_interp_jvp(pm_ctx* ctx, const float* const mesh[], int ncomp, const float* pos, int64_t N, const double* shift,
                  const float* pos_tan, const float* const mesh_tan[], float* out_tan, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_interp_jvp"));
  if (!mesh || !out_tan || (ncomp != 1 && ncomp != 3)) return fail(c, PM_EINVAL, "bad mesh / out_tan, or ncomp not 1 or 3");
  const float* all[6];
  for (int a = 0; a < ncomp; ++a) {
    if (!mesh[a] || (mesh_tan && !mesh_tan[a])) return fail(c, PM_EINVAL, "mesh[%d] / mesh_tan[%d] is NULL", a, a);
    all[a] = mesh[a];
    if (mesh_tan) all[ncomp + a] = mesh_tan[a];
  }
  PM_TRY(ensure_bins(c, pos, N, S(stream), false));
  GatherArgs ga = gather_values(ncomp, all, out_tan);
  ga.mode = GATHER_JVP;
  ga.pos_tan = pos_tan;
  ga.has_mesh_tan = mesh_tan != nullptr;
  return launch_gather(c, c->p.worder, split_shift(c, shift), ga, S(stream));
}

// ---- NEXT-4: analysis ------------------------------------------------------------------------------------
int pm_power_spectrum(pm_ctx* ctx, const float* pos, int64_t N, const float* pos2, int64_t N2, int deconvolve,
                      int nbins, double* k_mean, double* power, double* n_modes, void* stream) {
  Ctx* c = C(ctx);
  PM_TRY(need_method(c, 0, "pm_power_spectrum"));
  if (!pos || !k_mean || !power || !n_modes) return fail(c, PM_EINVAL, "NULL pointer");
  if (N < 1 || (pos2 && N2 < 1)) return fail(c, PM_EINVAL, "N must be >= 1");
  if (nbins < 1 || nbins > c->mg) return fail(c, PM_EINVAL, "nbins must be in [1, m]");
  cudaStream_t st = S(stream);
  if (c->ps_nbins < nbins) {
    if (c->ps_acc) cudaFree(c->ps_acc);
    c->ps_acc = nullptr;
    c->ps_nbins = 0;
    PM_CUDA(c, cudaMalloc((void**)&c->ps_acc, sizeof(double) * 3 * (size_t)nbins));
    c->ps_nbins = nbins;
  }
  const bool two = c->p.interlace == 1;
  const ShiftSplit none = split_shift(c, nullptr);
  float2* spec[4] = {c->dhat[0], c->ghat[0], c->ghat[1], c->ghat[2]};  // A1, A2, B1, B2
  for (int set = 0; set < (pos2 ? 2 : 1); ++set) {
    const float* p = set == 0 ? pos : pos2;
    const int64_t n = set == 0 ? N : N2;
    PM_TRY(ensure_bins(c, p, n, st, false));
    c->g_valid = false;
    PM_CUDA(c, cudaMemsetAsync(c->rho[0], 0, sizeof(float) * (size_t)c->G, st));
    PM_TRY(launch_scatter(c, c->p.worder, none, 1, nullptr, 0, &c->rho[0], st));
    PM_TRY(fft_r2c(c, c->rho[0], spec[2 * set], st));
    if (two) {
      PM_CUDA(c, cudaMemsetAsync(c->rho[1], 0, sizeof(float) * (size_t)c->G, st));
      PM_TRY(launch_scatter(c, c->p.worder, half_cell(c), 1, nullptr, 0, &c->rho[1], st));
      PM_TRY(fft_r2c(c, c->rho[1], spec[2 * set + 1], st));
    }
  }
  PM_CUDA(c, cudaMemsetAsync(c->ps_acc, 0, sizeof(double) * 3 * (size_t)nbins, st));
  PM_TRY(launch_power_bins(c, spec[0], two ? spec[1] : nullptr, pos2 ? spec[2] : nullptr,
                           (pos2 && two) ? spec[3] : nullptr, deconvolve != 0, nbins, c->ps_acc, st));
  // delta_hat = (G/N) rho_hat off n = 0:  V/G^2 (G/N_A)(G/N_B) = V / (N_A N_B)
  const double pnorm = c->p.box * c->p.box * c->p.box / ((double)N * (double)(pos2 ? N2 : N));
  return launch_power_finish(c, nbins, c->ps_acc, 2.0 * M_PI / c->p.box, pnorm, k_mean, power, n_modes, st);
}

int pm_sheet_resample(pm_ctx* ctx, const float* pos, int32_t n_p, int32_t r, float* pos_out, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!pos || !pos_out) return fail(c, PM_EINVAL, "NULL pointer");
  if (n_p < 2 || r < 1 || (int64_t)n_p * r > 4096) return fail(c, PM_EINVAL, "n_p >= 2, r >= 1, n_p * r <= 4096");
  return launch_sheet_resample(c, pos, n_p, r, pos_out, S(stream));
}

static int force_host_impl(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream, bool sync) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  PM_TRY(enter_device(c));
  if (!pos_host || !force_host) return fail(c, PM_EINVAL, "host pointer is NULL");
  if (N < 1 || N > c->cap) return fail(c, PM_EINVAL, "N outside [1, max_particles]");
  cudaStream_t st = S(stream);
  if (!c->host_pos_dev || !c->host_force_dev) {  // both or neither
    float *a = nullptr, *b = nullptr;
    const cudaError_t ea = cudaMalloc((void**)&a, sizeof(float) * 3 * (size_t)c->cap);
    const cudaError_t eb = ea == cudaSuccess ? cudaMalloc((void**)&b, sizeof(float) * 3 * (size_t)c->cap) : ea;
    if (ea != cudaSuccess || eb != cudaSuccess) {
      if (a) cudaFree(a);
      cudaGetLastError();
      return fail(c, PM_ENOMEM, "cudaMalloc of the host staging buffers failed");
    }
    c->host_pos_dev = a;
    c->host_force_dev = b;
  }
  const size_t bytes = sizeof(float) * 3 * (size_t)N;
  PM_CUDA(c, cudaMemcpyAsync(c->host_pos_dev, pos_host, bytes, cudaMemcpyHostToDevice, st));
  PM_TRY(pm_force(ctx, c->host_pos_dev, N, c->host_force_dev, stream));
  PM_CUDA(c, cudaMemcpyAsync(force_host, c->host_force_dev, bytes, cudaMemcpyDeviceToHost, st));
  if (sync) PM_CUDA(c, cudaStreamSynchronize(st));
  return PM_OK;
}

int pm_force_host(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream) {
  return force_host_impl(ctx, pos_host, N, force_host, stream, true);
}

int pm_force_host_async(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream) {
  return force_host_impl(ctx, pos_host, N, force_host, stream, false);
}

}  // extern "C"
