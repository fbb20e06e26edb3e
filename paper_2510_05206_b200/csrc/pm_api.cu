// pm_api.cu -- the extern "C" entry points of include/pmforce.h: argument checks, stage composition.
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
  for (int a = 0; a < 3; ++a) PM_CUDA(c, cudaMalloc((void**)&c->gbar[a], sizeof(float) * (size_t)c->G));
  c->vjp_ready = true;
  return PM_OK;
}

// delta spectra of the ctx meshes rho[0] (, rho[1]) -> force meshes g[0..2].  coeff_eff carries every
// scalar: coeff, the density-contrast factor m^3/N of Eq. 2.3 and cuFFT's missing 1/m^3.
int spectra_to_force_meshes(Ctx* c, int ngrids, double coeff_eff, cudaStream_t st) {
  return spectral_forward(c, c->rho[0], ngrids == 2 ? c->rho[1] : nullptr, c->g, coeff_eff, true, st);
}

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

// One complete force evaluation on the grid shifted by `sh`; out = alpha * F (+ out).
int force_single(Ctx* c, int64_t N, const ShiftSplit& sh, bool second_grid, float alpha, bool accumulate,
                 float* force, cudaStream_t st) {
  PM_TRY(assign_ctx_meshes(c, sh, second_grid, st));
  PM_TRY(spectra_to_force_meshes(c, second_grid ? 2 : 1, c->p.coeff / (double)N, st));
  stage_begin(c, PM_STAGE_INTERP, st);
  const float* gm[3] = {c->g[0], c->g[1], c->g[2]};
  PM_TRY(gather_any(c, sh, gather_values(3, gm, force, alpha, accumulate), st));
  stage_end(c, PM_STAGE_INTERP, st);
  return PM_OK;
}

// One complete VJP on the grid shifted by `sh`: pos_cot = alpha * lam^T dF/dX (+ pos_cot).
int force_vjp_single(Ctx* c, int64_t N, const ShiftSplit& sh, bool second_grid, const float* lam, float alpha,
                     bool accumulate, float* pos_cot, cudaStream_t st) {
  PM_TRY(ensure_vjp_buffers(c));
  const double coeff_eff = c->p.coeff / (double)N;
  // forward meshes g_a (needed by the direct term, Eq. C.12)
  PM_TRY(assign_ctx_meshes(c, sh, second_grid, st));
  PM_TRY(spectra_to_force_meshes(c, second_grid ? 2 : 1, coeff_eff, st));
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
  GatherArgs ga = {4, m4, true, lam, 3, 3, 1.0f, nullptr, alpha, accumulate, pos_cot};
  int rc = gather_any(c, sh, ga, st);
  if (rc == PM_EINVAL && c->p.method == 1) {  // ES kernel too wide for 4 staged meshes: 3 + 1
    GatherArgs g3 = {3, m4, true, lam, 3, 3, 0.0f, nullptr, alpha, accumulate, pos_cot};
    PM_TRY(gather_any(c, sh, g3, st));
    GatherArgs g1 = {1, m4 + 3, true, nullptr, 0, 0, 1.0f, nullptr, alpha, true, pos_cot};
    rc = gather_any(c, sh, g1, st);
  }
  PM_TRY(rc);
  if (second_grid) {
    const float* m1[1] = {c->rho[1]};
    GatherArgs g2 = {1, m1, true, nullptr, 0, 0, 1.0f, nullptr, alpha, true, pos_cot};
    PM_TRY(launch_gather(c, c->p.worder, half_cell(c), g2, st));
  }
  stage_end(c, PM_STAGE_VJP_GATHER, st);
  return PM_OK;
}

void reset_profile(Ctx* c) {
  c->launches = 0;
  for (int s = 0; s < PM_NUM_STAGES; ++s) c->ev_used[s] = false;
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
  if (pos_cot) {
    GatherArgs ga = {1, m1, true, nullptr, 0, 0, 1.0f, w, 1.0f, false, pos_cot};
    PM_TRY(launch_gather(c, c->p.worder, sh, ga, S(stream)));
  }
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
  if (pos_cot) {
    GatherArgs ga = {ncomp, mesh, true, out_cot, ncomp, ncomp, 0.0f, nullptr, 1.0f, false, pos_cot};
    PM_TRY(launch_gather(c, c->p.worder, sh, ga, S(stream)));
  }
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
  if (pos_cot) {
    GatherArgs ga = {1, m1, true, nullptr, 0, 0, 1.0f, cw, 1.0f, false, pos_cot};
    PM_TRY(launch_es_gather(c, ga, S(stream)));
  }
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
  if (pos_cot) {
    GatherArgs ga = {ncomp, fine, true, out_cot, ncomp, ncomp, 0.0f, nullptr, 1.0f, false, pos_cot};
    PM_TRY(launch_es_gather(c, ga, S(stream)));
  }
  return PM_OK;
}

// ---- whole path --------------------------------------------------------------------------------------
int pm_force(pm_ctx* ctx, const float* pos, int64_t N, float* force, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  if (!force) return fail(c, PM_EINVAL, "force is NULL");
  if (N < 1) return fail(c, PM_EINVAL, "N must be >= 1");
  cudaStream_t st = S(stream);
  reset_profile(c);
  stage_begin(c, PM_STAGE_BIN, st);
  c->zero_done = false;
  c->zero_req = c->rho[0];  // cleared by the histogram pass when it runs (pm_bin.cu, zero-fill rider)
  c->zero_req_bytes = sizeof(float) * (size_t)c->G;
  const int brc = ensure_bins(c, pos, N, st, false);
  c->zero_req = nullptr;
  PM_TRY(brc);
  stage_end(c, PM_STAGE_BIN, st);
  const ShiftSplit none = split_shift(c, nullptr);
  if (c->p.method == 0 && c->p.interlace == 2) {  // R1 mode 2: average of two complete evaluations
    PM_TRY(force_single(c, N, none, false, 0.5f, false, force, st));
    return force_single(c, N, half_cell(c), false, 0.5f, true, force, st);
  }
  return force_single(c, N, none, c->p.method == 0 && c->p.interlace == 1, 1.0f, false, force, st);
}

int pm_force_vjp(pm_ctx* ctx, const float* pos, int64_t N, const float* force_cot, float* pos_cot, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  if (!force_cot || !pos_cot) return fail(c, PM_EINVAL, "force_cot / pos_cot is NULL");
  if (N < 1) return fail(c, PM_EINVAL, "N must be >= 1");
  cudaStream_t st = S(stream);
  reset_profile(c);
  stage_begin(c, PM_STAGE_BIN, st);
  c->zero_done = false;
  c->zero_req = c->rho[0];  // cleared by the histogram pass when it runs (pm_bin.cu, zero-fill rider)
  c->zero_req_bytes = sizeof(float) * (size_t)c->G;
  const int brc = ensure_bins(c, pos, N, st, false);
  c->zero_req = nullptr;
  PM_TRY(brc);
  stage_end(c, PM_STAGE_BIN, st);
  const ShiftSplit none = split_shift(c, nullptr);
  if (c->p.method == 0 && c->p.interlace == 2) {
    PM_TRY(force_vjp_single(c, N, none, false, force_cot, 0.5f, false, pos_cot, st));
    return force_vjp_single(c, N, half_cell(c), false, force_cot, 0.5f, true, pos_cot, st);
  }
  return force_vjp_single(c, N, none, c->p.method == 0 && c->p.interlace == 1, force_cot, 1.0f, false, pos_cot, st);
}

int pm_force_host(pm_ctx* ctx, const float* pos_host, int64_t N, float* force_host, void* stream) {
  Ctx* c = C(ctx);
  if (!c) return PM_EINVAL;
  if (!pos_host || !force_host) return fail(c, PM_EINVAL, "host pointer is NULL");
  if (N < 1 || N > c->cap) return fail(c, PM_EINVAL, "N outside [1, max_particles]");
  cudaStream_t st = S(stream);
  if (!c->host_pos_dev) {
    PM_CUDA(c, cudaMalloc((void**)&c->host_pos_dev, sizeof(float) * 3 * (size_t)c->cap));
    PM_CUDA(c, cudaMalloc((void**)&c->host_force_dev, sizeof(float) * 3 * (size_t)c->cap));
  }
  const size_t bytes = sizeof(float) * 3 * (size_t)N;
  PM_CUDA(c, cudaMemcpyAsync(c->host_pos_dev, pos_host, bytes, cudaMemcpyHostToDevice, st));
  PM_TRY(pm_force(ctx, c->host_pos_dev, N, c->host_force_dev, stream));
  PM_CUDA(c, cudaMemcpyAsync(force_host, c->host_force_dev, bytes, cudaMemcpyDeviceToHost, st));
  PM_CUDA(c, cudaStreamSynchronize(st));
  return PM_OK;
}

}  // extern "C"
