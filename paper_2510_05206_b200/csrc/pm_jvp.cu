// pm_jvp.cu -- forward-mode rules of the interpolation operators, Eq. C.13, rule table :956-960:
//   scatter: rho~_j = rho~_in,j + sum_i [ w~_i W_j(X_i) - w_i X~_i . grad W_j(X_i) ]      (k_scatter, W_JVP)
//   gather : v~_i   = sum_j [ rho~_j W_j(X_i) - rho_j X~_i . grad W_j(X_i) ]               (k_gather, G_JVP / G_JVPT)
// with -grad W_j(X_i) = dW_j/dX_i (:860).  Instantiations for CIC / TSC / PCS, plain or shifted grid.
#include "pm_mesh_kernels.cuh"

namespace pmf {

template <int ORDER, bool SHIFTED>
static int scatter_jvp_os(Ctx* c, const ShiftSplit& sh, const ScatterSrc& src, float* mesh, cudaStream_t st) {
  using T = PMTraits<ORDER, SHIFTED>;
  typename T::Params tp;
  for (int a = 0; a < 3; ++a) tp.frac[a] = sh.frac[a];
  return run_scatter<T, 1, W_JVP>(c, tp, sh.roll, src, &mesh, st);
}

int launch_scatter_jvp(Ctx* c, int order, const ShiftSplit& sh, const float* w, const float* w_tan,
                       const float* pos_tan, float* mesh_tan, cudaStream_t st) {
  if (c->bin_n == 0) return PM_OK;
  ScatterSrc src = {w, 1, w_tan, pos_tan, (float)((double)c->mg / c->p.box)};
  switch (order * 2 + (sh.shifted ? 1 : 0)) {
    case 4: return scatter_jvp_os<2, false>(c, sh, src, mesh_tan, st);
    case 5: return scatter_jvp_os<2, true>(c, sh, src, mesh_tan, st);
    case 6: return scatter_jvp_os<3, false>(c, sh, src, mesh_tan, st);
    case 7: return scatter_jvp_os<3, true>(c, sh, src, mesh_tan, st);
    case 8: return scatter_jvp_os<4, false>(c, sh, src, mesh_tan, st);
    case 9: return scatter_jvp_os<4, true>(c, sh, src, mesh_tan, st);
  }
  return fail(c, PM_EINVAL, "worder must be 2, 3 or 4");
}

template <int ORDER, bool SHIFTED>
static int gather_jvp_os(Ctx* c, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  using T = PMTraits<ORDER, SHIFTED>;
  typename T::Params tp;
  for (int k = 0; k < 3; ++k) tp.frac[k] = sh.frac[k];
  switch (a.ncomp * 2 + (a.has_mesh_tan ? 1 : 0)) {
    case 2: return run_gather<T, 1, G_JVP>(c, tp, sh.roll, a, st);
    case 3: return run_gather<T, 2, G_JVPT>(c, tp, sh.roll, a, st);
    case 6: return run_gather<T, 3, G_JVP>(c, tp, sh.roll, a, st);
    case 7: return run_gather<T, 6, G_JVPT>(c, tp, sh.roll, a, st);
  }
  return fail(c, PM_EINVAL, "forward-mode gather: ncomp must be 1 or 3");
}

int launch_gather_jvp(Ctx* c, int order, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  switch (order * 2 + (sh.shifted ? 1 : 0)) {
    case 4: return gather_jvp_os<2, false>(c, sh, a, st);
    case 5: return gather_jvp_os<2, true>(c, sh, a, st);
    case 6: return gather_jvp_os<3, false>(c, sh, a, st);
    case 7: return gather_jvp_os<3, true>(c, sh, a, st);
    case 8: return gather_jvp_os<4, false>(c, sh, a, st);
    case 9: return gather_jvp_os<4, true>(c, sh, a, st);
  }
  return fail(c, PM_EINVAL, "worder must be 2, 3 or 4");
}

}  // namespace pmf
