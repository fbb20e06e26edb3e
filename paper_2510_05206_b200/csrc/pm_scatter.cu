// pm_scatter.cu -- a1 / a9: B-spline mass assignment (Eq. C.1, Table 1) and the vector scatter of
// cotangents (Eq. C.10): instantiations of k_scatter for CIC / TSC / PCS, plain or shifted grid.
#include "pm_mesh_kernels.cuh"

namespace pmf {

template <int ORDER, bool SHIFTED>
static int scatter_os(Ctx* c, const ShiftSplit& sh, int ncomp, const float* wsrc, int wstride,
                      float* const mesh[], cudaStream_t st) {
  using T = PMTraits<ORDER, SHIFTED>;
  typename T::Params tp;
  for (int a = 0; a < 3; ++a) tp.frac[a] = sh.frac[a];
  if (!wsrc) {  // unit weights: every component receives the same field
    // CIC: four warp-private accumulator tiles per CTA fit four CTAs on an SM -> the barrier-free kernel
    for (int a = 0; a < ncomp; ++a) {
      if constexpr (ORDER == 2)
        PM_TRY((run_scatter_warp<T>(c, tp, sh.roll, mesh[a], st)));
      else
        PM_TRY((run_scatter<T, 1, W_UNIT>(c, tp, sh.roll, weights_src(nullptr, 0), mesh + a, st)));
    }
    return PM_OK;
  }
  if (ncomp == 3) return run_scatter<T, 3, W_WEIGHTED>(c, tp, sh.roll, weights_src(wsrc, wstride), mesh, st);
  for (int a = 0; a < ncomp; ++a)
    PM_TRY((run_scatter<T, 1, W_WEIGHTED>(c, tp, sh.roll, weights_src(wsrc + a, wstride), mesh + a, st)));
  return PM_OK;
}

int launch_scatter(Ctx* c, int order, const ShiftSplit& sh, int ncomp, const float* wsrc, int wstride,
                   float* const mesh[], cudaStream_t st) {
  if (ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "ncomp must be 1..3");
  if (c->bin_n == 0) return PM_OK;
  switch (order * 2 + (sh.shifted ? 1 : 0)) {
    case 4: return scatter_os<2, false>(c, sh, ncomp, wsrc, wstride, mesh, st);
    case 5: return scatter_os<2, true>(c, sh, ncomp, wsrc, wstride, mesh, st);
    case 6: return scatter_os<3, false>(c, sh, ncomp, wsrc, wstride, mesh, st);
    case 7: return scatter_os<3, true>(c, sh, ncomp, wsrc, wstride, mesh, st);
    case 8: return scatter_os<4, false>(c, sh, ncomp, wsrc, wstride, mesh, st);
    case 9: return scatter_os<4, true>(c, sh, ncomp, wsrc, wstride, mesh, st);
  }
  return fail(c, PM_EINVAL, "worder must be 2, 3 or 4");
}

}  // namespace pmf
