// pm_gather.cu -- a5 / a11: B-spline gather (Eq. C.2) and the grad-W gathers of the VJP rules
// (Eq. C.6, Eq. C.12): instantiations of k_gather for CIC / TSC / PCS.
#include "pm_mesh_kernels.cuh"

namespace pmf {

template <class T, int NCOMP, bool GRAD>
static int go(Ctx* c, const typename T::Params& tp, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  return run_gather<T, NCOMP, GRAD>(c, tp, sh.roll, a.mesh, a.cot, a.cstride, a.ncot, a.const_coef, a.wmul, a.alpha,
                                    a.accumulate, a.out, st);
}

template <int ORDER, bool SHIFTED>
static int gather_os(Ctx* c, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  using T = PMTraits<ORDER, SHIFTED>;
  typename T::Params tp;
  for (int k = 0; k < 3; ++k) tp.frac[k] = sh.frac[k];
  switch (a.ncomp * 2 + (a.grad ? 1 : 0)) {
    case 2: return go<T, 1, false>(c, tp, sh, a, st);
    case 3: return go<T, 1, true>(c, tp, sh, a, st);
    case 4: return go<T, 2, false>(c, tp, sh, a, st);
    case 5: return go<T, 2, true>(c, tp, sh, a, st);
    case 6: return go<T, 3, false>(c, tp, sh, a, st);
    case 7: return go<T, 3, true>(c, tp, sh, a, st);
    case 9: return go<T, 4, true>(c, tp, sh, a, st);
  }
  return fail(c, PM_EINVAL, "gather: unsupported ncomp = %d", a.ncomp);
}

int launch_gather(Ctx* c, int order, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  if (c->bin_n == 0) return PM_OK;
  switch (order * 2 + (sh.shifted ? 1 : 0)) {
    case 4: return gather_os<2, false>(c, sh, a, st);
    case 5: return gather_os<2, true>(c, sh, a, st);
    case 6: return gather_os<3, false>(c, sh, a, st);
    case 7: return gather_os<3, true>(c, sh, a, st);
    case 8: return gather_os<4, false>(c, sh, a, st);
    case 9: return gather_os<4, true>(c, sh, a, st);
  }
  return fail(c, PM_EINVAL, "worder must be 2, 3 or 4");
}

}  // namespace pmf
