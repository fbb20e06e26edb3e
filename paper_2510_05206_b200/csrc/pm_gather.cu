// pm_gather.cu -- a5 / a11: B-spline gather (Eq. C.2) and the grad-W gathers of the VJP rules
// (Eq. C.6, Eq. C.12): instantiations of k_gather for CIC / TSC / PCS.
// The forward-mode gathers (Eq. C.13b) are instantiated in pm_jvp.cu.
#include "pm_mesh_kernels.cuh"

namespace pmf {

int launch_gather_jvp(Ctx* c, int order, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st);  // pm_jvp.cu

template <int ORDER, bool SHIFTED>
static int gather_os(Ctx* c, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  using T = PMTraits<ORDER, SHIFTED>;
  typename T::Params tp;
  for (int k = 0; k < 3; ++k) tp.frac[k] = sh.frac[k];
  switch (a.ncomp * 2 + (a.mode == GATHER_GRAD ? 1 : 0)) {
    case 2: return run_gather<T, 1, G_VALUES>(c, tp, sh.roll, a, st);
    case 3: return run_gather<T, 1, G_GRAD>(c, tp, sh.roll, a, st);
    case 4: return run_gather<T, 2, G_VALUES>(c, tp, sh.roll, a, st);
    case 5: return run_gather<T, 2, G_GRAD>(c, tp, sh.roll, a, st);
    case 6: return run_gather<T, 3, G_VALUES>(c, tp, sh.roll, a, st);
    case 7: return run_gather<T, 3, G_GRAD>(c, tp, sh.roll, a, st);
    case 9: return run_gather<T, 4, G_GRAD>(c, tp, sh.roll, a, st);
  }
  return fail(c, PM_EINVAL, "gather: unsupported ncomp = %d", a.ncomp);
}

int launch_gather(Ctx* c, int order, const ShiftSplit& sh, const GatherArgs& a, cudaStream_t st) {
  if (c->bin_n == 0) return PM_OK;
  if (a.mode == GATHER_JVP) return launch_gather_jvp(c, order, sh, a, st);
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
