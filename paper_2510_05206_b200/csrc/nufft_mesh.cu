// nufft_mesh.cu -- a6 / a8 / a12: spreading and interpolation with the exponential-of-semicircle kernel
// (Eq. 2.18-2.19): instantiations of k_scatter / k_gather for one
// kernel width.  Compiled once per supported width with -DES_W=<w>; nufft_dispatch.cu selects at run time.
#include "pm_mesh_kernels.cuh"

#if !defined(ES_W) || !defined(ES_PART)
#error "compile with -DES_W=<kernel width> -DES_PART=<0 scatter | 1 gather of values | 2 grad-W gather>"
#endif

namespace pmf {

template <int W>
int es_scatter_w(Ctx* c, int ncomp, const float* wsrc, int wstride, float* const mesh[], cudaStream_t st);
template <int W>
int es_gather_values_w(Ctx* c, const GatherArgs& a, cudaStream_t st);
template <int W>
int es_gather_grad_w(Ctx* c, const GatherArgs& a, cudaStream_t st);

template <class T>
static typename T::Params es_params(const Ctx* c) {
  typename T::Params tp;
  tp.frac[0] = tp.frac[1] = tp.frac[2] = 0u;
  tp.beta = (float)c->nufft_beta;
  return tp;
}

#if ES_PART == 0
template <>
int es_scatter_w<ES_W>(Ctx* c, int ncomp, const float* wsrc, int wstride, float* const mesh[], cudaStream_t st) {
  using T = ESTraits<ES_W>;
  const typename T::Params tp = es_params<T>(c);
  const int roll[3] = {0, 0, 0};
  if (!wsrc) {
    for (int a = 0; a < ncomp; ++a) PM_TRY((run_scatter<T, 1, W_UNIT>(c, tp, roll, weights_src(nullptr, 0), mesh + a, st)));
    return PM_OK;
  }
  if (ncomp == 3) return run_scatter<T, 3, W_WEIGHTED>(c, tp, roll, weights_src(wsrc, wstride), mesh, st);
  for (int a = 0; a < ncomp; ++a)
    PM_TRY((run_scatter<T, 1, W_WEIGHTED>(c, tp, roll, weights_src(wsrc + a, wstride), mesh + a, st)));
  return PM_OK;
}

#else
template <class T, int NCOMP, bool GRAD>
static int go(Ctx* c, const GatherArgs& a, cudaStream_t st) {
  constexpr size_t smem = sizeof(float) * (size_t)NCOMP * Geo<T>::COMP + 128;
  if (smem > 200 * 1024) return fail(c, PM_EINVAL, "ES gather: %d meshes of width %d do not fit in shared memory", NCOMP, T::P);
  const int roll[3] = {0, 0, 0};
  return run_gather<T, NCOMP, GRAD ? G_GRAD : G_VALUES>(c, es_params<T>(c), roll, a, st);
}

#if ES_PART == 1
template <>
int es_gather_values_w<ES_W>(Ctx* c, const GatherArgs& a, cudaStream_t st) {
  using T = ESTraits<ES_W>;
  switch (a.ncomp) {
    case 1: return go<T, 1, false>(c, a, st);
    case 2: return go<T, 2, false>(c, a, st);
    case 3: return go<T, 3, false>(c, a, st);
  }
  return fail(c, PM_EINVAL, "ES gather: unsupported ncomp = %d", a.ncomp);
}
#else
template <>
int es_gather_grad_w<ES_W>(Ctx* c, const GatherArgs& a, cudaStream_t st) {
  using T = ESTraits<ES_W>;
  switch (a.ncomp) {
    case 1: return go<T, 1, true>(c, a, st);
    case 2: return go<T, 2, true>(c, a, st);
    case 3: return go<T, 3, true>(c, a, st);
    case 4: return go<T, 4, true>(c, a, st);
  }
  return fail(c, PM_EINVAL, "ES gather: unsupported ncomp = %d", a.ncomp);
}
#endif
#endif

}  // namespace pmf
