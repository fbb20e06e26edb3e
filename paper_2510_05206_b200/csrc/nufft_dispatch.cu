// nufft_dispatch.cu -- run-time selection of the ES-kernel width (three translation units per width:
// scatter, gather of values, grad-W gather; see build.py).
#include "pm_internal.cuh"

namespace pmf {

template <int W>
int es_scatter_w(Ctx* c, int ncomp, const float* wsrc, int wstride, float* const mesh[], cudaStream_t st);
template <int W>
int es_gather_values_w(Ctx* c, const GatherArgs& a, cudaStream_t st);
template <int W>
int es_gather_grad_w(Ctx* c, const GatherArgs& a, cudaStream_t st);

#ifdef PMF_ES_WIDTHS  // development builds with fewer widths (build.py --es-widths): -D"PMF_ES_WIDTHS(X)=X(7)"
#define ES_WIDTHS(X) PMF_ES_WIDTHS(X)
#else
#define ES_WIDTHS(X) X(4) X(5) X(6) X(7) X(8)
#endif
#define DECL(W)                                                                                    \
  template <>                                                                                      \
  int es_scatter_w<W>(Ctx*, int, const float*, int, float* const[], cudaStream_t);                 \
  template <>                                                                                      \
  int es_gather_values_w<W>(Ctx*, const GatherArgs&, cudaStream_t);                                \
  template <>                                                                                      \
  int es_gather_grad_w<W>(Ctx*, const GatherArgs&, cudaStream_t);
ES_WIDTHS(DECL)
#undef DECL

int launch_es_scatter(Ctx* c, int ncomp, const float* wsrc, int wstride, float* const mesh[], cudaStream_t st) {
  if (ncomp < 1 || ncomp > 3) return fail(c, PM_EINVAL, "ncomp must be 1..3");
  if (c->bin_n == 0) return PM_OK;
  switch (c->nufft_w) {
#define CASE(W) \
  case W: return es_scatter_w<W>(c, ncomp, wsrc, wstride, mesh, st);
    ES_WIDTHS(CASE)
#undef CASE
  }
  return fail(c, PM_EINVAL, "ES kernel width %d is not built (built: 4..8)", c->nufft_w);
}

int launch_es_gather(Ctx* c, const GatherArgs& a, cudaStream_t st) {
  if (c->bin_n == 0) return PM_OK;
  if (a.mode == GATHER_JVP) return fail(c, PM_ESTATE, "forward-mode gathers are built for the PM kernels only");
  switch (c->nufft_w) {
#define CASE(W) \
  case W: return a.mode == GATHER_GRAD ? es_gather_grad_w<W>(c, a, st) : es_gather_values_w<W>(c, a, st);
    ES_WIDTHS(CASE)
#undef CASE
  }
  return fail(c, PM_EINVAL, "ES kernel width %d is not built (built: 4..8)", c->nufft_w);
}

}  // namespace pmf
