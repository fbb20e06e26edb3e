// pm_mesh_kernels.cuh -- the tile scatter (K2/K5) and tile gather (K4/K7) kernels, templated on the
// interpolation kernel ("Traits": B-splines of Table 1, or the exponential-of-semicircle kernel).
//
// One work item = one mesh tile (TX x TY x TZ cells) and at most CHUNK of its sorted particles.
//   scatter: the tile plus its halo is accumulated in shared memory with native 32-bit integer atomics
//            (sm_100a has no native fp32 shared atomic: atomicAdd(float*) on shared memory compiles to a
//            CAS loop, 2.5x slower measured).  The fixed-point scale is chosen per work item from
//            n * max|w|, so the sum can never overflow; the tile is flushed with red.global.add.v4.f32.
//   gather:  the tile plus halo of 1..4 meshes is staged in shared memory, each particle then reads its
//            P^3 nodes from there.
#pragma once
#include "pm_internal.cuh"

namespace pmf {

// ---- interpolation-kernel traits ---------------------------------------------------------------------
// axis<DERIV>(v, s0, w, dw): v = biased fixed-point coordinate (shift already subtracted); returns the
// index s0 of the first node relative to (tile origin - HLO) and the P weights W(j - u) (and d/du).

template <int ORDER, bool SHIFTED>
struct PMTraits {
  static constexpr int P = ORDER;
  static constexpr int HLO = (ORDER == 2 ? 0 : 1) + (SHIFTED ? 1 : 0);
  static constexpr int HHI = (ORDER == 2 ? 1 : 2);
  // largest value of the 3-D kernel: W(0)^3 = 1 (CIC), (3/4)^3 (TSC), (2/3)^3 (PCS)
  static constexpr float WMAX3 = ORDER == 2 ? 1.0f : (ORDER == 3 ? 0.421875f : 0.2962963f);
  struct Params {
    uint32_t frac[3];
  };
  template <bool DERIV>
  static __device__ __forceinline__ void axis(uint32_t v, const Params&, int& s0, float (&w)[P], float (&dw)[P]) {
    constexpr float INV = 1.0f / (float)REC_ONE;
    if (ORDER == 2) {  // CIC: nodes floor(u), floor(u)+1; weights 1-t, t (Table 1)
      const float t = (float)(v & REC_MASK) * INV;
      s0 = (int)(v >> REC_FRAC) - REC_BIAS + HLO;
      w[0] = 1.0f - t;
      w[1] = t;
      if (DERIV) { dw[0] = -1.0f; dw[1] = 1.0f; }  // one-sided at nodes (R12)
    } else if (ORDER == 3) {  // TSC: i0 = floor(u + 1/2), d = u - i0 in [-1/2, 1/2) (Table 1)
      const uint32_t vh = v + (REC_ONE >> 1);
      const float d = (float)((int)(vh & REC_MASK) - (int)(REC_ONE >> 1)) * INV;
      s0 = (int)(vh >> REC_FRAC) - REC_BIAS - 1 + HLO;
      const float a = 0.5f - d, b = 0.5f + d;
      w[0] = 0.5f * a * a;
      w[1] = 0.75f - d * d;
      w[2] = 0.5f * b * b;
      if (DERIV) { dw[0] = -a; dw[1] = -2.0f * d; dw[2] = b; }
    } else {  // PCS: nodes floor(u)-1 .. floor(u)+2 at distances 1+t, t, 1-t, 2-t (Table 1)
      const float t = (float)(v & REC_MASK) * INV;
      const float o = 1.0f - t;
      s0 = (int)(v >> REC_FRAC) - REC_BIAS - 1 + HLO;
      w[0] = o * o * o * (1.0f / 6.0f);
      w[1] = (4.0f - 6.0f * t * t + 3.0f * t * t * t) * (1.0f / 6.0f);
      w[2] = (4.0f - 6.0f * o * o + 3.0f * o * o * o) * (1.0f / 6.0f);
      w[3] = t * t * t * (1.0f / 6.0f);
      if (DERIV) {
        dw[0] = -0.5f * o * o;
        dw[1] = -2.0f * t + 1.5f * t * t;
        dw[2] = 2.0f * o - 1.5f * o * o;
        dw[3] = 0.5f * t * t;
      }
    }
  }
};

// Exponential-of-semicircle kernel phi(z) = exp(beta (sqrt(1 - z^2) - 1)), z = 2 (j - u)/w, nodes
// j = ceil(u - w/2) .. + w - 1 (refs [82,83]; readings R10, R13).
template <int W>
struct ESTraits {
  static constexpr int P = W;
  static constexpr bool ODD = (W & 1) != 0;
  static constexpr int HLO = ODD ? (W - 1) / 2 : W / 2 - 1;
  static constexpr int HHI = ODD ? (W + 1) / 2 : W / 2;
  static constexpr float WMAX3 = 1.0f;  // phi(0) = 1
  struct Params {
    uint32_t frac[3];  // unused (no shift), kept for a uniform interface
    float beta;
  };
  template <bool DERIV>
  static __device__ __forceinline__ void axis(uint32_t v, const Params& p, int& s0, float (&w)[P], float (&dw)[P]) {
    constexpr float INV = 1.0f / (float)REC_ONE;
    float d;  // u - (reference node)
    int ref;  // reference node (biased): nodes are ref - HLOREF .. ref - HLOREF + W - 1
    if (ODD) {
      const uint32_t vh = v + (REC_ONE >> 1);
      d = (float)((int)(vh & REC_MASK) - (int)(REC_ONE >> 1)) * INV;  // [-1/2, 1/2)
      ref = (int)(vh >> REC_FRAC);
      s0 = ref - REC_BIAS - (W - 1) / 2 + HLO;
    } else {
      d = (float)(v & REC_MASK) * INV;  // [0, 1)
      ref = (int)(v >> REC_FRAC);
      s0 = ref - REC_BIAS - (W / 2 - 1) + HLO;
    }
    constexpr int K0 = ODD ? -(W - 1) / 2 : -(W / 2 - 1);
    constexpr float TWO_W = 2.0f / (float)W;
#pragma unroll
    for (int k = 0; k < W; ++k) {
      const float z = ((float)(K0 + k) - d) * TWO_W;
      const float q = fmaxf(1.0f - z * z, 0.0f);
      const float s = sqrtf(q);
      const float phi = expf(p.beta * (s - 1.0f));
      w[k] = phi;
      // d/du phi(2 (j-u)/w) = -(2/w) phi'(z), phi'(z) = -beta z phi / sqrt(1 - z^2), 0 at |z| >= 1 (R13)
      if (DERIV) dw[k] = q > 0.0f ? TWO_W * p.beta * z * phi / s : 0.0f;
    }
  }
};

template <class T>
struct Geo {
  static constexpr int P = T::P, HLO = T::HLO, HHI = T::HHI;
  static constexpr int ZLO = (HLO + 3) / 4 * 4, ZHI = (HHI + 3) / 4 * 4;
  static constexpr int SX = TX + HLO + HHI, SY = TY + HLO + HHI, SZ = TZ + ZLO + ZHI;
  static constexpr int PLANE = SX * SY * SZ;         // smem words per component
  static constexpr int NGROUP = SX * SY * (SZ / 4);  // float4 groups per component
};

template <int N>
struct MeshPtrs {
  float* p[N];
};
template <int N>
struct CMeshPtrs {
  const float* p[N];
};

__device__ __forceinline__ int wrap(int v, int m) {
  v %= m;
  return v < 0 ? v + m : v;
}

__device__ __forceinline__ void red_add_v4(float* addr, float4 v) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z),
               "f"(v.w)
               : "memory");
}

__device__ __forceinline__ float pow2i(int e) { return __int_as_float((e + 127) << 23); }  // e in [-126, 127]

struct TileOrigin {
  int x0, y0, z0;
};
__device__ __forceinline__ TileOrigin tile_origin(uint32_t tile, const BinView& bv) {
  TileOrigin o;
  const int tz = (int)(tile % (uint32_t)bv.ntz);
  const int r = (int)(tile / (uint32_t)bv.ntz);
  o.z0 = tz * TZ;
  o.y0 = (r % bv.nty) * TY;
  o.x0 = (r / bv.nty) * TX;
  return o;
}

// Subtract the fractional shift from a record coordinate (both REC_FRAC fixed point; rec carries REC_BIAS).
__device__ __forceinline__ uint32_t apply_shift(uint32_t rec, uint32_t frac) { return rec - frac; }

// ---- K2 / K5: tile scatter ---------------------------------------------------------------------------
template <class T, int NCOMP, bool WEIGHTED>
__global__ void __launch_bounds__(BLOCK) k_scatter(BinView bv, typename T::Params tp, int3 roll,
                                                   const float* __restrict__ wsrc, int wstride,
                                                   MeshPtrs<NCOMP> mesh) {
  using G = Geo<T>;
  constexpr int P = T::P;
  extern __shared__ __align__(16) int s_acc[];
  __shared__ float s_red[(BLOCK / 32) * NCOMP];
  const int tid = threadIdx.x;
  const uint32_t nitems = *bv.nitems;
  const int m = bv.m;

  for (uint32_t it = blockIdx.x; it < nitems; it += gridDim.x) {
    const WorkItem wi = bv.items[it];
    const uint32_t n = wi.end - wi.begin;
    const TileOrigin o = tile_origin(wi.tile, bv);

    // particles of this item -> registers
    uint4 r[PPT];
    float wv[PPT][NCOMP];
    float wabs[NCOMP];
#pragma unroll
    for (int a = 0; a < NCOMP; ++a) wabs[a] = 0.0f;
#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      const uint32_t i = wi.begin + (uint32_t)(k * BLOCK + tid);
      if (i < wi.end) {
        r[k] = bv.rec[i];
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) {
          wv[k][a] = WEIGHTED ? __ldg(wsrc + (size_t)r[k].w * wstride + a) : 1.0f;
          wabs[a] += fabsf(wv[k][a]);
        }
      }
    }
    for (int j = tid; j < NCOMP * G::PLANE / 4; j += BLOCK) reinterpret_cast<int4*>(s_acc)[j] = make_int4(0, 0, 0, 0);

    // Fixed-point scale 2^sexp per component.  No node can receive more than B = WMAX3 * sum_i |w_i|
    // (WMAX3 = largest 3-D kernel value), so B * scale <= 2^30 (signed) / 2^31 (unit weights, unsigned)
    // plus n/2 of rounding never overflows 32 bits.
    float scale[NCOMP], inv_scale[NCOMP];
    if (WEIGHTED) {
#pragma unroll
      for (int a = 0; a < NCOMP; ++a) {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) wabs[a] += __shfl_xor_sync(0xffffffffu, wabs[a], d);
        if ((tid & 31) == 0) s_red[(tid >> 5) * NCOMP + a] = wabs[a];
      }
      __syncthreads();
#pragma unroll
      for (int a = 0; a < NCOMP; ++a) {
        float tot = 0.0f;
#pragma unroll
        for (int j = 0; j < BLOCK / 32; ++j) tot += s_red[j * NCOMP + a];
        const float bound = tot * (T::WMAX3 * 1.0001f);
        int e = 0;
        const float f = frexpf(bound, &e);
        const int cl = (f == 0.5f) ? e - 1 : e;  // ceil(log2(bound))
        int sexp = (bound > 0.0f && bound < 3.0e38f) ? 30 - cl : 0;
        sexp = max(-100, min(100, sexp));
        scale[a] = pow2i(sexp);
        inv_scale[a] = pow2i(-sexp);
      }
    } else {
      const float bound = (float)n * T::WMAX3;
      int e = 0;
      const float f = frexpf(bound, &e);
      const int cl = (f == 0.5f) ? e - 1 : e;
      const int sexp = min(31, 31 - cl);
#pragma unroll
      for (int a = 0; a < NCOMP; ++a) {
        scale[a] = pow2i(sexp);
        inv_scale[a] = pow2i(-sexp);
      }
      __syncthreads();
    }

#pragma unroll
    for (int k = 0; k < PPT; ++k) {
      const uint32_t i = wi.begin + (uint32_t)(k * BLOCK + tid);
      if (i < wi.end) {
        int sx, sy, sz;
        float wx[P], wy[P], wz[P], dummy[P];
        T::template axis<false>(apply_shift(r[k].x, tp.frac[0]), tp, sx, wx, dummy);
        T::template axis<false>(apply_shift(r[k].y, tp.frac[1]), tp, sy, wy, dummy);
        T::template axis<false>(apply_shift(r[k].z, tp.frac[2]), tp, sz, wz, dummy);
        sz += G::ZLO - G::HLO;
        const int base = (sx * G::SY + sy) * G::SZ + sz;
        float ws[NCOMP];
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) ws[a] = wv[k][a] * scale[a];
#pragma unroll
        for (int a = 0; a < P; ++a)
#pragma unroll
          for (int b = 0; b < P; ++b) {
            const float wxy = wx[a] * wy[b];
            const int row = base + (a * G::SY + b) * G::SZ;
#pragma unroll
            for (int c = 0; c < P; ++c) {
              const float wxyz = wxy * wz[c];
#pragma unroll
              for (int q = 0; q < NCOMP; ++q) {
                if (WEIGHTED)
                  atomicAdd(&s_acc[q * G::PLANE + row + c], __float2int_rn(ws[q] * wxyz));
                else
                  atomicAdd(reinterpret_cast<unsigned*>(&s_acc[q * G::PLANE + row + c]),
                            __float2uint_rn(ws[q] * wxyz));
              }
            }
          }
      }
    }
    __syncthreads();

    // flush: vectorised global reductions along z (red.global.add.v4.f32), empty groups skipped
    for (int j = tid; j < NCOMP * G::NGROUP; j += BLOCK) {
      const int comp = j / G::NGROUP, rr = j - comp * G::NGROUP;
      const int4 v = reinterpret_cast<const int4*>(s_acc)[comp * (G::PLANE / 4) + rr];
      if ((v.x | v.y | v.z | v.w) == 0) continue;
      const int q = rr % (G::SZ / 4), row = rr / (G::SZ / 4);
      const int sy = row % G::SY, sx = row / G::SY;
      float4 f;
      if (WEIGHTED) {
        float is = inv_scale[0];
#pragma unroll
        for (int a = 1; a < NCOMP; ++a)
          if (comp == a) is = inv_scale[a];
        f = make_float4(__int2float_rn(v.x) * is, __int2float_rn(v.y) * is, __int2float_rn(v.z) * is,
                        __int2float_rn(v.w) * is);
      } else {
        const float is = inv_scale[0];
        f = make_float4(__uint2float_rn((unsigned)v.x) * is, __uint2float_rn((unsigned)v.y) * is,
                        __uint2float_rn((unsigned)v.z) * is, __uint2float_rn((unsigned)v.w) * is);
      }
      const int gx = wrap(o.x0 - G::HLO + sx - roll.x, m), gy = wrap(o.y0 - G::HLO + sy - roll.y, m);
      const int gz = wrap(o.z0 - G::ZLO + 4 * q - roll.z, m);
      float* p = mesh.p[comp] + ((size_t)gx * m + gy) * m;
      if ((gz & 3) == 0) {
        red_add_v4(p + gz, f);
      } else {  // integer part of the shift not a multiple of 4: scalar reductions, each wrapped
        atomicAdd(p + gz, f.x);
        atomicAdd(p + wrap(gz + 1, m), f.y);
        atomicAdd(p + wrap(gz + 2, m), f.z);
        atomicAdd(p + wrap(gz + 3, m), f.w);
      }
    }
    __syncthreads();
  }
}

// ---- K4 / K7: tile gather ----------------------------------------------------------------------------
// GRAD = false: v[i*NCOMP + a] = sum_j mesh_a[j] W_j(X_i)                                    (Eq. C.2)
// GRAD = true : v[i*3 + b]     = sum_a coef_a(i) sum_j mesh_a[j] d/du_b W_j(X_i)             (Eq. C.6, C.12)
// out = alpha * v (+ out if accumulate); the caller folds 1/Delta (d/dX = (1/Delta) d/du) into alpha.
template <class T, int NCOMP, bool GRAD>
__global__ void __launch_bounds__(BLOCK) k_gather(BinView bv, typename T::Params tp, int3 roll,
                                                  CMeshPtrs<NCOMP> mesh, const float* __restrict__ cot,
                                                  int cstride, int ncot, float const_coef,
                                                  const float* __restrict__ wmul, float alpha,
                                                  int accumulate, float* __restrict__ out) {
  using G = Geo<T>;
  constexpr int P = T::P;
  extern __shared__ __align__(16) float s_val[];
  const int tid = threadIdx.x;
  const uint32_t nitems = *bv.nitems;
  const int m = bv.m;

  for (uint32_t it = blockIdx.x; it < nitems; it += gridDim.x) {
    const WorkItem wi = bv.items[it];
    const TileOrigin o = tile_origin(wi.tile, bv);

    // stage tile + halo of every component
    for (int j = tid; j < NCOMP * G::NGROUP; j += BLOCK) {
      const int comp = j / G::NGROUP, rr = j - comp * G::NGROUP;
      const int q = rr % (G::SZ / 4), row = rr / (G::SZ / 4);
      const int sy = row % G::SY, sx = row / G::SY;
      const int gx = wrap(o.x0 - G::HLO + sx - roll.x, m), gy = wrap(o.y0 - G::HLO + sy - roll.y, m);
      const int gz = wrap(o.z0 - G::ZLO + 4 * q - roll.z, m);
      const float* p = mesh.p[comp] + ((size_t)gx * m + gy) * m;
      float4 v;
      if ((gz & 3) == 0) {
        v = __ldg(reinterpret_cast<const float4*>(p + gz));
      } else {
        v = make_float4(__ldg(p + gz), __ldg(p + wrap(gz + 1, m)), __ldg(p + wrap(gz + 2, m)),
                        __ldg(p + wrap(gz + 3, m)));
      }
      reinterpret_cast<float4*>(s_val)[comp * (G::PLANE / 4) + rr] = v;
    }
    __syncthreads();

    for (uint32_t i = wi.begin + tid; i < wi.end; i += BLOCK) {
      const uint4 r = bv.rec[i];
      int sx, sy, sz;
      float wx[P], wy[P], wz[P], dx[P], dy[P], dz[P];
      T::template axis<GRAD>(apply_shift(r.x, tp.frac[0]), tp, sx, wx, dx);
      T::template axis<GRAD>(apply_shift(r.y, tp.frac[1]), tp, sy, wy, dy);
      T::template axis<GRAD>(apply_shift(r.z, tp.frac[2]), tp, sz, wz, dz);
      sz += G::ZLO - G::HLO;
      const int base = (sx * G::SY + sy) * G::SZ + sz;
      if (!GRAD) {
        float acc[NCOMP];
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) acc[a] = 0.0f;
#pragma unroll
        for (int a = 0; a < P; ++a)
#pragma unroll
          for (int b = 0; b < P; ++b) {
            const float wxy = wx[a] * wy[b];
            const int row = base + (a * G::SY + b) * G::SZ;
#pragma unroll
            for (int c = 0; c < P; ++c) {
              const float wxyz = wxy * wz[c];
#pragma unroll
              for (int q = 0; q < NCOMP; ++q) acc[q] = fmaf(wxyz, s_val[q * G::PLANE + row + c], acc[q]);
            }
          }
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) {
          float* dst = out + (size_t)r.w * NCOMP + a;
          *dst = accumulate ? fmaf(alpha, acc[a], *dst) : alpha * acc[a];
        }
      } else {
        float coef[NCOMP];
        const float cc = const_coef * (wmul ? __ldg(wmul + r.w) : 1.0f);
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) coef[a] = a < ncot ? __ldg(cot + (size_t)r.w * cstride + a) : cc;
        float gx = 0.0f, gy = 0.0f, gz = 0.0f;
#pragma unroll
        for (int a = 0; a < P; ++a)
#pragma unroll
          for (int b = 0; b < P; ++b) {
            const int row = base + (a * G::SY + b) * G::SZ;
            const float wdx = dx[a] * wy[b], wdy = wx[a] * dy[b], wxy = wx[a] * wy[b];
#pragma unroll
            for (int c = 0; c < P; ++c) {
              float val = 0.0f;
#pragma unroll
              for (int q = 0; q < NCOMP; ++q) val = fmaf(coef[q], s_val[q * G::PLANE + row + c], val);
              gx = fmaf(wdx * wz[c], val, gx);
              gy = fmaf(wdy * wz[c], val, gy);
              gz = fmaf(wxy * dz[c], val, gz);
            }
          }
        float* dst = out + (size_t)r.w * 3;
        dst[0] = accumulate ? fmaf(alpha, gx, dst[0]) : alpha * gx;
        dst[1] = accumulate ? fmaf(alpha, gy, dst[1]) : alpha * gy;
        dst[2] = accumulate ? fmaf(alpha, gz, dst[2]) : alpha * gz;
      }
    }
    __syncthreads();
  }
}

// ---- host-side launch helpers ------------------------------------------------------------------------
inline int mesh_grid(const Ctx* c) {
  int64_t bound = (int64_t)c->ntiles + c->bin_n / CHUNK + 1;
  int64_t cap = (int64_t)c->num_sms * 8;
  return (int)(bound < cap ? bound : cap);
}

template <class T, int NCOMP, bool WEIGHTED>
int run_scatter(Ctx* c, const typename T::Params& tp, const int roll[3], const float* wsrc, int wstride,
                float* const mesh[], cudaStream_t st) {
  using G = Geo<T>;
  const size_t smem = sizeof(int) * (size_t)NCOMP * G::PLANE;
  auto kern = k_scatter<T, NCOMP, WEIGHTED>;
  static bool attr_done = false;
  if (!attr_done) {
    PM_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_done = true;
  }
  MeshPtrs<NCOMP> mp;
  for (int a = 0; a < NCOMP; ++a) mp.p[a] = mesh[a];
  kern<<<mesh_grid(c), BLOCK, smem, st>>>(bin_view(c), tp, make_int3(roll[0], roll[1], roll[2]), wsrc, wstride, mp);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

template <class T, int NCOMP, bool GRAD>
int run_gather(Ctx* c, const typename T::Params& tp, const int roll[3], const float* const mesh[],
               const float* cot, int cstride, int ncot, float const_coef, const float* wmul, float alpha,
               bool accumulate, float* out, cudaStream_t st) {
  using G = Geo<T>;
  const size_t smem = sizeof(float) * (size_t)NCOMP * G::PLANE;
  auto kern = k_gather<T, NCOMP, GRAD>;
  static bool attr_done = false;
  if (!attr_done) {
    PM_CUDA(c, cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    attr_done = true;
  }
  CMeshPtrs<NCOMP> mp;
  for (int a = 0; a < NCOMP; ++a) mp.p[a] = mesh[a];
  const float a_eff = GRAD ? (float)((double)alpha * (double)c->mg / c->p.box) : alpha;
  kern<<<mesh_grid(c), BLOCK, smem, st>>>(bin_view(c), tp, make_int3(roll[0], roll[1], roll[2]), mp, cot, cstride,
                                          ncot, const_coef, wmul, a_eff, accumulate ? 1 : 0, out);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
