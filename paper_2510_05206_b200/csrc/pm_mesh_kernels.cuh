// pm_mesh_kernels.cuh -- the tile scatter (K2/K5) and tile gather (K4/K7) kernels, templated on the
// interpolation kernel ("Traits": B-splines of Table 1, or the exponential-of-semicircle kernel).
//
// One work item = one mesh tile (TX x TY x TZ cells) and at most ITEM_MAX of its sorted particles.
//   scatter: the tile plus its halo is accumulated in shared memory with native 32-bit integer atomics
//            (sm_100a has no native fp32 shared atomic: atomicAdd(float*) on shared memory compiles to a
//            CAS loop, 2.5x slower measured).  The fixed-point scale is chosen per work item from
//            n * max|w|, so the sum can never overflow; the tile is flushed with red.global.add.v4.f32.
//   gather:  the tile plus halo of 1..4 meshes is staged in shared memory, each particle then reads its
//            P^3 nodes from there.
#pragma once
#include <cuda.h>

#include "pm_internal.cuh"

namespace pmf {

// ---- interpolation-kernel traits ---------------------------------------------------------------------
// axis<DERIV>(v, s0, w, dw): v = biased fixed-point coordinate (shift already subtracted); returns the
// index s0 of the first node relative to (tile origin - HLO) and the P weights W(j - u) (and d/du).

template <int ORDER, bool SHIFTED>
struct PMTraits {
  static constexpr int P = ORDER;
  static constexpr bool SHIFT = SHIFTED;  // a fractional grid shift is subtracted from the record coordinate
  static constexpr bool SKEW = false;     // see ESTraits
  static constexpr bool ES = false;
  static constexpr int HLO = (ORDER == 2 ? 0 : 1) + (SHIFTED ? 1 : 0);
  static constexpr int HHI = (ORDER == 2 ? 1 : 2);
  // largest value of the 3-D kernel: W(0)^3 = 1 (CIC), (3/4)^3 (TSC), (2/3)^3 (PCS)
  static constexpr float WMAX3 = ORDER == 2 ? 1.0f : (ORDER == 3 ? 0.421875f : 0.2962963f);
  // largest value of |dW/du| W W: 1 (CIC), 1 * (3/4)^2 (TSC), (2/3)^3 (PCS: max|W'| = 2/3 at |x| = 2/3)
  static constexpr float DWMAX3 = ORDER == 2 ? 1.0f : (ORDER == 3 ? 0.5625f : 0.2962963f);
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

// Launch shape of the ES (NUFFT) spreading / interpolation kernels.  The stencil walk of ONE particle is w^3 = 64 .. 512
// nodes, fully unrolled: a thread holds ONE record at a time (eight / four unrolled copies of the walk were 290 KB of
// code -- instruction-fetch stalls -- and 252 registers: one CTA of 8 warps per SM, ncu round 2) and the register
// allocation aims at three resident CTAs.  cfg3 (w = 7): spread 34.4 -> 20.1 ms with these two alone.
constexpr int ES_PPT = 1;     // records per thread and batch, k_scatter
constexpr int ES_KB = 1;      // records in flight per thread, k_gather
constexpr int ES_MINCTA = 3;  // resident CTAs per SM the single-field ES scatter is compiled for
// Widths whose kernels use the skewed walk over dense rows (skew_match below).  Measured on cfg3 (spread / interp, ms):
// w = 8: 21.7 / 59.5 against 29.9 / 78.4 without; w = 7: 18.3 / 37.8 against 20.1 / 53.7; w = 6: 14.4 / 29.9 against
// 13.5 / 35.3; w = 5 (8 steps for 5 columns): 8.7 / 17.1 against 6.2 / 15.1 -- not used below 6.
constexpr bool es_skew_width(int w) { return w >= 6; }
// Float -> fixed point without the conversion unit (unit-weight ES spreading).  F2I shares the quarter-rate pipe with
// the kernel's exp / sqrt; one F2I per node kept it 67 % busy (ncu round 2).  Instead the deposit x < 2^24 is computed as
// the DENORMAL float x * 2^-149, whose bit pattern IS the integer round-to-nearest-even(x) (the lowest binade of the
// normal numbers continues the same integer scale).  The factor is split between the z weights (2^-64) and the x weights
// (2^-85) so that every operand stays a normal number and only the final product rounds to the integer grid.  Denormal
// arithmetic runs at full rate in the FMA pipe; the build must not flush them (no -ftz / --use_fast_math).
constexpr float ES_DENORM_Z = 5.421010862427522e-20f;   // 2^-64
constexpr float ES_DENORM_X = 2.5849394142282115e-26f;  // 2^-85

// Exponential-of-semicircle kernel phi(z) = exp(beta (sqrt(1 - z^2) - 1)), z = 2 (j - u)/w, nodes
// j = ceil(u - w/2) .. + w - 1 (refs [82,83]; readings R10, R13).
template <int W>
struct ESTraits {
  static constexpr int P = W;
  static constexpr bool SHIFT = false;
  static constexpr bool ODD = (W & 1) != 0;
  static constexpr int HLO = ODD ? (W - 1) / 2 : W / 2 - 1;
  static constexpr int HHI = ODD ? (W + 1) / 2 : W / 2;
  static constexpr float WMAX3 = 1.0f;  // phi(0) = 1
  static constexpr float DWMAX3 = 1.0f; // (forward-mode scatter is not instantiated for the ES kernel)
  struct Params {
    uint32_t frac[3];  // unused (no shift), kept for a uniform interface
    float beta;
  };
  static constexpr int K0 = ODD ? -(W - 1) / 2 : -(W / 2 - 1);  // first node of the stencil relative to the reference node
  // first node s0 (relative to tile origin - HLO) and d = u - (reference node) of a record coordinate
  static __device__ __forceinline__ void origin(uint32_t v, int& s0, float& d) {
    constexpr float INV = 1.0f / (float)REC_ONE;
    if (ODD) {
      const uint32_t vh = v + (REC_ONE >> 1);
      d = (float)((int)(vh & REC_MASK) - (int)(REC_ONE >> 1)) * INV;  // [-1/2, 1/2)
      s0 = (int)(vh >> REC_FRAC) - REC_BIAS - (W - 1) / 2 + HLO;
    } else {
      d = (float)(v & REC_MASK) * INV;  // [0, 1)
      s0 = (int)(v >> REC_FRAC) - REC_BIAS - (W / 2 - 1) + HLO;
    }
  }
  // kernel value (and d/du) at stencil node k (kf = K0 + k as a float; k may be a run-time value)
  template <bool DERIV>
  static __device__ __forceinline__ void node_weight(float kf, float d, const Params& p, float& w, float& dw) {
    constexpr float TWO_W = 2.0f / (float)W;
    const float z = (kf - d) * TWO_W;
    const float q = fmaxf(1.0f - z * z, 0.0f);
    const float s = sqrtf(q);
    const float phi = expf(p.beta * (s - 1.0f));
    w = phi;
    // d/du phi(2 (j-u)/w) = -(2/w) phi'(z), phi'(z) = -beta z phi / sqrt(1 - z^2), 0 at |z| >= 1 (R13)
    if (DERIV) dw = q > 0.0f ? TWO_W * p.beta * z * phi / s : 0.0f;
  }
  template <bool DERIV>
  static __device__ __forceinline__ void axis(uint32_t v, const Params& p, int& s0, float (&w)[P], float (&dw)[P]) {
    float d;
    origin(v, s0, d);
#pragma unroll
    for (int k = 0; k < W; ++k) node_weight<DERIV>((float)(K0 + k), d, p, w[k], dw[k]);
  }
  // Skewed stencil walk (skew_match below): the z loop has ZS = 8 steps per (x, y) row; step j of a lane whose walk
  // is rotated by rot visits column (j + rot) of the row -- columns 8 .. 14 are columns 0 .. 6 of the NEXT row of the
  // walk.  wU / wW: the z weight of step j if it falls into the current / the next row (the other one is 0); columns
  // W .. 7 carry weight 0 (the walk passes over them so that every step advances the bank by one).
  static constexpr bool SKEW = es_skew_width(W);
  static constexpr bool ES = true;
  static constexpr int ZS = 8;
  template <bool DERIV>
  static __device__ __forceinline__ void axis_skew(float d, const Params& p, int rot, float (&wU)[ZS], float (&wW)[ZS],
                                                   float (&dU)[ZS], float (&dW)[ZS]) {
#pragma unroll
    for (int j = 0; j < ZS; ++j) {
      const int n = j + rot, c = n & (ZS - 1);
      float w, dw = 0.0f;
      node_weight<DERIV>((float)(K0 + c), d, p, w, dw);
      if (c >= W) w = 0.0f, dw = 0.0f;
      const bool nextrow = n >= ZS;
      wU[j] = nextrow ? 0.0f : w;
      wW[j] = nextrow ? w : 0.0f;
      if (DERIV) {
        dU[j] = nextrow ? 0.0f : dw;
        dW[j] = nextrow ? dw : 0.0f;
      }
    }
  }
};

// Shared-memory tile geometry.  A staged tile covers nodes [x0 - HLO, x0 + TX + HHI) x [y0 - HLO, ...) and, along
// z, [z0 - ZLO, z0 - ZLO + TZ + HZ) with ZLO = HLO rounded up to 4 (16-byte vector reductions, and a TMA box
// must start on a 16-byte boundary of the innermost dimension: an unaligned start coordinate raises "illegal
// instruction" on sm_100a).  Each (x, y) row is stored in two pieces: the first TZ = 32 nodes in the MAIN plane
// with a row pitch of exactly 32 words, the remaining HZ (4 or 8) in the HALO plane.  With a pitch of 32 the
// bank of a main-plane node is its z index alone, so a warp whose 32 lanes hold particles at 32 different z
// (one lattice row in Lagrangian order) is conflict-free whatever their (x, y) cells are; a dense pitch of
// TZ + halo made every access a 2-way conflict (ncu: 51 % of the shared wavefronts).
template <class T>
struct Geo {
  static constexpr int P = T::P, HLO = T::HLO, HHI = T::HHI;
  static constexpr int ZLO = (HLO + 3) / 4 * 4;
  static constexpr int HZ = ZLO + (HHI + 3) / 4 * 4;                 // halo columns per row
  // DENSE (skewed walk, ES kernels): one piece per (x, y) row, pitch TZ + HZ = 40 words.  With the 8-step z loop of
  // the skewed walk a step to the next column (+1), to the next row (+40 - 7) and to the next x slab
  // ((SY - (W - 1)) * 40 - 7 = 353 words: SY - (W - 1) = 9, even widths pad SY by one row for it) all advance the bank
  // by exactly one.
  static constexpr bool DENSE = T::SKEW;
  static constexpr int PITCH = TZ + HZ;
  static constexpr int SX = TX + HLO + HHI, SY = TY + HLO + HHI + ((DENSE && P % 2 == 0) ? 1 : 0), NROW = SX * SY;
  static constexpr int MAIN = NROW * TZ, HAL = NROW * HZ;            // words per component
  // component block (128-byte multiple); DENSE: at least 8 words of slack behind the last row -- the zero-weight
  // columns of the skewed walk (up to column 41 of a row) touch them
  static constexpr int COMP = (MAIN + HAL + (T::SKEW ? 8 : 0) + 31) / 32 * 32;
  static constexpr int NGM = NROW * (TZ / 4), NGH = NROW * (HZ / 4); // float4 groups per component
  static constexpr int NGROUP = NGM + NGH;
  static_assert(TZ == 32, "the main plane's row pitch must be 32 words");
  static_assert(HZ == 4 || HZ == 8, "halo columns");
  static_assert(!DENSE || (HZ == 8 && SY - (P - 1) == 9), "the skewed walk needs rows of 40 words and a slab step of 9 rows");
};

// Address of node column s (0 <= s < TZ + HZ, relative to the box start) in row `row` of a component block:
//   s < TZ : MAIN[row * TZ + s]        else : HAL[row * HZ + s - TZ]
// NodeCol holds the per-column part; the row part is one multiply-add (row * pitch + base).
struct NodeCol {
  int base, pitch;
};
template <class G>
__device__ __forceinline__ NodeCol node_col(int row0, int s) {  // row0 = index of the particle's first row
  NodeCol c;
  if constexpr (G::DENSE) {
    c.pitch = G::PITCH;
    c.base = row0 * G::PITCH + s;
  } else {
    const bool main = s < TZ;
    c.pitch = main ? TZ : G::HZ;
    c.base = main ? row0 * TZ + s : G::MAIN + row0 * G::HZ + (s - TZ);
  }
  return c;
}
// float4 group j of a component block -> (row, z offset of its first node relative to the box start)
template <class G>
__device__ __forceinline__ void group_pos(int j, int& row, int& zoff) {
  if constexpr (G::DENSE) {
    row = j / (G::PITCH / 4);
    zoff = 4 * (j - row * (G::PITCH / 4));
  } else if (j < G::NGM) {
    row = j / (TZ / 4);
    zoff = 4 * (j - row * (TZ / 4));
  } else {
    const int h = j - G::NGM;
    row = h / (G::HZ / 4);
    zoff = TZ + 4 * (h - row * (G::HZ / 4));
  }
}

template <int N>
struct MeshPtrs {
  float* p[N];
};
template <int N>
struct CMeshPtrs {
  const float* p[N];
};
template <int N>
struct TMapSet {
  CUtensorMap m[N];
};

__device__ __forceinline__ void red_add_v4(float* addr, float4 v) {
  asm volatile("red.global.add.v4.f32 [%0], {%1, %2, %3, %4};" ::"l"(addr), "f"(v.x), "f"(v.y), "f"(v.z),
               "f"(v.w)
               : "memory");
}

__device__ __forceinline__ float pow2i(int e) { return __int_as_float((e + 127) << 23); }  // e in [-126, 127]

struct TileOrigin {
  int x0, y0, z0;
};
__device__ __forceinline__ TileOrigin tile_origin(const WorkItem& wi) {  // k_items packed the tile coordinates
  TileOrigin o;
  o.x0 = (int)(wi.txyz & 1023u) * TX;
  o.y0 = (int)((wi.txyz >> 10) & 1023u) * TY;
  o.z0 = (int)(wi.txyz >> 20) * TZ;
  return o;
}
__device__ __forceinline__ int wrap_lo(int v, int m) {                               // v in [-2m, m)
  v += v < 0 ? m : 0;
  v += v < 0 ? m : 0;
  return v;
}
__device__ __forceinline__ int wrap_hi(int v, int m) {                               // v in [0, 3m)
  v -= v >= m ? m : 0;
  v -= v >= m ? m : 0;
  return v;
}

// Subtract the fractional shift from a record coordinate (both REC_FRAC fixed point; rec carries REC_BIAS).
template <class T>
__device__ __forceinline__ uint32_t apply_shift(uint32_t rec, uint32_t frac) {
  return T::SHIFT ? rec - frac : rec;
}

// Dynamic tile schedule of the persistent scatter / gather kernels.  A CTA starts with item blockIdx.x and
// then draws item ids from a global counter, so the items in flight are always a compact window of
// consecutive tiles: the halo planes two neighbouring tiles share are touched close together in time and
// are served from L2.  (A static stride lets CTAs drift apart: ncu showed the TMA halo reads of the gather
// all going to DRAM.)  The last CTA to finish zeroes both counters for the next launch on the stream.
// The counter is bumped with a raw atom.global.add: nvcc turns atomicAdd() under a lane-dependent branch into
// a warp-aggregated sequence whose broadcast SHFL consumes the result AT ONCE, which exposes the contended
// counter's whole round trip once per item (ncu: 18-20 % of the scatter's stall samples on that SHFL).  With the
// raw instruction the result is first touched where the caller reads it, one work item later.
__device__ __forceinline__ uint32_t atom_inc_raw(uint32_t* p) {
  uint32_t r;
  asm volatile("atom.global.add.u32 %0, [%1], 1;" : "=r"(r) : "l"(p) : "memory");
  return r;
}
// ptxas ALSO aggregates the raw add when it can prove the address warp-uniform (VOTEU / POPC / ATOMG.ADD / SHFL.IDX:
// ncu round 2 showed 9 % of the warp-private scatter's stall samples on that SHFL, once per work item).  The wrapping
// increment atom.inc has no popcount form, so it stays a plain per-thread ATOMG whose result is first touched where
// the caller reads it (the bound 2^31 - 1 is never reached: the counter counts work items; with the bound 2^32 - 1 ptxas turns inc back into add).
__device__ __forceinline__ uint32_t atom_inc_noagg(uint32_t* p) {
  uint32_t r;
  asm volatile("atom.global.inc.u32 %0, [%1], 2147483647;" : "=r"(r) : "l"(p) : "memory");
  return r;
}
__device__ __forceinline__ uint32_t sched_next(uint32_t* sched) { return gridDim.x + atom_inc_noagg(&sched[0]); }
__device__ __forceinline__ void sched_done(uint32_t* sched) {
  if (atomicAdd(&sched[1], 1u) == gridDim.x - 1u) {
    sched[0] = 0u;
    sched[1] = 0u;
  }
}

// record loads: read once per kernel -> streaming (evict-first) so they do not push mesh tiles out of L2
template <bool IDX>  // IDX: the caller reads the original index (.w)
__device__ __forceinline__ void load_rec(uint4& r, const BinView& bv, uint32_t i) {
  r = __ldcs(bv.rec + i);
}
__device__ __forceinline__ uint32_t rec_index(const BinView& bv, uint32_t i) { return bv.rec[i].w; }

// ---- skewed stencil walk of the ES kernels ---------------------------------------------------------------------
// One thread walks the W x W x W nodes of its particle; the 32 lanes of a warp sit at unrelated z, so a shared-memory
// access of the warp hits a bank 3.5 times on average (32 balls into 32 bins: measured 3.8-way replays, the NUFFT
// kernels ran at 0.21 / 0.43 of the conflict-free ceilings).  In the DENSE tile layout the walk x slab -> y row -> 8 z
// columns advances the bank by exactly one per step for every lane, so the warp is conflict-free for the whole walk
// iff the lanes START in 32 different banks.  Lane l may start rot_l in [0, 8) columns into its first row (the skipped
// columns are visited at the end of the walk): skew_match picks the rotations so that the starting banks
// (B_l + rot_l) mod 32 are distinct wherever a matching exists.  All intervals [B_l, B_l + 8) have the same length, so
// handing out the banks in the order of B_l -- each lane the first free bank at or after its own -- is optimal on a
// line; the circle is cut behind the bank v that minimises D_v = #{l : B_l <= v} - (v + 1), from where the sorted
// assignment never wraps.  In closed form, with E_v the number of lanes in banks before v (in cut order) and o the
// rank of a lane among those of its bank:  slot = E + o + max_{u <= v, occupied} (u - E_u).  A lane whose slot lies 8
// or more behind its bank finds no free bank (0.5 lanes per warp for uniformly random B) and takes any rotation.
// Call with all 32 lanes; `valid` lanes take part.  Returns rot in [0, 8).
__device__ __forceinline__ int skew_match(int B, bool valid) {
  constexpr unsigned FULL = 0xffffffffu;
  const int v = (int)(threadIdx.x & 31u);
  unsigned mine = __ballot_sync(FULL, valid);  // -> valid lanes whose bank is v
#pragma unroll
  for (int k = 0; k < 5; ++k) {
    const unsigned bk = __ballot_sync(FULL, (B >> k) & 1);
    mine &= ((v >> k) & 1) ? bk : ~bk;
  }
  const int c = __popc(mine);
  const unsigned peers = __shfl_sync(FULL, mine, B);
  const int o = __popc(peers & ((1u << v) - 1u));
  int S = c;  // inclusive prefix over the banks
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int t = __shfl_up_sync(FULL, S, d);
    if (v >= d) S += t;
  }
  const int total = __shfl_sync(FULL, S, 31);
  int key = ((S - (v + 1) + 64) << 5) | v;  // first minimum of D
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) key = min(key, __shfl_xor_sync(FULL, key, d));
  const int vmin = key & 31;
  const int Smin = (key >> 5) - 64 + vmin + 1;
  const int cut = (vmin + 1) & 31;
  const int vp = (v - cut) & 31;
  const int Sr = cut == 0 ? S : (v >= cut ? S - Smin : S + total - Smin);
  const int E = Sr - c;
  const int term = c > 0 ? vp - E : -1000;
  int M = __shfl_sync(FULL, term, (v + cut) & 31);  // lane i: the term of the bank with cut-order index i
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int t = __shfl_up_sync(FULL, M, d);
    if (v >= d) M = max(M, t);
  }
  const int Bp = (B - cut) & 31;
  const int rot = __shfl_sync(FULL, E, B) + o + __shfl_sync(FULL, M, Bp) - Bp;
  return rot & 7;
}

// address step from column 8 + c of row (a, b) of the walk to column c of the row that follows it: (a, b + 1), the first
// row of the next slab, or (after the last row) the first row of the walk
template <class G>
__host__ __device__ constexpr int skew_next_off(int a, int b) {
  return b < G::P - 1 ? G::PITCH - 8
                      : (a < G::P - 1 ? (G::SY - (G::P - 1)) * G::PITCH - 8
                                      : -((G::P - 1) * G::SY + (G::P - 1)) * G::PITCH - 8);
}

// ---- K2 / K5: tile scatter ---------------------------------------------------------------------------
// Persistent CTAs draw work items from the dynamic schedule, two items ahead: while item i is deposited, the
// records of item i+1 are already being loaded into the registers item i frees (rolling prefetch), and its
// WorkItem was fetched during the flush of item i-1.  The accumulator tile is zeroed once; every flush writes
// zeros back.  With NBUF = 2 accumulator tiles the flush of item i and the deposit of item i+1 use different
// buffers, so a work item costs ONE barrier (ncu before: barrier 33 %, long scoreboard 28 % of the stall
// cycles with two barriers and loads issued after the deposit).  roll is in [0, m).
// resident CTAs per SM the register allocation aims at (the unit-weight CIC assign is the headline kernel)
// What a particle deposits.  W_UNIT: W_j(X_i).  W_WEIGHTED: w_i^a W_j(X_i), a < NCOMP (Eq. C.1, C.10).
// W_JVP (NCOMP = 1): the tangent of the scatter, Eq. C.13a: w~_i W_j(X_i) + w_i X~_i . dW_j(X_i)/dX_i.
enum { W_UNIT = 0, W_WEIGHTED = 1, W_JVP = 2 };
struct ScatterSrc {
  const float* w;        // W_WEIGHTED: [N * wstride], component a at w[i*wstride + a]; W_JVP: [N] or NULL (ones)
  int wstride;
  const float* w_tan;    // W_JVP: [N] or NULL
  const float* pos_tan;  // W_JVP: [N,3] or NULL
  float tan_scale;       // W_JVP: 1/Delta (d/dX = (1/Delta) d/du)
};
template <class T, int NCOMP, int WMODE>
constexpr int scatter_min_ctas() {
  // vector scatter of the VJP (3 components): at 151 registers ONE CTA was resident per SM (ncu: 12.5 % warps
  // active, 3.5 ms at 512^3); two CTAs for CIC / TSC cap the allocation at 128
  return WMODE == W_JVP ? 1
                        : (NCOMP == 1 && WMODE == W_UNIT) ? (T::P == 2 ? 4 : (T::P <= 4 ? 3 : (T::ES ? ES_MINCTA : 1)))
                                                          : (NCOMP == 1 ? (T::ES ? ES_MINCTA : 2)
                                                                        : ((T::P <= 3 || T::ES) ? 2 : 1));
}
template <class T, int NCOMP, int WMODE, int NBUF>
__global__ void __launch_bounds__(BLOCK, scatter_min_ctas<T, NCOMP, WMODE>()) k_scatter(BinView bv, typename T::Params tp, int3 roll,
                                                   ScatterSrc src, MeshPtrs<NCOMP> mesh) {
  constexpr bool WEIGHTED = WMODE != W_UNIT;
  constexpr int PPT_ = T::ES ? ES_PPT : PPT;  // records per thread held in registers at a time
  constexpr int CHUNK_ = BLOCK * PPT_;
  constexpr bool JVP = WMODE == W_JVP;
  constexpr int NPAY = JVP ? 4 : NCOMP;  // floats a particle carries: its weights, or {w~, w t_x, w t_y, w t_z}
  static_assert(!JVP || NCOMP == 1, "the forward-mode scatter deposits one field");
  const float* __restrict__ wsrc = src.w;
  const int wstride = src.wstride;
  using G = Geo<T>;
  constexpr int P = T::P;
  constexpr int NG = NCOMP * G::NGROUP;                          // groups to flush
  constexpr int NSLOT = (NG + BLOCK - 1) / BLOCK;                // groups per thread
  constexpr bool PRE = NSLOT <= 6;                               // group coordinates kept in registers
  constexpr int ACC = NCOMP * G::COMP;                           // words per accumulator buffer
  extern __shared__ __align__(16) int s_acc_all[];
  __shared__ float s_red[(BLOCK / 32) * NCOMP];
  __shared__ uint32_t s_next[2];
  const int tid = threadIdx.x;
  const uint32_t nitems = *bv.nitems;
  const int m = bv.m;

  for (int j = tid; j < NBUF * ACC / 4; j += BLOCK) reinterpret_cast<int4*>(s_acc_all)[j] = make_int4(0, 0, 0, 0);
  if (tid == 0) s_next[0] = sched_next(bv.sched);  // the item after this CTA's first

  // (comp, sx, sy, z offset) of the groups this thread flushes, packed 4 | 8 | 8 | 12 bits
  auto group_coords = [](int j) -> uint32_t {
    const int comp = j / G::NGROUP;
    int row, zoff;
    group_pos<G>(j - comp * G::NGROUP, row, zoff);
    const int sx = row / G::SY, sy = row - sx * G::SY;
    return (uint32_t)zoff | ((uint32_t)sy << 12) | ((uint32_t)sx << 20) | ((uint32_t)comp << 28);
  };
  uint32_t gc[PRE ? NSLOT : 1];
  if (PRE) {
#pragma unroll
    for (int k = 0; k < NSLOT; ++k) gc[k] = group_coords(min(tid + k * BLOCK, NG - 1));
  }
  __syncthreads();

  // records of a work item -> registers
  WorkItem wi, nwi;
  wi.begin = wi.end = wi.txyz = nwi.begin = nwi.end = nwi.txyz = 0;
  uint4 r[PPT_];
  auto load_batch = [&](uint32_t b0, uint32_t end) {  // up to CHUNK_ records starting at b0
#pragma unroll
    for (int k = 0; k < PPT_; ++k) {
      const uint32_t i = b0 + (uint32_t)(k * BLOCK + tid);
      if (i < end) load_rec<WEIGHTED>(r[k], bv, i);
    }
  };
  uint32_t it = blockIdx.x, nxt = s_next[0];
  int par = 1;
  int* s_acc = s_acc_all;
  if (it < nitems) {
    wi = bv.items[it];
    load_batch(wi.begin, wi.end);
  }
  if (nxt < nitems) nwi = bv.items[nxt];
  while (it < nitems) {
    // item i+2: the atomic is issued now and its result is only touched right before the barrier below (stored
    // at once, thread 0 would wait ~microseconds for the contended counter with the whole CTA behind it)
    uint32_t fetched = 0;
    if (tid == 0) fetched = atom_inc_noagg(&bv.sched[0]);  // raw: gridDim.x is added where it is stored
    const uint32_t n = wi.end - wi.begin;
    const uint32_t ibegin = wi.begin, iend = wi.end;
    const TileOrigin o = tile_origin(wi);
    const uint32_t nbegin = nwi.begin, nend = nxt < nitems ? nwi.end : nwi.begin;  // empty when there is no next item

    float wv[PPT_][NPAY];
    float wabs[NCOMP];
#pragma unroll
    for (int a = 0; a < NCOMP; ++a) wabs[a] = 0.0f;
    // what particle `idx` (caller order) deposits, and its contribution to the bound of the node sums
    auto payload = [&](uint32_t idx, float (&pv)[NPAY]) {
      if constexpr (JVP) {
        const float w = wsrc ? __ldg(wsrc + idx) : 1.0f;
        pv[0] = src.w_tan ? __ldg(src.w_tan + idx) : 0.0f;
        float t0 = 0.0f, t1 = 0.0f, t2 = 0.0f;
        if (src.pos_tan) {
          const float* t = src.pos_tan + (size_t)idx * 3;
          t0 = __ldg(t), t1 = __ldg(t + 1), t2 = __ldg(t + 2);
        }
        const float ws = w * src.tan_scale;
        pv[1] = ws * t0, pv[2] = ws * t1, pv[3] = ws * t2;
        // largest deposit of a particle: |w~| W_max^3 + |w t|_1 max|dW/du| W_max^2 (Table 1: CIC 1, TSC 9/16, PCS 8/27)
        wabs[0] += fabsf(pv[0]) * T::WMAX3 + (fabsf(pv[1]) + fabsf(pv[2]) + fabsf(pv[3])) * T::DWMAX3;
      } else {
#pragma unroll
        for (int a = 0; a < NCOMP; ++a) {
          pv[a] = WEIGHTED ? __ldg(wsrc + (size_t)idx * wstride + a) : 1.0f;
          wabs[a] += fabsf(pv[a]);
        }
      }
    };
    auto load_weights = [&](uint32_t b0) {  // payloads of the batch held in r[]
#pragma unroll
      for (int k = 0; k < PPT_; ++k) {
        const uint32_t i = b0 + (uint32_t)(k * BLOCK + tid);
        if (i < iend) payload(r[k].w, wv[k]);
      }
    };
    load_weights(ibegin);
    if (WEIGHTED && n > (uint32_t)CHUNK_) {  // dense tile: the bound needs the weights of the later batches too
      for (uint32_t i = ibegin + CHUNK_ + tid; i < iend; i += BLOCK) {
        float pv[NPAY];
        payload(rec_index(bv, i), pv);
      }
    }

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
        const float bound = tot * ((JVP ? 1.0f : T::WMAX3) * 1.0001f);
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
      // ES kernels convert without F2I (es_bits below), which needs every single deposit below 2^24
      const int sexp = min(T::ES ? 22 : 31, 31 - cl);
#pragma unroll
      for (int a = 0; a < NCOMP; ++a) {
        scale[a] = pow2i(sexp);
        inv_scale[a] = pow2i(-sexp);
      }
    }

    for (uint32_t b0 = ibegin;;) {
      const bool last = b0 + CHUNK_ >= iend;  // uniform
#pragma unroll
      for (int k = 0; k < PPT_; ++k) {
        const uint32_t i = b0 + (uint32_t)(k * BLOCK + tid);
        if constexpr (T::SKEW) {  // ES kernels: skewed walk over dense rows (skew_match)
          static_assert(!JVP, "the forward-mode scatter is not built for the ES kernel");
          const bool valid = i < iend;
          int sx = 0, sy = 0, sz = 0;
          float wx[P], wy[P], dummy[P], dz0 = 0.0f;
          if (valid) {
            T::template axis<false>(r[k].x, tp, sx, wx, dummy);
            T::template axis<false>(r[k].y, tp, sy, wy, dummy);
            T::origin(r[k].z, sz, dz0);
          }
          const int row0 = sx * G::SY + sy, col0 = sz + (G::ZLO - G::HLO);
          // (warp-uniform) no lane of the warp holds a particle: nothing to match
          const int rot = __any_sync(0xffffffffu, valid) ? skew_match((row0 * 8 + col0) & 31, valid) : 0;
          if (valid) {
            float wU[8], wW[8], dU[8], dW[8];
            T::template axis_skew<false>(dz0, tp, rot, wU, wW, dU, dW);
            int nx[8];
#pragma unroll
            for (int j = 0; j < 8; ++j) nx[j] = (j + rot) >= 8 ? 1 : 0;
            float ws[NCOMP];
#pragma unroll
            for (int q = 0; q < NCOMP; ++q) ws[q] = wv[k][q] * scale[q];
            if (NCOMP == 1) {
              const float fz = WEIGHTED ? ws[0] : ws[0] * ES_DENORM_Z;  // unit weights: see ES_DENORM_Z
#pragma unroll
              for (int j = 0; j < 8; ++j) wU[j] *= fz, wW[j] *= fz;
              if (!WEIGHTED) {
#pragma unroll
                for (int a = 0; a < P; ++a) wx[a] *= ES_DENORM_X;
              }
            }
            int* p0 = s_acc + (row0 * G::PITCH + col0 + rot);
#pragma unroll
            for (int a = 0; a < P; ++a)
#pragma unroll
              for (int b = 0; b < P; ++b) {
                const int a2 = b < P - 1 ? a : (a < P - 1 ? a + 1 : 0), b2 = b < P - 1 ? b + 1 : 0;
                const int nextoff = skew_next_off<G>(a, b);
                const float cur = wx[a] * wy[b], nxt = wx[a2] * wy[b2];
                int* rp = p0 + (a * G::SY + b) * G::PITCH;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  int* node = rp + (j + nx[j] * nextoff);
                  const float wgt = fmaf(nxt, wW[j], cur * wU[j]);  // one of wU[j], wW[j] is an exact zero
                  if (NCOMP == 1 && !WEIGHTED) {  // the one product, rounded once, as a denormal: ES_DENORM_Z
                    atomicAdd(reinterpret_cast<unsigned*>(node), __float_as_uint(wgt));
                  } else if (NCOMP == 1) {
                    atomicAdd(node, __float2int_rn(wgt));
                  } else {
#pragma unroll
                    for (int q = 0; q < NCOMP; ++q) atomicAdd(node + q * G::COMP, __float2int_rn(wgt * ws[q]));
                  }
                }
              }
          }
        } else if (i < iend) {
          int sx, sy, sz;
          float wx[P], wy[P], wz[P], dx[P], dy[P], dz[P];
          T::template axis<JVP>(apply_shift<T>(r[k].x, tp.frac[0]), tp, sx, wx, dx);
          T::template axis<JVP>(apply_shift<T>(r[k].y, tp.frac[1]), tp, sy, wy, dy);
          T::template axis<JVP>(apply_shift<T>(r[k].z, tp.frac[2]), tp, sz, wz, dz);
          NodeCol nc[P];
#pragma unroll
          for (int c = 0; c < P; ++c) nc[c] = node_col<G>(sx * G::SY + sy, sz + (G::ZLO - G::HLO) + c);
          if constexpr (JVP) {
            // w~ Wx Wy Wz + (w tx) dWx Wy Wz + (w ty) Wx dWy Wz + (w tz) Wx Wy dWz, the scale folded into z
            const float wt = wv[k][0], ax = wv[k][1], ay = wv[k][2], az = wv[k][3];
#pragma unroll
            for (int c = 0; c < P; ++c) {
              wz[c] *= scale[0];
              dz[c] *= scale[0] * az;
            }
#pragma unroll
            for (int a = 0; a < P; ++a) {
              const float pxa = fmaf(ax, dx[a], wt * wx[a]);
#pragma unroll
              for (int b = 0; b < P; ++b) {
                const float e1 = fmaf(wy[b], pxa, ay * wx[a] * dy[b]);
                const float e2 = wx[a] * wy[b];
#pragma unroll
                for (int c = 0; c < P; ++c)
                  atomicAdd(s_acc + ((a * G::SY + b) * nc[c].pitch + nc[c].base),
                            __float2int_rn(fmaf(e1, wz[c], e2 * dz[c])));
              }
            }
          } else {
            float wzs[NCOMP][P];  // the scale (and the particle's weight) folded into the z weights
            constexpr bool DENORM = T::ES && !WEIGHTED && NCOMP == 1;  // see ES_DENORM_Z
#pragma unroll
            for (int q = 0; q < NCOMP; ++q)
#pragma unroll
              for (int c = 0; c < P; ++c) wzs[q][c] = wz[c] * (wv[k][q] * scale[q] * (DENORM ? ES_DENORM_Z : 1.0f));
            if (DENORM) {
#pragma unroll
              for (int a = 0; a < P; ++a) wx[a] *= ES_DENORM_X;
            }
#pragma unroll
            for (int a = 0; a < P; ++a)
#pragma unroll
              for (int b = 0; b < P; ++b) {
                const float wxy = wx[a] * wy[b];
#pragma unroll
                for (int c = 0; c < P; ++c) {
                  int* node = s_acc + ((a * G::SY + b) * nc[c].pitch + nc[c].base);
#pragma unroll
                  for (int q = 0; q < NCOMP; ++q) {
                    if (WEIGHTED)
                      atomicAdd(node + q * G::COMP, __float2int_rn(wxy * wzs[q][c]));
                    else if (DENORM)
                      atomicAdd(reinterpret_cast<unsigned*>(node + q * G::COMP), __float_as_uint(wxy * wzs[q][c]));
                    else
                      atomicAdd(reinterpret_cast<unsigned*>(node + q * G::COMP), __float2uint_rn(wxy * wzs[q][c]));
                  }
                }
              }
          }
        }
        if (last) {  // slot k is free: request the next item's record (its first batch)
          const uint32_t ni = nbegin + (uint32_t)(k * BLOCK + tid);
          if (ni < nend) load_rec<WEIGHTED>(r[k], bv, ni);
        }
      }
      if (last) break;
      b0 += CHUNK_;
      load_batch(b0, iend);  // dense tile: further batches of the same item
      load_weights(b0);
    }
    if (tid == 0) s_next[par] = fetched + gridDim.x;
    __syncthreads();
    const uint32_t nn = s_next[par];
    par ^= 1;
    WorkItem nnwi = nwi;
    if (nn < nitems) nnwi = bv.items[nn];  // consumed after the flush

    // flush: vectorised global reductions along z (red.global.add.v4.f32), empty groups skipped; the
    // accumulators are zeroed on the way out.
    const int bx = wrap_lo(o.x0 - G::HLO - roll.x, m), by = wrap_lo(o.y0 - G::HLO - roll.y, m);
    const int bz = wrap_lo(o.z0 - G::ZLO - roll.z, m);
#pragma unroll
    for (int k = 0; k < (PRE ? NSLOT : 1); ++k) {
      for (int j = tid + k * BLOCK; j < (PRE ? min(NG, (k + 1) * BLOCK) : NG); j += BLOCK) {
        const int jc = NCOMP == 1 ? 0 : j / G::NGROUP;  // component blocks are padded to COMP words
        int4* src = reinterpret_cast<int4*>(s_acc) + (j + jc * (G::COMP / 4 - G::NGROUP));
        const int4 v = *src;
        if ((v.x | v.y | v.z | v.w) == 0) continue;
        *src = make_int4(0, 0, 0, 0);
        const uint32_t g = PRE ? gc[k] : group_coords(j);
        const int comp = NCOMP == 1 ? 0 : (int)(g >> 28);
        float is = inv_scale[0];
#pragma unroll
        for (int a = 1; a < NCOMP; ++a)
          if (comp == a) is = inv_scale[a];
        float4 f;
        if (WEIGHTED)
          f = make_float4(__int2float_rn(v.x) * is, __int2float_rn(v.y) * is, __int2float_rn(v.z) * is,
                          __int2float_rn(v.w) * is);
        else
          f = make_float4(__uint2float_rn((unsigned)v.x) * is, __uint2float_rn((unsigned)v.y) * is,
                          __uint2float_rn((unsigned)v.z) * is, __uint2float_rn((unsigned)v.w) * is);
        const int gx = wrap_hi(bx + (int)((g >> 20) & 255u), m), gy = wrap_hi(by + (int)((g >> 12) & 255u), m);
        const int gz = wrap_hi(bz + (int)(g & 4095u), m);
        float* p = mesh.p[comp] + (size_t)(unsigned)(gx * m + gy) * (unsigned)m;
        if ((gz & 3) == 0) {
          red_add_v4(p + gz, f);
        } else {  // integer part of the shift not a multiple of 4: scalar reductions, each wrapped
          atomicAdd(p + gz, f.x);
          atomicAdd(p + wrap_hi(gz + 1, m), f.y);
          atomicAdd(p + wrap_hi(gz + 2, m), f.z);
          atomicAdd(p + wrap_hi(gz + 3, m), f.w);
        }
      }
    }
    if (NBUF == 1)
      __syncthreads();  // the single buffer must be clean before the next deposit
    else
      s_acc = (s_acc == s_acc_all) ? s_acc_all + ACC : s_acc_all;
    it = nxt;
    wi = nwi;
    nxt = nn;
    nwi = nnwi;
  }
  if (tid == 0) sched_done(bv.sched);
}

// ---- K2, warp-private variant: unit weights, one field -------------------------------------------------
// One WARP per work item, the accumulator tile private to the warp: there is no CTA barrier anywhere (in the
// CTA-cooperative kernel above 35 % of the warp samples sat at the barrier between deposit and flush, ncu
// round 1).  A lane deposits every 32nd record of the item (coalesced 512-byte record loads, WD records per lane
// in flight, refilled as they are consumed, the next item's first records at the end), then the warp flushes its
// tile.  Used where WS_WARPS accumulator tiles per CTA fit several CTAs on an SM (CIC); the cooperative kernel
// serves the wider kernels, weights and vector fields.
constexpr int WS_WARPS = 4;  // warps per CTA
constexpr int WD = 10;       // records in flight per lane (128 registers per thread at 4 CTAs of 128 threads)

__device__ __forceinline__ void wsched_done(uint32_t* sched, uint32_t nwarps) {
  if (atomicAdd(&sched[1], 1u) == nwarps - 1u) {
    sched[0] = 0u;
    sched[1] = 0u;
  }
}

template <class T, bool FASTCIC>
__global__ void __launch_bounds__(WS_WARPS * 32, 4) k_scatter_warp(BinView bv, typename T::Params tp, int3 roll,
                                                                   float* __restrict__ mesh, int zeroed, uint32_t wb) {
  using G = Geo<T>;
  constexpr int P = T::P;
  extern __shared__ __align__(16) int s_acc_all[];
  const unsigned lane = threadIdx.x & 31u;
  int* s_acc = s_acc_all + (threadIdx.x >> 5) * G::COMP;
  const uint32_t nitems = *bv.nitems;
  const uint32_t nwarps = gridDim.x * WS_WARPS;
  const int m = bv.m;

  for (int j = (int)lane; j < G::COMP / 4; j += 32) reinterpret_cast<int4*>(s_acc)[j] = make_int4(0, 0, 0, 0);
  __syncwarp();

  // flush geometry of this lane (see the flush below): group fl_gq of every row, rows fl_rsub, fl_rsub + RPI, ...
  constexpr int FL_GPR = TZ / 4 + G::HZ / 4;  // float4 groups per (x, y) row: 8 in the MAIN plane, 1 or 2 in the HALO plane
  constexpr int FL_RPI = 32 / FL_GPR;         // rows per warp iteration
  static_assert(FL_RPI <= G::SY, "one wrap of sy per step");
  const int fl_rsub = (int)lane / FL_GPR, fl_gq = (int)lane - fl_rsub * FL_GPR;
  const bool fl_on = fl_rsub < FL_RPI, fl_main = fl_gq < TZ / 4;
  const int fl_zoff = fl_main ? 4 * fl_gq : TZ + 4 * (fl_gq - TZ / 4);
  const int fl_pitch = fl_main ? TZ : G::HZ, fl_base = fl_main ? 4 * fl_gq : G::MAIN + 4 * (fl_gq - TZ / 4);

  // Dynamic schedule in BATCHES of wb consecutive work items: warp g starts with batch g, further batches come
  // from the global counter.  The counter's round trip is long when every warp of the grid hammers it (one
  // same-address atomic per item: on the oversampled meshes, 256 particles per item, ncu round 2 showed 56 % of the
  // stall samples waiting for it, whatever instruction touched the result first), so (i) a batch is requested when
  // the previous one is STARTED and its id is first touched wb items later, (ii) wb = 8 items per request when the
  // items are light; wb = 1 for the heavy items of the headline, where balance matters more (host: run_scatter_warp).
  uint32_t q = (blockIdx.x * WS_WARPS + (threadIdx.x >> 5)) * wb, qend = q + wb;
  uint32_t claim = 0;  // lane 0: raw counter value = index of the next batch minus nwarps
  if (lane == 0) claim = atom_inc_noagg(&bv.sched[0]);
  auto next_id = [&]() -> uint32_t {  // warp-uniform
    if (q == qend) {
      q = (__shfl_sync(0xffffffffu, claim, 0) + nwarps) * wb;
      qend = q + wb;
      if (lane == 0) claim = atom_inc_noagg(&bv.sched[0]);
    }
    return q++;
  };
  uint32_t it = next_id(), nxt = next_id();
  WorkItem wi, nwi;
  wi.begin = wi.end = wi.txyz = nwi.begin = nwi.end = nwi.txyz = 0;
  uint4 r[WD];
  uint32_t keep = 0;  // xor of the records' .w: see the deposit loop
#pragma unroll
  for (int k = 0; k < WD; ++k) r[k] = make_uint4(0u, 0u, 0u, 0u);
  if (it < nitems) {
    wi = bv.items[it];
#pragma unroll
    for (int k = 0; k < WD; ++k) {
      const uint32_t i = wi.begin + (uint32_t)(k * 32) + lane;
      if (i < wi.end) load_rec<false>(r[k], bv, i);
    }
  }
  if (nxt < nitems) nwi = bv.items[nxt];

  while (it < nitems) {
    const uint32_t nn = next_id();  // item i+2
    const uint32_t n = wi.end - wi.begin;
    const uint32_t iend = wi.end;
    const TileOrigin o = tile_origin(wi);
    const uint32_t nbegin = nwi.begin, nend = nxt < nitems ? nwi.end : nwi.begin;

    // fixed-point scale: no node can receive more than n * WMAX3 (see k_scatter)
    const float bound = (float)n * T::WMAX3;
    int e = 0;
    const float f = frexpf(bound, &e);
    const int sexp = min(31, 31 - ((f == 0.5f) ? e - 1 : e));
    const float scale = pow2i(sexp), inv_scale = pow2i(-sexp);

    for (uint32_t b0 = wi.begin;; b0 += WD * 32) {
      const bool last = b0 + WD * 32 >= iend;  // uniform
#pragma unroll
      for (int k = 0; k < WD; ++k) {
        const uint32_t i = b0 + (uint32_t)(k * 32) + lane;
        const uint4 rk = r[k];
        // Keep the unused .w (original index) of the record LIVE until here (one LOP3 per record).  Otherwise
        // ptxas reuses its register as scratch while the next 128-bit record load into r[k] is still in flight,
        // and every such write waits for the load to land (write-after-write on the load's destination): ncu
        // showed 66 % of the stall samples on the first instruction after each prefetch, 1.24 ms instead of
        // 0.74 ms.  (An empty asm does not do it: it leaves no use in the PTX that ptxas sees.)
        keep ^= rk.w;
        const uint32_t pi = last ? nbegin + (uint32_t)(k * 32) + lane : i + (uint32_t)(WD * 32);
        if (pi < (last ? nend : iend)) load_rec<false>(r[k], bv, pi);
        if (i < iend) {
          if constexpr (FASTCIC && P == 2 && !T::SHIFT && G::ZLO == 0) {
            // Unshifted CIC (the headline assign): the first z node is always in the MAIN plane (sz < TZ by the
            // binning), so the four rows of a z node are ONE base address plus compile-time offsets; only
            // sz = TZ - 1 sends the second z node to the HALO plane (a branch, not per-node selects).  The
            // generic addressing below spent ~20 of its 72 instructions per particle on pitch/base selects
            // and the kernel is issue-bound (ncu: 70 % issue active).
            constexpr float INV = 1.0f / (float)REC_ONE;
            const float tx = (float)(rk.x & REC_MASK) * INV, ty = (float)(rk.y & REC_MASK) * INV;
            const float tzs = (float)(rk.z & REC_MASK) * (INV * scale);
            const int sx = (int)(rk.x >> REC_FRAC) - REC_BIAS, sy = (int)(rk.y >> REC_FRAC) - REC_BIAS;
            const int sz = (int)(rk.z >> REC_FRAC) - REC_BIAS;
            const int row0 = sx * G::SY + sy;
            const float ox = 1.0f - tx, oy = 1.0f - ty, ozs = scale - tzs;
            const float w00 = ox * oy, w01 = ox * ty, w10 = tx * oy, w11 = tx * ty;
            unsigned* p0 = reinterpret_cast<unsigned*>(s_acc) + (row0 * TZ + sz);
            atomicAdd(p0, __float2uint_rn(w00 * ozs));
            atomicAdd(p0 + TZ, __float2uint_rn(w01 * ozs));
            atomicAdd(p0 + G::SY * TZ, __float2uint_rn(w10 * ozs));
            atomicAdd(p0 + (G::SY + 1) * TZ, __float2uint_rn(w11 * ozs));
            const unsigned u00 = __float2uint_rn(w00 * tzs), u01 = __float2uint_rn(w01 * tzs);
            const unsigned u10 = __float2uint_rn(w10 * tzs), u11 = __float2uint_rn(w11 * tzs);
            // second z node: next word of the MAIN plane, or (sz = TZ - 1) the first column of the HALO plane, whose
            // rows have another pitch.  Selected, not branched: with 32 lanes at 32 different z one lane of almost
            // every warp is at sz = TZ - 1, and the branch made 64 % of the warps run both sides (ncu round 2: 10.6
            // instead of 8 ATOMS per warp and particle, and the shared-memory pipe is the busiest unit, 66 %).
            const bool inm = sz < TZ - 1;
            unsigned* p1 = inm ? p0 + 1 : reinterpret_cast<unsigned*>(s_acc) + (G::MAIN + row0 * G::HZ);
            const int py = inm ? TZ : G::HZ, px = inm ? G::SY * TZ : G::SY * G::HZ;
            atomicAdd(p1, u00);
            atomicAdd(p1 + py, u01);
            atomicAdd(p1 + px, u10);
            atomicAdd(p1 + px + py, u11);
            continue;
          }
          int sx, sy, sz;
          float wx[P], wy[P], wz[P], dummy[P];
          T::template axis<false>(apply_shift<T>(rk.x, tp.frac[0]), tp, sx, wx, dummy);
          T::template axis<false>(apply_shift<T>(rk.y, tp.frac[1]), tp, sy, wy, dummy);
          T::template axis<false>(apply_shift<T>(rk.z, tp.frac[2]), tp, sz, wz, dummy);
          NodeCol nc[P];
#pragma unroll
          for (int c = 0; c < P; ++c) {
            nc[c] = node_col<G>(sx * G::SY + sy, sz + (G::ZLO - G::HLO) + c);
            wz[c] *= scale;
          }
#pragma unroll
          for (int a = 0; a < P; ++a)
#pragma unroll
            for (int b = 0; b < P; ++b) {
              const float wxy = wx[a] * wy[b];
#pragma unroll
              for (int c = 0; c < P; ++c)
                atomicAdd(reinterpret_cast<unsigned*>(s_acc + ((a * G::SY + b) * nc[c].pitch + nc[c].base)),
                          __float2uint_rn(wxy * wz[c]));
            }
        }
      }
      if (last) break;
    }
    __syncwarp();  // the lanes' deposits are visible below
    WorkItem nnwi = nwi;
    if (nn < nitems) nnwi = bv.items[nn];

    // flush (as in k_scatter): red.global.add.v4.f32 per group of 4 nodes along z, empty groups skipped.
    // Exclusive groups are STORED instead: when the mesh is known to be zero before this launch (`zeroed`, set by
    // pm_force for its own mesh) and the tile is a single work item (bit 31 of wi.tile, set by k_items*), the
    // nodes [t0 + HHI, tend - HLO) of every axis receive deposits from this item alone (a neighbour's kernel
    // support ends before them), so no reduction is needed there and the L2 does not have to fetch the zeroed
    // line from DRAM first (ncu: 0.54 GB of the scatter's 2.69 GB of DRAM reads were that read-modify-write).
    // A lane keeps ONE float4 group of a row (fl_gq) and walks the rows, RPI rows per warp iteration: the z part of the
    // address and of the exclusive-interior test is per lane and item, the (x, y) part advances incrementally -- no
    // divisions and a third of the instructions of a flat walk over the groups.  On the oversampled meshes (256
    // particles per tile against 729 groups) the flush was three quarters of the kernel's instructions.
    const int bx = wrap_lo(o.x0 - G::HLO - roll.x, m), by = wrap_lo(o.y0 - G::HLO - roll.y, m);
    const int bz = wrap_lo(o.z0 - G::ZLO - roll.z, m);
    const bool excl_item = zeroed && (wi.tile >> 31);
    const int nx = min(TX, m - o.x0), ny = min(TY, m - o.y0), nz = min(TZ, m - o.z0);  // cells of a ragged last tile
    const int gz = wrap_hi(bz + fl_zoff, m);
    const bool excl_z = excl_item && fl_zoff >= G::ZLO + G::HHI && fl_zoff + 3 - G::ZLO < nz - G::HLO;
    if (fl_on) {
      int sx = 0, sy = fl_rsub;
      for (int row = fl_rsub; row < G::NROW; row += FL_RPI) {
        int4* src = reinterpret_cast<int4*>(s_acc + row * fl_pitch + fl_base);
        const int4 v = *src;
        if ((v.x | v.y | v.z | v.w) != 0) {
          *src = make_int4(0, 0, 0, 0);
          const float4 fv = make_float4(__uint2float_rn((unsigned)v.x) * inv_scale, __uint2float_rn((unsigned)v.y) * inv_scale,
                                        __uint2float_rn((unsigned)v.z) * inv_scale, __uint2float_rn((unsigned)v.w) * inv_scale);
          const int gx = wrap_hi(bx + sx, m), gy = wrap_hi(by + sy, m);
          float* p = mesh + (size_t)(unsigned)(gx * m + gy) * (unsigned)m;
          const bool excl = excl_z && sx >= G::HLO + G::HHI && sx < nx && sy >= G::HLO + G::HHI && sy < ny;
          if (excl) {
            if ((gz & 3) == 0) {
              *reinterpret_cast<float4*>(p + gz) = fv;
            } else {
              p[gz] = fv.x;
              p[wrap_hi(gz + 1, m)] = fv.y;
              p[wrap_hi(gz + 2, m)] = fv.z;
              p[wrap_hi(gz + 3, m)] = fv.w;
            }
          } else if ((gz & 3) == 0) {
            red_add_v4(p + gz, fv);
          } else {  // integer part of the shift not a multiple of 4: scalar reductions, each wrapped
            atomicAdd(p + gz, fv.x);
            atomicAdd(p + wrap_hi(gz + 1, m), fv.y);
            atomicAdd(p + wrap_hi(gz + 2, m), fv.z);
            atomicAdd(p + wrap_hi(gz + 3, m), fv.w);
          }
        }
        sy += FL_RPI;
        if (sy >= G::SY) {
          sy -= G::SY;
          ++sx;
        }
      }
    }
    __syncwarp();  // the tile is clean before the next deposit
    it = nxt;
    wi = nwi;
    nxt = nn;
    nwi = nnwi;
  }
  if (lane == 0) wsched_done(bv.sched, nwarps);
  if (keep == 0x9e3779b9u && nitems == 0xffffffffu) mesh[0] = 0.f;  // never true: gives `keep` a consumer
}

// ---- TMA / mbarrier primitives (sm_90+ PTX; SASS: UTMALDG, SYNCS) --------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  const uint32_t a = smem_u32(bar);
  uint32_t ok = 0;
  do {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(a), "r"(parity)
        : "memory");
  } while (!ok);
}
// box (innermost first) at coordinates (c0, c1, c2) = (z, y, x); out-of-bounds elements are zero-filled
__device__ __forceinline__ void tma_load_3d(void* dst, const CUtensorMap* map, uint64_t* bar, int c0, int c1, int c2) {
  asm volatile(
      "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4, %5}], [%2];"
      ::"r"(smem_u32(dst)), "l"(map), "r"(smem_u32(bar)), "r"(c0), "r"(c1), "r"(c2)
      : "memory");
}

// ---- K4 / K7: tile gather ----------------------------------------------------------------------------
// GMODE G_VALUES: v[i*NST + a] = sum_j mesh_a[j] W_j(X_i)                                          (Eq. C.2)
//       G_GRAD  : v[i*3 + b]   = sum_a coef_a(i) sum_j mesh_a[j] d/du_b W_j(X_i)                   (Eq. C.6, C.12)
//       G_JVP   : v[i*NO + a]  = sum_j mesh_a[j] (t_i . d/du) W_j(X_i)              [+ sum_j mesh~_a[j] W_j(X_i)]
//                 (Eq. C.13b; G_JVPT: the NO tangent meshes are staged behind the NO primal ones, NST = 2 NO)
// out = alpha * v + out_scale * out; the caller folds 1/Delta (d/dX = (1/Delta) d/du) into alpha / tan_scale.
//
// Persistent CTAs draw work items from the dynamic schedule.  Thread 0 stages the tile + halo box of every
// component with one TMA tensor copy each (north_star "TMA staging of mesh tiles"), completion on an
// mbarrier (an L2 evict-last hint on the copies was measured and changed nothing); with STAGES = 2
// the box of the CTA's next item is in flight while the particles of the current one are interpolated.
// TMA zero-fills what lies beyond the mesh edge, it does not wrap: tiles whose box crosses an edge (a few
// per cent) are patched by the threads with periodic loads after the copy has landed.  roll in [0, m); when
// roll.z is not a multiple of 4 no box start is 16-byte aligned and the threads stage everything (manual).
enum { G_VALUES = 0, G_GRAD = 1, G_JVP = 2, G_JVPT = 3 };

struct GatherDev {  // per-launch arguments beyond the meshes
  const float* cot;      // G_GRAD: coef_a(i) = a < ncot ? cot[i*cstride + a] : const_coef * (wmul ? wmul[i] : 1)
  int cstride, ncot;
  float const_coef;
  const float* wmul;
  const float* pos_tan;  // G_JVP*: tangent positions [N,3] or NULL (then only the tangent meshes contribute)
  float tan_scale;       // G_JVP*: 1/Delta
  float alpha, out_scale;
  float* out;
  // Fused tail of the drift-kick-drift step (Eq. 2.14b-c, G_VALUES with NST = 3, out = V): after the kick
  // V_i <- out_scale V_i + alpha A_i the particle is drifted, X_i <- wrap(X_i + drift_tau V_i) with every
  // operation rounded to fp32 and no fused multiply-add (reading R18).
  float* drift_pos;
  float drift_tau, box;
  // Reductions of the adjoint kick (Table 3), dot_with = V* [N,3]:
  //   *dot_acc += dot_scale sum_i dot_with_i . v_i      (beta*:  V* . A)
  //   *dot_out +=           sum_i dot_with_i . out_i    (alpha*: V* . V^{n-1}, the kicked-back velocity)
  const float* dot_with;
  double* dot_acc;
  double* dot_out;
  float dot_scale;
};

template <class T, int NST, int GMODE, int STAGES>
__global__ void __launch_bounds__(BLOCK) k_gather(BinView bv, typename T::Params tp, int3 roll,
                                                  const __grid_constant__ TMapSet<2 * NST> maps,
                                                  CMeshPtrs<NST> mesh, GatherDev gd, int manual) {
  using G = Geo<T>;
  constexpr int P = T::P;
  constexpr bool GRAD = GMODE == G_GRAD;
  constexpr bool JVP = GMODE == G_JVP || GMODE == G_JVPT;
  constexpr bool DERIV = GRAD || JVP;
  constexpr int NO = GMODE == G_JVPT ? NST / 2 : NST;  // outputs per particle (G_GRAD: 3)
  static_assert(GMODE != G_JVPT || NST % 2 == 0, "G_JVPT stages the primal and the tangent meshes");
  constexpr int KB = T::ES ? ES_KB : 4;  // records in flight per thread
  constexpr uint32_t BOX_BYTES = (uint32_t)(NST * (G::MAIN + G::HAL) * sizeof(float));
  extern __shared__ __align__(128) unsigned char s_raw[];
  __shared__ __align__(8) uint64_t s_bar[STAGES];
  __shared__ uint32_t s_next[2];
  __shared__ double s_dots[2 * (BLOCK / 32)];
  // 128-byte aligned TMA destinations; the offset is applied to the shared-space pointer so that the loads
  // below stay LDS (a round trip through uintptr_t made them generic LD with 64-bit address arithmetic)
  float* s_base = reinterpret_cast<float*>(s_raw + ((128u - (smem_u32(s_raw) & 127u)) & 127u));
  const int tid = threadIdx.x;
  const uint32_t nitems = *bv.nitems;
  const int m = bv.m;
  float* __restrict__ out = gd.out;
  const float alpha = gd.alpha, out_scale = gd.out_scale;
  double dsum0 = 0.0, dsum1 = 0.0;

  if (tid == 0) {
#pragma unroll
    for (int s = 0; s < STAGES; ++s) mbar_init(&s_bar[s], 1);
    fence_barrier_init();
    fence_proxy_async();
    s_next[0] = sched_next(bv.sched);  // the item after this CTA's first
  }
  if (G::DENSE) {  // the slack behind the rows is read (with weight zero) by the skewed walk: it must hold finite values
    constexpr int SLACK = G::COMP - (G::MAIN + G::HAL);
    for (int j = tid; j < STAGES * NST * SLACK; j += BLOCK)
      s_base[(j / SLACK) * G::COMP + (G::MAIN + G::HAL) + j % SLACK] = 0.0f;
  }
  __syncthreads();

  auto box_start = [&](const TileOrigin& o, int& cx, int& cy, int& cz) {
    cx = wrap_lo(o.x0 - G::HLO - roll.x, m);
    cy = wrap_lo(o.y0 - G::HLO - roll.y, m);
    cz = wrap_lo(o.z0 - G::ZLO - roll.z, m);
  };
  auto issue = [&](const WorkItem& w, int stage) {  // thread 0
    if (manual & 1) return;
    const TileOrigin o = tile_origin(w);
    int cx, cy, cz;
    box_start(o, cx, cy, cz);
    mbar_expect_tx(&s_bar[stage], BOX_BYTES);
#pragma unroll
    for (int a = 0; a < NST; ++a) {  // main plane (first TZ nodes of every row) and halo plane (the rest)
      float* dst = s_base + (stage * NST + a) * G::COMP;
      tma_load_3d(dst, &maps.m[2 * a], &s_bar[stage], cz, cy, cx);  // DENSE: the whole rows in one box
      if (!G::DENSE) tma_load_3d(dst + G::MAIN, &maps.m[2 * a + 1], &s_bar[stage], cz + TZ, cy, cx);
    }
  };

  uint32_t phases = 0;  // bit s: parity the next wait on stage s uses
  int stage = 0, par = 1;
  uint32_t it = blockIdx.x, nxt = s_next[0];
  WorkItem wi, nwi;
  wi.begin = wi.end = wi.txyz = nwi.begin = nwi.end = nwi.txyz = 0;
  uint4 r[KB];  // records in flight: the slot a particle frees is refilled KB * BLOCK records ahead
#pragma unroll
  for (int k = 0; k < KB; ++k) r[k] = make_uint4(0u, 0u, 0u, 0u);
  if (it < nitems) {
    wi = bv.items[it];
    if (tid == 0) issue(wi, 0);
#pragma unroll
    for (int k = 0; k < KB; ++k) {
      const uint32_t i = wi.begin + (uint32_t)(k * BLOCK + tid);
      if (i < wi.end) load_rec<true>(r[k], bv, i);
    }
  }
  if (nxt < nitems) nwi = bv.items[nxt];

  while (it < nitems) {
    uint32_t fetched = 0;  // item i+2: issued now, stored right before the barrier at the end of the item
    if (tid == 0) {
      fetched = atom_inc_noagg(&bv.sched[0]);  // raw: gridDim.x is added where it is stored
      if (STAGES == 2 && nxt < nitems) issue(nwi, stage ^ 1);
    }
    const TileOrigin o = tile_origin(wi);
    const float* s_val = s_base + stage * NST * G::COMP;
    const uint32_t nbegin = nwi.begin, nend = nxt < nitems ? nwi.end : nwi.begin;  // empty when there is no next item

    if (!(manual & 1)) {
      mbar_wait(&s_bar[stage], (phases >> stage) & 1u);
      phases ^= 1u << stage;
    }

    int cx, cy, cz;
    box_start(o, cx, cy, cz);
    if ((manual & 1) || cx + G::SX > m || cy + G::SY > m || cz + TZ + G::HZ > m) {  // uniform: box crosses a mesh edge
      float* s_w = s_base + stage * NST * G::COMP;
      for (int j = tid; j < NST * G::NGROUP; j += BLOCK) {
        const int comp = j / G::NGROUP, rr = j - comp * G::NGROUP;
        int row, zoff;
        group_pos<G>(rr, row, zoff);
        const int sy = row % G::SY, sx = row / G::SY;
        if (!(manual & 1) && cx + sx < m && cy + sy < m && cz + zoff + 3 < m) continue;  // TMA delivered it
        // true modulo: on the smallest meshes (m < 24) the box is longer than two periods of the mesh
        const float* p = mesh.p[comp] + ((size_t)((cx + sx) % m) * m + (cy + sy) % m) * m;
        const int gz = cz + zoff;
        const float4 v = make_float4(__ldg(p + gz % m), __ldg(p + (gz + 1) % m), __ldg(p + (gz + 2) % m),
                                     __ldg(p + (gz + 3) % m));
        reinterpret_cast<float4*>(s_w + comp * G::COMP)[rr] = v;
      }
      fence_proxy_async();  // generic-proxy writes before the async proxy refills this buffer
      __syncthreads();
    }

    for (uint32_t b0 = wi.begin;; b0 += KB * BLOCK) {  // at least once: the last pass requests the next item's records
      const bool last = b0 + KB * BLOCK >= wi.end;  // uniform
#pragma unroll
      for (int k = 0; k < KB; ++k) {
        const uint32_t i = b0 + (uint32_t)(k * BLOCK + tid);
        const uint4 rk = r[k];
        // refill the slot: the record one batch ahead, or (last batch) the next item's first batch
        const uint32_t pi = last ? nbegin + (uint32_t)(k * BLOCK + tid) : i + (uint32_t)(KB * BLOCK);
        if (pi < (last ? nend : wi.end)) load_rec<true>(r[k], bv, pi);
        const bool valid = i < wi.end;
        if (!T::SKEW && !valid) continue;
        int sx = 0, sy = 0, sz = 0;
        float wx[P], wy[P], wz[P], dx[P], dy[P], dz[P];
        // skewed walk (ES kernels, skew_match): z weights per step, for the current and for the next row of the walk
        float wU[T::SKEW ? 8 : 1], wW[T::SKEW ? 8 : 1], dU[T::SKEW ? 8 : 1], dW[T::SKEW ? 8 : 1];
        int nx[T::SKEW ? 8 : 1];
        const float* p0 = nullptr;
        if constexpr (T::SKEW) {
          float dz0 = 0.0f;
          if (valid) {
            T::template axis<DERIV>(rk.x, tp, sx, wx, dx);
            T::template axis<DERIV>(rk.y, tp, sy, wy, dy);
            T::origin(rk.z, sz, dz0);
          }
          const int row0 = sx * G::SY + sy, col0 = sz + (G::ZLO - G::HLO);
          if (!__any_sync(0xffffffffu, valid)) continue;  // warp-uniform
          const int rot = skew_match((row0 * 8 + col0) & 31, valid);
          if (!valid) continue;
          T::template axis_skew<DERIV>(dz0, tp, rot, wU, wW, dU, dW);
#pragma unroll
          for (int j = 0; j < 8; ++j) nx[j] = (j + rot) >= 8 ? 1 : 0;
          p0 = s_val + (row0 * G::PITCH + col0 + rot);
        } else {
          T::template axis<DERIV>(apply_shift<T>(rk.x, tp.frac[0]), tp, sx, wx, dx);
          T::template axis<DERIV>(apply_shift<T>(rk.y, tp.frac[1]), tp, sy, wy, dy);
          T::template axis<DERIV>(apply_shift<T>(rk.z, tp.frac[2]), tp, sz, wz, dz);
        }
        // (TMA's 128-byte swizzle of the MAIN plane was measured: it is correct but RAISES the bank conflicts of
        // Lagrangian-ordered particles from 85 M to 136 M wavefronts, 1.09 -> 1.21 ms: with a row pitch of 32 words
        // lanes at distinct z already sit in distinct banks, and the swizzle scatters them.)
        NodeCol nc[P];
#pragma unroll
        for (int c = 0; c < P; ++c) nc[c] = node_col<G>(sx * G::SY + sy, sz + (G::ZLO - G::HLO) + c);
        if (GMODE == G_VALUES) {
          float acc[NST];
#pragma unroll
          for (int a = 0; a < NST; ++a) acc[a] = 0.0f;
          if constexpr (T::SKEW) {
#pragma unroll
            for (int a = 0; a < P; ++a)
#pragma unroll
              for (int b = 0; b < P; ++b) {
                const int a2 = b < P - 1 ? a : (a < P - 1 ? a + 1 : 0), b2 = b < P - 1 ? b + 1 : 0;
                const int nextoff = skew_next_off<G>(a, b);
                const float cur = wx[a] * wy[b], nxt = wx[a2] * wy[b2];
                const float* rp = p0 + (a * G::SY + b) * G::PITCH;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  const float wgt = fmaf(nxt, wW[j], cur * wU[j]);
                  const float* node = rp + (j + nx[j] * nextoff);
#pragma unroll
                  for (int q = 0; q < NST; ++q) acc[q] = fmaf(wgt, node[q * G::COMP], acc[q]);
                }
              }
          } else {
#pragma unroll
          for (int a = 0; a < P; ++a)
#pragma unroll
            for (int b = 0; b < P; ++b) {
              const float wxy = wx[a] * wy[b];
#pragma unroll
              for (int c = 0; c < P; ++c) {
                const float wxyz = wxy * wz[c];
                const float* node = s_val + ((a * G::SY + b) * nc[c].pitch + nc[c].base);
#pragma unroll
                for (int q = 0; q < NST; ++q) acc[q] = fmaf(wxyz, node[q * G::COMP], acc[q]);
              }
            }
          }
          float* dst = out + (size_t)rk.w * NST;
          float nv[NST];
#pragma unroll
          for (int a = 0; a < NST; ++a) {
            nv[a] = out_scale != 0.0f ? fmaf(alpha, acc[a], out_scale * dst[a]) : alpha * acc[a];
            dst[a] = nv[a];
          }
          if (NST == 3) {  // DKD tails (uniform branches on launch arguments)
            if (gd.dot_with) {
              const float* dw = gd.dot_with + (size_t)rk.w * 3;
              const float d0 = __ldg(dw), d1 = __ldg(dw + 1), d2 = __ldg(dw + 2);
              dsum0 += (double)d0 * (double)acc[0] + (double)d1 * (double)acc[1] + (double)d2 * (double)acc[2];
              dsum1 += (double)d0 * (double)nv[0] + (double)d1 * (double)nv[1] + (double)d2 * (double)nv[2];
            }
            if (gd.drift_pos) {
              float* xp = gd.drift_pos + (size_t)rk.w * 3;
#pragma unroll
              for (int a = 0; a < 3; ++a) xp[a] = drift_fp32(xp[a], nv[a], gd.drift_tau, gd.box);
            }
          }
        } else if (GRAD) {
          float coef[NST];
          const float cc = gd.const_coef * (gd.wmul ? __ldg(gd.wmul + rk.w) : 1.0f);
#pragma unroll
          for (int a = 0; a < NST; ++a) coef[a] = a < gd.ncot ? __ldg(gd.cot + (size_t)rk.w * gd.cstride + a) : cc;
          float gx = 0.0f, gy = 0.0f, gz = 0.0f;
          if constexpr (T::SKEW) {
#pragma unroll
            for (int a = 0; a < P; ++a)
#pragma unroll
              for (int b = 0; b < P; ++b) {
                const int a2 = b < P - 1 ? a : (a < P - 1 ? a + 1 : 0), b2 = b < P - 1 ? b + 1 : 0;
                const int nextoff = skew_next_off<G>(a, b);
                const float cdx = dx[a] * wy[b], cdy = wx[a] * dy[b], cxy = wx[a] * wy[b];
                const float ndx = dx[a2] * wy[b2], ndy = wx[a2] * dy[b2], nxy = wx[a2] * wy[b2];
                const float* rp = p0 + (a * G::SY + b) * G::PITCH;
#pragma unroll
                for (int j = 0; j < 8; ++j) {
                  const float* node = rp + (j + nx[j] * nextoff);
                  float val = 0.0f;
#pragma unroll
                  for (int q = 0; q < NST; ++q) val = fmaf(coef[q], node[q * G::COMP], val);
                  gx = fmaf(fmaf(ndx, wW[j], cdx * wU[j]), val, gx);
                  gy = fmaf(fmaf(ndy, wW[j], cdy * wU[j]), val, gy);
                  gz = fmaf(fmaf(nxy, dW[j], cxy * dU[j]), val, gz);
                }
              }
          } else {
#pragma unroll
          for (int a = 0; a < P; ++a)
#pragma unroll
            for (int b = 0; b < P; ++b) {
              const float wdx = dx[a] * wy[b], wdy = wx[a] * dy[b], wxy = wx[a] * wy[b];
#pragma unroll
              for (int c = 0; c < P; ++c) {
                const float* node = s_val + ((a * G::SY + b) * nc[c].pitch + nc[c].base);
                float val = 0.0f;
#pragma unroll
                for (int q = 0; q < NST; ++q) val = fmaf(coef[q], node[q * G::COMP], val);
                gx = fmaf(wdx * wz[c], val, gx);
                gy = fmaf(wdy * wz[c], val, gy);
                gz = fmaf(wxy * dz[c], val, gz);
              }
            }
          }
          float* dst = out + (size_t)rk.w * 3;
          dst[0] = out_scale != 0.0f ? fmaf(alpha, gx, out_scale * dst[0]) : alpha * gx;
          dst[1] = out_scale != 0.0f ? fmaf(alpha, gy, out_scale * dst[1]) : alpha * gy;
          dst[2] = out_scale != 0.0f ? fmaf(alpha, gz, out_scale * dst[2]) : alpha * gz;
        } else {  // JVP, Eq. C.13b: (t . d/du) W = tx dWx Wy Wz + ty Wx dWy Wz + tz Wx Wy dWz
          static_assert(!T::SKEW || !JVP, "the forward-mode gather is not built for the ES kernel");
          float tx = 0.0f, ty = 0.0f, tz = 0.0f;
          if (gd.pos_tan) {
            const float* tp3 = gd.pos_tan + (size_t)rk.w * 3;
            tx = __ldg(tp3) * gd.tan_scale, ty = __ldg(tp3 + 1) * gd.tan_scale, tz = __ldg(tp3 + 2) * gd.tan_scale;
          }
          float acc[NO];
#pragma unroll
          for (int a = 0; a < NO; ++a) acc[a] = 0.0f;
#pragma unroll
          for (int a = 0; a < P; ++a)
#pragma unroll
            for (int b = 0; b < P; ++b) {
              const float wxy = wx[a] * wy[b];
              const float txy = tx * dx[a] * wy[b] + ty * wx[a] * dy[b];
              const float tzxy = tz * wxy;
#pragma unroll
              for (int c = 0; c < P; ++c) {
                const float wd = fmaf(txy, wz[c], tzxy * dz[c]);
                const float* node = s_val + ((a * G::SY + b) * nc[c].pitch + nc[c].base);
#pragma unroll
                for (int q = 0; q < NO; ++q) {
                  acc[q] = fmaf(wd, node[q * G::COMP], acc[q]);
                  if (GMODE == G_JVPT) acc[q] = fmaf(wxy * wz[c], node[(NO + q) * G::COMP], acc[q]);
                }
              }
            }
          float* dst = out + (size_t)rk.w * NO;
#pragma unroll
          for (int a = 0; a < NO; ++a) dst[a] = out_scale != 0.0f ? fmaf(alpha, acc[a], out_scale * dst[a]) : alpha * acc[a];
        }
      }
      if (last) break;
    }
    if (tid == 0) s_next[par] = fetched + gridDim.x;
    __syncthreads();  // every thread is done with this stage: it may be refilled
    const uint32_t nn = s_next[par];
    par ^= 1;
    WorkItem nnwi = nwi;
    if (nn < nitems) nnwi = bv.items[nn];
    if (STAGES == 2) {
      stage ^= 1;
    } else if (tid == 0 && nxt < nitems) {
      issue(nwi, 0);
    }
    it = nxt;
    wi = nwi;
    nxt = nn;
    nwi = nnwi;
  }
  if (GMODE == G_VALUES && NST == 3 && gd.dot_with) {  // one pair of double atomics per CTA
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) {
      dsum0 += __shfl_xor_sync(0xffffffffu, dsum0, d);
      dsum1 += __shfl_xor_sync(0xffffffffu, dsum1, d);
    }
    if ((tid & 31) == 0) {
      s_dots[2 * (tid >> 5)] = dsum0;
      s_dots[2 * (tid >> 5) + 1] = dsum1;
    }
    __syncthreads();
    if (tid == 0) {
      double a0 = 0.0, a1 = 0.0;
      for (int w = 0; w < BLOCK / 32; ++w) {
        a0 += s_dots[2 * w];
        a1 += s_dots[2 * w + 1];
      }
      if (gd.dot_acc) atomicAdd(gd.dot_acc, (double)gd.dot_scale * a0);
      if (gd.dot_out) atomicAdd(gd.dot_out, a1);
    }
  }
  if (tid == 0) sched_done(bv.sched);
}

// ---- host-side launch helpers ------------------------------------------------------------------------
inline int norm_roll(int r, int m) {
  r %= m;
  return r < 0 ? r + m : r;
}

// Grid of a persistent mesh kernel: resident CTAs per SM x SMs, capped by an upper bound of the item count.
inline int mesh_grid(const Ctx* c, int occ) {
  int64_t bound = (int64_t)c->ntiles + c->bin_n / ITEM_MAX + 1;
  int64_t cap = (int64_t)c->num_sms * (occ < 1 ? 1 : occ);
  return (int)(bound < cap ? bound : cap);
}

template <class T, int NCOMP, int WMODE>
int run_scatter(Ctx* c, const typename T::Params& tp, const int roll[3], const ScatterSrc& src, float* const mesh[],
                cudaStream_t st) {
  using G = Geo<T>;
  constexpr size_t acc_bytes = sizeof(int) * (size_t)NCOMP * G::COMP;
  constexpr int NBUF = 2 * acc_bytes <= 48 * 1024 ? 2 : 1;  // two accumulator tiles when they are cheap
  const size_t smem = NBUF * acc_bytes;
  auto kern = k_scatter<T, NCOMP, WMODE, NBUF>;
  int occ = 0;
  PM_TRY(kernel_occupancy(c, (const void*)kern, BLOCK, smem, &occ));
  MeshPtrs<NCOMP> mp;
  for (int a = 0; a < NCOMP; ++a) mp.p[a] = mesh[a];
  const int m = c->mg;
  kern<<<mesh_grid(c, occ), BLOCK, smem, st>>>(bin_view(c), tp,
                                               make_int3(norm_roll(roll[0], m), norm_roll(roll[1], m), norm_roll(roll[2], m)),
                                               src, mp);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}
inline ScatterSrc weights_src(const float* w, int wstride) {
  ScatterSrc s = {w, wstride, nullptr, nullptr, 0.f};
  return s;
}

// Unit-weight, single-field scatter with warp-private tiles (k_scatter_warp).
template <class T>
int run_scatter_warp(Ctx* c, const typename T::Params& tp, const int roll[3], float* mesh, cudaStream_t st) {
  const int zeroed = c->scatter_mesh_zeroed ? 1 : 0;
  using G = Geo<T>;
  constexpr size_t smem = sizeof(int) * (size_t)WS_WARPS * G::COMP;
  auto kern = k_scatter_warp<T, true>;
  int occ = 0;
  PM_TRY(kernel_occupancy(c, (const void*)kern, WS_WARPS * 32, smem, &occ));
  const int64_t bound = ((int64_t)c->ntiles + c->bin_n / ITEM_MAX + 1 + WS_WARPS - 1) / WS_WARPS;
  const int64_t cap = (int64_t)c->num_sms * occ;
  const int m = c->mg;
  // work items per schedule request: light items (oversampled meshes) in batches of up to 8, heavy ones singly
  const int64_t per_item = c->bin_n / (c->ntiles > 0 ? c->ntiles : 1);
  const uint32_t wb = per_item >= 1024 ? 1u : (per_item >= 512 ? 2u : (per_item >= 256 ? 4u : 8u));
  kern<<<(int)(bound < cap ? bound : cap), WS_WARPS * 32, smem, st>>>(
      bin_view(c), tp, make_int3(norm_roll(roll[0], m), norm_roll(roll[1], m), norm_roll(roll[2], m)), mesh, zeroed, wb);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

template <class T, int NST, int GMODE>
int run_gather(Ctx* c, const typename T::Params& tp, const int roll[3], const GatherArgs& ga, cudaStream_t st) {
  using G = Geo<T>;
  constexpr size_t stage_bytes = sizeof(float) * (size_t)NST * G::COMP;
  constexpr int STAGES = 2 * stage_bytes <= 100 * 1024 ? 2 : 1;
  constexpr size_t smem = STAGES * stage_bytes + 128;
  auto kern = k_gather<T, NST, GMODE, STAGES>;
  int occ = 0;
  PM_TRY(kernel_occupancy(c, (const void*)kern, BLOCK, smem, &occ));
  CMeshPtrs<NST> mp;
  TMapSet<2 * NST> maps;
  const int m = c->mg;
  for (int a = 0; a < NST; ++a) {
    mp.p[a] = ga.mesh[a];
    PM_TRY(make_mesh_tmap(c, ga.mesh[a], G::SX, G::SY, G::DENSE ? G::PITCH : TZ, &maps.m[2 * a]));
    PM_TRY(make_mesh_tmap(c, ga.mesh[a], G::SX, G::SY, G::HZ, &maps.m[2 * a + 1]));  // unused by DENSE tiles
  }
  const double inv_delta = (double)c->mg / c->p.box;
  GatherDev gd;
  gd.cot = ga.cot;
  gd.cstride = ga.cstride;
  gd.ncot = ga.ncot;
  gd.const_coef = ga.const_coef;
  gd.wmul = ga.wmul;
  gd.pos_tan = ga.pos_tan;
  gd.tan_scale = (float)inv_delta;
  gd.alpha = GMODE == G_GRAD ? (float)((double)ga.alpha * inv_delta) : ga.alpha;
  gd.out_scale = ga.out_scale;
  gd.out = ga.out;
  gd.drift_pos = ga.drift_pos;
  gd.drift_tau = ga.drift_tau;
  gd.box = (float)c->p.box;
  gd.dot_with = ga.dot_with;
  gd.dot_acc = ga.dot_acc;
  gd.dot_out = ga.dot_out;
  gd.dot_scale = ga.dot_scale;
  const int3 nr = make_int3(norm_roll(roll[0], m), norm_roll(roll[1], m), norm_roll(roll[2], m));
  kern<<<mesh_grid(c, occ), BLOCK, smem, st>>>(bin_view(c), tp, nr, maps, mp, gd, (nr.z & 3) ? 1 : 0);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

}  // namespace pmf
