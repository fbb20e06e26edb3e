// pm_bin.cu -- a0: on-device counting sort of particles into mesh tiles (north_star: "Particles are
// sorted into cell tiles with an on-device counting/Morton sort").  Not in the paper; the build's own step.
//
// Default, single pass (k_bin_pass<2>): every tile owns a bucket of `capt` record slots (twice the mean load);
//   one read of the positions: cell coordinate (fp64-accurate, see cell_coord), slot claim in the tile's bucket
//   (warp-aggregated, order-preserving), record {ux, uy, uz, i} stored; claims beyond the bucket go to an
//   overflow list that k_ov_permute sorts by tile behind the buckets.  k_scan_* scan the overflow counts and
//   the work-item counts, k_items_bucketed writes the work items (tile, begin, end) of at most ITEM_MAX particles.
//   12N read + 16N written.
// PM_FLAG_BIN_TWOPASS (and N too large for 32-bit bucket indices): histogram (k_bin_pass<0>), scan, permute
//   (k_bin_pass<1>), k_items: 12N + 12N read, 16N written, 16 B/particle of workspace instead of 68.
#include "pm_internal.cuh"

namespace pmf {

struct BinGeom {
  int m, ntx, nty, ntz, xbl;
  int fast_tiles;    // m is a multiple of every tile edge: the box edge is a tile boundary (see tile_fast)
  float c_hi, c_lo;  // m / box split into two floats (c_hi + c_lo = m/box to ~2^-48)
  double inv_dx;     // m / box
};

// Cell coordinate u = x * m/L of one axis as (integer cell in [0, m), 26-bit fraction).
// SURVEY 7 "hard parts": the plain fp32 product is not accurate enough.  Fast path: error-free fp32 product
// p + e = x * (c_hi + c_lo) (FMA residual), p split into round(p) and an exact remainder -- fp32 pipes only, one
// float->int conversion.  Anything outside [0, m) (x outside [0, L), or rounded up to m) takes the fp64 path.
// Both binning passes call this same function, so they always agree on the tile of a particle.
__device__ __forceinline__ void cell_coord(float x, const BinGeom& g, int& cell, uint32_t& frac) {
  const float p = __fmul_rn(x, g.c_hi);
  const float e = __fmaf_rn(x, g.c_lo, __fmaf_rn(x, g.c_hi, -p));
  const float t = __fadd_rn(p, 12582912.0f);  // 1.5 * 2^23: the integer nearest to p sits in the low mantissa bits
  const float r = __fsub_rn(p, __fsub_rn(t, 12582912.0f));  // exact, in [-1/2, 1/2]
  const int fi = __float2int_rn(__fadd_rn(r, e) * (float)REC_ONE);
  cell = (__float_as_int(t) - 0x4B400000) + (fi >> REC_FRAC);
  frac = (uint32_t)fi & REC_MASK;
  if (!(fabsf(p) < 4.0e6f) || (unsigned)cell >= (unsigned)g.m) {  // rare: wrap in fp64
    double u = (double)x * g.inv_dx;
    const double dm = (double)g.m;
    u -= dm * floor(u / dm);
    if (!(u >= 0.0) || u >= dm) u = 0.0;  // non-finite input, or rounded up to m
    const double fl = floor(u);
    cell = (int)fl;
    uint32_t f = (uint32_t)__double2ll_rn((u - fl) * (double)REC_ONE);
    if (f >= REC_ONE) f = REC_ONE - 1u;
    frac = f;
  }
}

__device__ __forceinline__ uint32_t tile_and_local(float x, float y, float z, const BinGeom& g, uint32_t& fx,
                                                   uint32_t& fy, uint32_t& fz) {
  int cx, cy, cz;
  cell_coord(x, g, cx, fx);
  cell_coord(y, g, cy, fy);
  cell_coord(z, g, cz, fz);
  const int tx = cx / TX, ty = cy / TY, tz = cz / TZ;
  // (u_local + REC_BIAS) * 2^REC_FRAC
  fx |= (uint32_t)(cx - tx * TX + REC_BIAS) << REC_FRAC;
  fy |= (uint32_t)(cy - ty * TY + REC_BIAS) << REC_FRAC;
  fz |= (uint32_t)(cz - tz * TZ + REC_BIAS) << REC_FRAC;
  return tile_id(tx, ty, tz, g.nty, g.ntz, g.xbl);
}

__device__ __forceinline__ uint32_t tile_exact(float x, float y, float z, const BinGeom& g) {
  int cx, cy, cz;
  uint32_t f;
  cell_coord(x, g, cx, f);
  cell_coord(y, g, cy, f);
  cell_coord(z, g, cz, f);
  return tile_id(cx / TX, cy / TY, cz / TZ, g.nty, g.ntz, g.xbl);
}

// Histogram pass: only the tile is needed.  v = x * (m/L)/T is u/T to ~1e-5 tiles in plain fp32; unless v lies
// within 1e-3 of a tile boundary (or outside the box) floor(v) IS the tile the exact coordinate gives, and
// the pass skips the error-free product (it is issue-bound: ncu 70 % issue active, 40 % of HBM).  The rare
// boundary cases take the exact path, so both passes always agree.
__device__ __forceinline__ bool tile_fast(float x, float ct, int nt, int& t) {
  const float vm = __fmaf_rn(x, ct, -0.5f);
  const float tt = __fadd_rn(vm, 12582912.0f);  // 1.5 * 2^23: nearest integer to v - 1/2 in the low mantissa bits
  t = __float_as_int(tt) - 0x4B400000;
  const float r = __fsub_rn(vm, __fsub_rn(tt, 12582912.0f));  // v - (t + 1/2), in [-1/2, 1/2]
  return fabsf(r) < 0.499f && (unsigned)t < (unsigned)nt;
}
__device__ __forceinline__ uint32_t tile_only(float x, float y, float z, const BinGeom& g) {
  int tx, ty, tz;
  const bool ok = tile_fast(x, g.c_hi * (1.0f / TX), g.ntx, tx) & tile_fast(y, g.c_hi * (1.0f / TY), g.nty, ty) &
                  tile_fast(z, g.c_hi * (1.0f / TZ), g.ntz, tz);
  if (!ok || !g.fast_tiles) return tile_exact(x, y, z, g);
  return tile_id(tx, ty, tz, g.nty, g.ntz, g.xbl);
}

// The lanes of a warp hold 32 CONSECUTIVE particles.  Each run of equal keys elects its first lane, which
// performs ONE atomic for the run; a lane's slot is run base + rank in the run, so that a coherent input
// (Lagrangian order) keeps its order inside a tile -- the scatter / gather kernels rely on that for
// conflict-free shared-memory access.  Lanes whose key is NO_TILE take no slot.
struct Claim {
  int head;       // lane that performs the atomic of this lane's run
  uint32_t len;   // run length (meaningful on the head lane)
  uint32_t rank;  // this lane's position in its run
};
__device__ __forceinline__ Claim warp_runs(uint32_t key) {
  const unsigned lane = threadIdx.x & 31u;
  const uint32_t prev = __shfl_up_sync(0xffffffffu, key, 1);
  const unsigned heads = __ballot_sync(0xffffffffu, lane == 0 || key != prev);
  const unsigned le = heads & (0xffffffffu >> (31u - lane));  // heads at or below this lane
  const unsigned above = heads & ~(0xffffffffu >> (31u - lane));
  Claim c;
  c.head = 31 - __clz(le);
  c.len = (uint32_t)((above ? __ffs(above) - 1 : 32) - c.head);
  c.rank = lane - (unsigned)c.head;
  return c;
}

constexpr int BIN_BLOCK = 256;
constexpr int BIN_WARP_PART = 128;  // particles per warp and iteration (3 float4 per lane)
constexpr uint32_t NO_TILE = 0xffffffffu;

// Claim slots for K keys per lane at once: the K atomics of a lane are issued back to back and only then
// consumed, so their round trips to L2 overlap (issued one by one, each claim waited for the previous).
template <bool PERMUTE, int K>
__device__ __forceinline__ void claim_slots(uint32_t* __restrict__ counters, const uint32_t (&key)[K],
                                            uint32_t (&slot)[K]) {
  const unsigned lane = threadIdx.x & 31u;
  Claim c[K];
  uint32_t base[K];
#pragma unroll
  for (int k = 0; k < K; ++k) c[k] = warp_runs(key[k]);
#pragma unroll
  for (int k = 0; k < K; ++k) {
    base[k] = 0;
    if ((int)lane == c[k].head && key[k] != NO_TILE) {
      if (PERMUTE)
        base[k] = atomicAdd(&counters[key[k]], c[k].len);
      else
        atomicAdd(&counters[key[k]], c[k].len);  // histogram only: no return value (RED)
    }
  }
  if (PERMUTE) {
#pragma unroll
    for (int k = 0; k < K; ++k) slot[k] = __shfl_sync(0xffffffffu, base[k], c[k].head) + c[k].rank;
  }
}

// MODE 0: tile histogram (first pass of the two-pass path).  MODE 1: second pass of the two-pass path: claim
// a slot at tile_off[tile], store the record.  MODE 2: the single-pass ("bucketed") path: every tile owns a
// bucket of `capt` record slots at rec[tile * capt]; a particle whose claim lands beyond the bucket goes to the
// overflow list (record + tile id), which k_ov_permute sorts into rec[ov_base ...) afterwards.  No histogram
// and no second read of the positions: 12N read + 16N written instead of 24N + 16N.
// Positions are read as coalesced float4 (north_star "coalesced float4 position loads") and transposed
// through a warp-private shared-memory strip so that lane l handles particles 32k + l, k = 0..3; the next
// chunk's loads are in flight while the current one is processed.
struct Buckets {
  uint32_t capt;       // slots per tile bucket
  uint32_t* ov_count;  // overflow list length
  uint4* ov_rec;       // overflow records (unsorted)
  uint32_t* ov_tile;   // their tiles
};

// Overflow list space is reserved per WARP in chunks of OV_CHUNK entries (one atomic on the list counter per
// chunk, not per warp call: with half of the particles overflowing, config 4, two million same-address atomics
// were a millisecond of their own).  ov_pos / ov_left are warp-uniform.  Entries a warp reserves and does not
// use are holes: tile = NO_TILE, skipped by k_ov_permute.
constexpr uint32_t OV_CHUNK = 1024;

__device__ __forceinline__ void ov_fill_holes(const Buckets& bk, uint32_t ov_pos, uint32_t ov_left) {
  for (uint32_t j = threadIdx.x & 31u; j < ov_left; j += 32) bk.ov_tile[ov_pos + j] = NO_TILE;
}

template <int MODE>
__device__ __forceinline__ void put_record(uint4* __restrict__ rec, const Buckets& bk, uint32_t tile, uint32_t toff,
                                           uint32_t slot, bool valid, uint4 r, uint32_t& ov_pos, uint32_t& ov_left) {
  if (MODE == 1) {
    if (valid) rec[toff + slot] = r;
  } else if (MODE == 2) {
    const bool ov = valid && slot >= bk.capt;
    if (valid && !ov) rec[toff + slot] = r;
    const unsigned ovm = __ballot_sync(0xffffffffu, ov);
    if (ovm) {
      const unsigned lane = threadIdx.x & 31u;
      const uint32_t cnt = (uint32_t)__popc(ovm);
      if (cnt > ov_left) {  // warp-uniform: drop the rest of the chunk, reserve a new one
        ov_fill_holes(bk, ov_pos, ov_left);
        uint32_t base = 0;
        if (lane == 0) base = atomicAdd(bk.ov_count, OV_CHUNK);
        ov_pos = __shfl_sync(0xffffffffu, base, 0);
        ov_left = OV_CHUNK;
      }
      if (ov) {
        const uint32_t j = ov_pos + (uint32_t)__popc(ovm & ((1u << lane) - 1u));
        bk.ov_rec[j] = r;
        bk.ov_tile[j] = tile;
      }
      ov_pos += cnt;
      ov_left -= cnt;
    }
  }
}

template <int MODE>
__global__ void __launch_bounds__(BIN_BLOCK) k_bin_pass(const float* __restrict__ pos, int64_t n, BinGeom g,
                                                        uint32_t* __restrict__ counters,
                                                        const uint32_t* __restrict__ tile_off,
                                                        uint4* __restrict__ rec, int aligned,
                                                        float4* __restrict__ zfill, int64_t zn, int zq, Buckets bk) {
  constexpr bool PERMUTE = MODE != 0;
  __shared__ __align__(16) float s_strip[BIN_BLOCK / 32][BIN_WARP_PART * 3];
  const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  float* s = s_strip[warp];
  const int64_t nchunk = aligned ? n / BIN_WARP_PART : 0;
  const int64_t gwarp = (int64_t)blockIdx.x * (BIN_BLOCK / 32) + warp;
  const int64_t nwarps = (int64_t)gridDim.x * (BIN_BLOCK / 32);
  const float4* p4 = reinterpret_cast<const float4*>(pos);
  float4 a = make_float4(0.f, 0.f, 0.f, 0.f), b = a, c = a;
  uint32_t ov_pos = 0, ov_left = 0;  // this warp's reserved piece of the overflow list (MODE 2)
  if (gwarp < nchunk) {
    const float4* src = p4 + gwarp * (BIN_WARP_PART * 3 / 4);
    a = __ldcs(src + lane), b = __ldcs(src + 32 + lane), c = __ldcs(src + 64 + lane);
  }
  for (int64_t ch = gwarp; ch < nchunk; ch += nwarps) {
    reinterpret_cast<float4*>(s)[lane] = a;
    reinterpret_cast<float4*>(s)[32 + lane] = b;
    reinterpret_cast<float4*>(s)[64 + lane] = c;
    __syncwarp();
    if (ch + nwarps < nchunk) {
      const float4* src = p4 + (ch + nwarps) * (BIN_WARP_PART * 3 / 4);
      a = __ldcs(src + lane), b = __ldcs(src + 32 + lane), c = __ldcs(src + 64 + lane);
    }
    if (MODE != 1 && zfill) {  // zero-fill rider (see ensure_bins): chunk ch clears float4s [ch zq, (ch+1) zq)
      for (int j = (int)lane; j < zq; j += 32) {
        const int64_t idx = ch * zq + j;
        if (idx < zn) __stcs(zfill + idx, make_float4(0.f, 0.f, 0.f, 0.f));
      }
    }
    uint32_t tile[4], slot[4], fx[4], fy[4], fz[4], toff[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const int j = 32 * k + (int)lane;
      const float x = s[3 * j], y = s[3 * j + 1], z = s[3 * j + 2];
      fx[k] = fy[k] = fz[k] = 0;
      tile[k] = PERMUTE ? tile_and_local(x, y, z, g, fx[k], fy[k], fz[k]) : tile_only(x, y, z, g);
      if (MODE == 1) toff[k] = __ldg(tile_off + tile[k]);
      if (MODE == 2) toff[k] = tile[k] * bk.capt;
    }
    claim_slots<PERMUTE, 4>(counters, tile, slot);
    if (PERMUTE) {
#pragma unroll
      for (int k = 0; k < 4; ++k)
        put_record<MODE>(rec, bk, tile[k], toff[k], slot[k], true,
                         make_uint4(fx[k], fy[k], fz[k], (uint32_t)(ch * BIN_WARP_PART + 32 * k + (int)lane)), ov_pos,
                         ov_left);
    }
    __syncwarp();
  }
  // scalar tail (and the whole array when pos is not 16-byte aligned); whole warps stay in the loop
  const int64_t first = nchunk * BIN_WARP_PART;
  const int64_t rest = n - first;
  const int64_t rest_round = (rest + 31) / 32 * 32;
  for (int64_t j = gwarp * 32 + lane; j < rest_round; j += nwarps * 32) {
    const bool valid = j < rest;
    uint32_t fx = 0, fy = 0, fz = 0;
    uint32_t tile[1] = {NO_TILE}, slot[1] = {0};
    const int64_t i = first + j;
    if (valid) {
      const float x = pos[3 * i], y = pos[3 * i + 1], z = pos[3 * i + 2];
      tile[0] = PERMUTE ? tile_and_local(x, y, z, g, fx, fy, fz) : tile_only(x, y, z, g);
    }
    claim_slots<PERMUTE, 1>(counters, tile, slot);
    if (PERMUTE) {
      uint32_t toff = 0;
      if (valid) toff = MODE == 1 ? tile_off[tile[0]] : tile[0] * bk.capt;
      put_record<MODE>(rec, bk, tile[0], toff, slot[0], valid, make_uint4(fx, fy, fz, (uint32_t)i), ov_pos, ov_left);
    }
  }
  if (MODE == 2) ov_fill_holes(bk, ov_pos, ov_left);
}

// Overflow of the single-pass path: sort the overflow list by tile into rec[ov_base + ov_off[tile] ...).  The
// list was appended warp by warp, so consecutive entries mostly share a tile: one atomic per run of equal tiles
// (claim_slots), not per entry -- the dense tiles of a clustered input would otherwise serialise on a handful of
// cursor addresses.  Holes (NO_TILE) take no slot.
__global__ void __launch_bounds__(256) k_ov_permute(const uint32_t* __restrict__ ov_count,
                                                    const uint4* __restrict__ ov_rec,
                                                    const uint32_t* __restrict__ ov_tile,
                                                    const uint32_t* __restrict__ ov_off, uint32_t* __restrict__ ov_cur,
                                                    uint4* __restrict__ rec, uint32_t ov_base) {
  const uint32_t n = *ov_count;
  const uint32_t lane = threadIdx.x & 31u;
  const uint32_t stride = gridDim.x * blockDim.x;
  for (uint32_t b = blockIdx.x * blockDim.x + (threadIdx.x & ~31u); b < n; b += stride) {  // warp-uniform
    const uint32_t j = b + lane;
    uint32_t key[1] = {NO_TILE}, slot[1] = {0};
    if (j < n) key[0] = ov_tile[j];
    claim_slots<true, 1>(ov_cur, key, slot);
    if (key[0] != NO_TILE) rec[ov_base + ov_off[key[0]] + slot[0]] = ov_rec[j];
  }
}

// ---- exclusive scan of (count, nchunks) over the tiles: reduce / scan-of-partials / rescan ----------
constexpr int SCAN_T = 1024, SCAN_E = 4, SCAN_B = SCAN_T * SCAN_E;

__device__ __forceinline__ uint32_t nchunks_of(uint32_t cnt) { return (cnt + ITEM_MAX - 1) / ITEM_MAX; }
// What the scan sums per tile.  Two-pass path (capt = 0): (particles, work items).  Single-pass path: (overflow
// particles, work items of the bucket + work items of the overflow segment).
__device__ __forceinline__ uint2 scan_pair(uint32_t cnt, uint32_t capt) {
  if (capt == 0) return make_uint2(cnt, nchunks_of(cnt));
  const uint32_t ov = cnt > capt ? cnt - capt : 0u;
  return make_uint2(ov, nchunks_of(cnt - ov) + nchunks_of(ov));
}

__device__ uint2 block_exclusive_scan(uint2 v, uint2* total) {  // blockDim.x == SCAN_T
  __shared__ uint2 wsum[32];
  const unsigned lane = threadIdx.x & 31u, wid = threadIdx.x >> 5;
  uint2 incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const uint32_t a = __shfl_up_sync(0xffffffffu, incl.x, d), b = __shfl_up_sync(0xffffffffu, incl.y, d);
    if ((int)lane >= d) { incl.x += a; incl.y += b; }
  }
  if (lane == 31) wsum[wid] = incl;
  __syncthreads();
  if (wid == 0) {
    uint2 w = wsum[lane];
    uint2 wi = w;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const uint32_t a = __shfl_up_sync(0xffffffffu, wi.x, d), b = __shfl_up_sync(0xffffffffu, wi.y, d);
      if ((int)lane >= d) { wi.x += a; wi.y += b; }
    }
    wsum[lane] = make_uint2(wi.x - w.x, wi.y - w.y);
    if (lane == 31 && total) *total = wi;
  }
  __syncthreads();
  const uint2 off = wsum[wid];
  __syncthreads();
  return make_uint2(off.x + incl.x - v.x, off.y + incl.y - v.y);
}

__global__ void __launch_bounds__(SCAN_T) k_scan_reduce(const uint32_t* __restrict__ cnt, int n,
                                                        uint2* __restrict__ partial, uint32_t capt) {
  __shared__ uint2 tot;
  uint2 s = make_uint2(0, 0);
  const int base = blockIdx.x * SCAN_B + threadIdx.x * SCAN_E;
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e)
    if (base + e < n) { const uint2 v = scan_pair(cnt[base + e], capt); s.x += v.x; s.y += v.y; }
  block_exclusive_scan(s, &tot);
  if (threadIdx.x == 0) partial[blockIdx.x] = tot;
}

__global__ void __launch_bounds__(SCAN_T) k_scan_partials(uint2* __restrict__ partial, int nb,
                                                          uint32_t* __restrict__ tile_off,
                                                          uint32_t* __restrict__ item_off, int ntiles,
                                                          uint32_t* __restrict__ nitems) {
  __shared__ uint2 tot;
  uint2 carry = make_uint2(0, 0);
  for (int b0 = 0; b0 < nb; b0 += SCAN_T) {
    const int i = b0 + threadIdx.x;
    const uint2 v = i < nb ? partial[i] : make_uint2(0, 0);
    const uint2 ex = block_exclusive_scan(v, &tot);
    if (i < nb) partial[i] = make_uint2(ex.x + carry.x, ex.y + carry.y);
    carry.x += tot.x;
    carry.y += tot.y;
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    tile_off[ntiles] = carry.x;
    item_off[ntiles] = carry.y;
    *nitems = carry.y;
  }
}

__global__ void __launch_bounds__(SCAN_T) k_scan_final(uint32_t* __restrict__ cnt, int n,
                                                       const uint2* __restrict__ partial,
                                                       uint32_t* __restrict__ tile_off,
                                                       uint32_t* __restrict__ item_off, uint32_t capt) {
  const int base = blockIdx.x * SCAN_B + threadIdx.x * SCAN_E;
  uint2 c[SCAN_E];
  uint2 s = make_uint2(0, 0);
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e) {
    c[e] = base + e < n ? scan_pair(cnt[base + e], capt) : make_uint2(0u, 0u);
    s.x += c[e].x;
    s.y += c[e].y;
  }
  uint2 ex = block_exclusive_scan(s, nullptr);
  const uint2 p = partial[blockIdx.x];
  ex.x += p.x;
  ex.y += p.y;
#pragma unroll
  for (int e = 0; e < SCAN_E; ++e)
    if (base + e < n) {
      tile_off[base + e] = ex.x;
      item_off[base + e] = ex.y;
      ex.x += c[e].x;
      ex.y += c[e].y;
      if (capt == 0) cnt[base + e] = 0u;  // becomes the cursor of pass 2 (the single-pass path keeps the counts)
    }
}

__global__ void __launch_bounds__(256) k_items(const uint32_t* __restrict__ tile_off,
                                               const uint32_t* __restrict__ item_off, int ntiles, int nty, int ntz,
                                               int xbl, WorkItem* __restrict__ items) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  const uint32_t b = tile_off[t], e = tile_off[t + 1];
  uint32_t it = item_off[t];
  // inverse of tile_id()
  const int tz = t % ntz;
  int r = t / ntz;
  const int xl = r & ((1 << xbl) - 1);
  r >>= xbl;
  const int ty = r % nty, tx = ((r / nty) << xbl) | xl;
  const uint32_t txyz = (uint32_t)tx | ((uint32_t)ty << 10) | ((uint32_t)tz << 20);
  const uint32_t k = nchunks_of(e - b);
  const uint32_t per = k ? (e - b + k - 1) / k : 0;  // even split: no tiny remainder items
  for (uint32_t j = 0; j < k; ++j) {  // exactly the k slots the scan reserved (a slot may stay empty)
    WorkItem w;
    w.tile = (uint32_t)t | (k == 1 ? 0x80000000u : 0u);  // single item: exclusive interior (see k_scatter_warp)
    w.begin = min(b + j * per, e);
    w.end = min(w.begin + per, e);
    w.txyz = txyz;
    items[it++] = w;
  }
}

// Work items of the single-pass path: the tile's bucket rec[t capt, + min(cnt, capt)) and, if it overflowed,
// its overflow segment rec[ov_base + ov_off[t], + cnt - capt).
__global__ void __launch_bounds__(256) k_items_bucketed(const uint32_t* __restrict__ cnt,
                                                        const uint32_t* __restrict__ ov_off,
                                                        const uint32_t* __restrict__ item_off, int ntiles, int nty,
                                                        int ntz, int xbl, uint32_t capt, uint32_t ov_base,
                                                        WorkItem* __restrict__ items) {
  const int t = blockIdx.x * blockDim.x + threadIdx.x;
  if (t >= ntiles) return;
  const uint32_t c = cnt[t];
  const uint32_t ov = c > capt ? c - capt : 0u;
  uint32_t it = item_off[t];
  const int tz = t % ntz;
  int r = t / ntz;
  const int xl = r & ((1 << xbl) - 1);
  r >>= xbl;
  const int ty = r % nty, tx = ((r / nty) << xbl) | xl;
  const uint32_t txyz = (uint32_t)tx | ((uint32_t)ty << 10) | ((uint32_t)tz << 20);
  for (int seg = 0; seg < 2; ++seg) {
    const uint32_t b = seg == 0 ? (uint32_t)t * capt : ov_base + ov_off[t];
    const uint32_t e = b + (seg == 0 ? c - ov : ov);
    const uint32_t k = nchunks_of(e - b);
    const uint32_t per = k ? (e - b + k - 1) / k : 0;
    for (uint32_t j = 0; j < k; ++j) {
      WorkItem w;
      w.tile = (uint32_t)t | ((k == 1 && ov == 0) ? 0x80000000u : 0u);  // the tile's only item
      w.begin = min(b + j * per, e);
      w.end = min(w.begin + per, e);
      w.txyz = txyz;
      items[it++] = w;
    }
  }
}

BinView bin_view(const Ctx* c) {
  BinView v;
  v.rec = c->rec;
  v.items = c->items;
  v.nitems = c->nitems;
  v.sched = c->sched;
  v.m = c->mg;
  v.ntx = c->ntx;
  v.nty = c->nty;
  v.ntz = c->ntz;
  v.xbl = c->xbl;
  return v;
}

int ensure_bins(Ctx* c, const float* pos, int64_t N, cudaStream_t st, bool pin) {
  if (!pos) return fail(c, PM_EINVAL, "pos is NULL");
  if (N < 0 || N > c->cap) return fail(c, PM_EINVAL, "N = %lld outside [0, max_particles = %lld]", (long long)N, (long long)c->cap);
  if (!pin && c->bin_valid && c->bin_pinned && c->bin_pos == pos && c->bin_n == N) return PM_OK;
  c->bin_valid = false;
  c->g_valid = false;  // force meshes of other records
  BinGeom g;
  g.m = c->mg;
  g.ntx = c->ntx;
  g.nty = c->nty;
  g.ntz = c->ntz;
  g.xbl = c->xbl;
  g.fast_tiles = (c->mg % TX == 0 && c->mg % TY == 0 && c->mg % TZ == 0) ? 1 : 0;
  g.inv_dx = (double)c->mg / c->p.box;
  g.c_hi = (float)g.inv_dx;
  g.c_lo = (float)(g.inv_dx - (double)g.c_hi);
  const int nt = c->ntiles;
  const int nb = (nt + SCAN_B - 1) / SCAN_B;
  uint2* partial = reinterpret_cast<uint2*>(c->scan_tmp);
  PM_CUDA(c, cudaMemsetAsync(c->tile_cnt, 0, sizeof(uint32_t) * (size_t)nt, st));
  const int aligned = ((reinterpret_cast<uintptr_t>(pos) & 15u) == 0) ? 1 : 0;
  // persistent grid: resident CTAs per SM (register-limited) x SMs, capped by the work
  const int64_t work = aligned ? (N + BIN_WARP_PART - 1) / BIN_WARP_PART : (N + 31) / 32;  // warp iterations
  int grid = (int)((work + BIN_BLOCK / 32 - 1) / (BIN_BLOCK / 32));
  if (grid < 1) grid = 1;
  int grid0 = grid;  // the histogram pass needs fewer registers: its own residency
  if (grid > c->num_sms * c->bin_occ) grid = c->num_sms * c->bin_occ;
  if (grid0 > c->num_sms * c->bin_occ0) grid0 = c->num_sms * c->bin_occ0;
  // Zero-fill rider: the first pass over the positions also clears the assignment mesh pm_force needs next
  // (one 16-byte store per lane and iteration at G = N), which saves the separate cudaMemset pass and its
  // launch; the binning passes run at 40-80 % of the HBM roofline, so the stores fit beside their traffic.
  float4* zfill = nullptr;
  int64_t zn = 0, nchunk = aligned ? N / BIN_WARP_PART : 0;
  int zq = 0;
  if (c->zero_req && nchunk > 0 && (c->zero_req_bytes & 15u) == 0 &&
      (int64_t)(c->zero_req_bytes / 16) <= nchunk * 4096) {
    zfill = reinterpret_cast<float4*>(c->zero_req);
    zn = (int64_t)(c->zero_req_bytes / 16);
    zq = (int)((zn + nchunk - 1) / nchunk);
    c->zero_done = true;
  }
  c->zero_req = nullptr;
  Buckets bk;
  bk.capt = c->bin_capt;
  bk.ov_count = c->ov_count;
  bk.ov_rec = c->ov_rec;
  bk.ov_tile = c->ov_tile;
  if (c->bin_capt) {
    // single pass: bucketed permute, scan of the overflow counts, work items, overflow sort
    PM_CUDA(c, cudaMemsetAsync(c->ov_count, 0, sizeof(uint32_t), st));
    PM_CUDA(c, cudaMemsetAsync(c->ov_cur, 0, sizeof(uint32_t) * (size_t)nt, st));
    if (N > 0)
      k_bin_pass<2><<<grid, BIN_BLOCK, 0, st>>>(pos, N, g, c->tile_cnt, nullptr, c->rec, aligned, zfill, zn, zq, bk);
    k_scan_reduce<<<nb, SCAN_T, 0, st>>>(c->tile_cnt, nt, partial, bk.capt);
    k_scan_partials<<<1, SCAN_T, 0, st>>>(partial, nb, c->tile_off, c->item_off, nt, c->nitems);
    k_scan_final<<<nb, SCAN_T, 0, st>>>(c->tile_cnt, nt, partial, c->tile_off, c->item_off, bk.capt);
    k_items_bucketed<<<(nt + 255) / 256, 256, 0, st>>>(c->tile_cnt, c->tile_off, c->item_off, nt, c->nty, c->ntz,
                                                       c->xbl, bk.capt, c->ov_base, c->items);
    k_ov_permute<<<c->num_sms * 4, 256, 0, st>>>(c->ov_count, c->ov_rec, c->ov_tile, c->tile_off, c->ov_cur, c->rec,
                                                 c->ov_base);
    count_launch(c, N > 0 ? 6 : 5);
  } else {
    if (N > 0)
      k_bin_pass<0><<<grid0, BIN_BLOCK, 0, st>>>(pos, N, g, c->tile_cnt, nullptr, nullptr, aligned, zfill, zn, zq, bk);
    k_scan_reduce<<<nb, SCAN_T, 0, st>>>(c->tile_cnt, nt, partial, 0u);
    k_scan_partials<<<1, SCAN_T, 0, st>>>(partial, nb, c->tile_off, c->item_off, nt, c->nitems);
    k_scan_final<<<nb, SCAN_T, 0, st>>>(c->tile_cnt, nt, partial, c->tile_off, c->item_off, 0u);
    if (N > 0)
      k_bin_pass<1><<<grid, BIN_BLOCK, 0, st>>>(pos, N, g, c->tile_cnt, c->tile_off, c->rec, aligned, nullptr, 0, 0, bk);
    k_items<<<(nt + 255) / 256, 256, 0, st>>>(c->tile_off, c->item_off, nt, c->nty, c->ntz, c->xbl, c->items);
    count_launch(c, N > 0 ? 6 : 4);
  }
  PM_CUDA(c, cudaGetLastError());
  c->bin_valid = true;
  c->bin_pos = pos;
  c->bin_n = N;
  c->bin_pinned = pin;
  return PM_OK;
}

int bin_occupancy(int pass) {
  int o = 0;
  if (pass == 0) {
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&o, k_bin_pass<0>, BIN_BLOCK, 0);
  } else {
    int a = 0, b = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&a, k_bin_pass<1>, BIN_BLOCK, 0);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b, k_bin_pass<2>, BIN_BLOCK, 0);
    o = a < b ? a : b;
  }
  return o < 1 ? 1 : o;
}

}  // namespace pmf

extern "C" int pm_bin(pm_ctx* ctx, const float* pos, int64_t N, void* stream) {
  if (!ctx) return PM_EINVAL;
  const int rc = pmf::enter_device(pmf::C(ctx));
  if (rc != PM_OK) return rc;
  return pmf::ensure_bins(pmf::C(ctx), pos, N, (cudaStream_t)stream, true);
}
