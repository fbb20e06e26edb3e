// pm_xfft.cu -- a2-a4 / a7 / a10 fused along x: the x-direction passes of the forward and inverse 3-D FFTs and the
// Fourier-space kernel (K3, K6, and its transpose) in ONE kernel.
//
// The 3-D transforms are split as (y,z) planes x lines.  cuFFT does the batched 2-D (y,z) transforms (library
// call, "FFT"); this kernel then takes, for 8 neighbouring (y,z) columns at a time, the whole x line
// into shared memory, runs the forward x-FFT, applies the Green's function / gradient symbols / deconvolution /
// interlace combine of pm_kspace.cu (Tables 1-2) and runs the inverse x-FFTs (two of them: the y
// and z gradient symbols are constant along x, so those two components share one inverse transform), so that
// the spectrum is read once and the three force spectra are written once.  Unfused, the same work is five more
// passes over the data: forward x pass (read + write), k-space kernel (read, 3 writes), three inverse x passes
// (read + write each): 6.4 GB instead of 2.1 GB at 512^3.
//
// FFT: in-place mixed-radix (8 / 16) Cooley-Tukey in shared memory.  Forward = decimation in frequency (natural
// order in, digit-reversed out), inverse = decimation in time with the stages in reverse order (digit-reversed in,
// natural out), so no reordering pass is needed: the pointwise kernel maps a position to its frequency.
// Unnormalised both ways, like cuFFT; the 1/m^3 is folded into coeff_eff by the caller.
// Built for m = 64 ... 1024, powers of two; other sizes take the unfused path (cuFFT 3-D + pm_kspace.cu).
#include <math.h>

#include <vector>

#include "pm_internal.cuh"

namespace pmf {

constexpr int XC = 8;    // (y,z) columns per CTA: 64 contiguous bytes of every x plane
#ifndef PMF_XEPT
#define PMF_XEPT 16  // 8 (512 threads, 2 CTAs/SM at m = 512) was measured: 0.85 ms instead of 0.83 ms
#endif
#ifndef PMF_XTW_DERIVE
#define PMF_XTW_DERIVE 1
#endif
constexpr int XEPT = PMF_XEPT; // elements per thread -> N * XC / XEPT threads per CTA

__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
__device__ __forceinline__ float2 cmulx(float2 a, float2 b) {
  return make_float2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x);
}
__device__ __forceinline__ float2 cmulc(float2 a, float2 b) {  // a * conj(b)
  return make_float2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
// multiply by SIGN * i  (SIGN = -1: forward transform, e^{-2 pi i/4} = -i; SIGN = +1: inverse)
template <int SIGN>
__device__ __forceinline__ float2 mul_i(float2 a) {
  return SIGN < 0 ? make_float2(a.y, -a.x) : make_float2(-a.y, a.x);
}

// ---- small DFTs in registers, X_k = sum_n x_n e^{SIGN 2 pi i n k / R}, natural order in and out ---------
template <int SIGN>
__device__ __forceinline__ void dft4(float2& a0, float2& a1, float2& a2, float2& a3) {
  const float2 t0 = cadd(a0, a2), t1 = csub(a0, a2), t2 = cadd(a1, a3), t3 = mul_i<SIGN>(csub(a1, a3));
  a0 = cadd(t0, t2);
  a2 = csub(t0, t2);
  a1 = cadd(t1, t3);
  a3 = csub(t1, t3);
}

template <int R, int SIGN>
struct Dft;

template <int SIGN>
struct Dft<5, SIGN> {  // the upsampled NUFFT grids sigma = 5/4: m_f = 5 * 2^k
  static __device__ __forceinline__ void run(float2 (&v)[5]) {
    constexpr float c1 = 0.30901699437494742f, c2 = -0.80901699437494742f;  // cos(2 pi / 5), cos(4 pi / 5)
    constexpr float s1 = 0.95105651629515357f, s2 = 0.58778525229247313f;   // sin(2 pi / 5), sin(4 pi / 5)
    const float2 t1 = cadd(v[1], v[4]), t2 = cadd(v[2], v[3]), t3 = csub(v[1], v[4]), t4 = csub(v[2], v[3]);
    const float2 x0 = v[0];
    const float2 m1 = make_float2(x0.x + c1 * t1.x + c2 * t2.x, x0.y + c1 * t1.y + c2 * t2.y);
    const float2 m2 = make_float2(x0.x + c2 * t1.x + c1 * t2.x, x0.y + c2 * t1.y + c1 * t2.y);
    const float2 n1 = mul_i<SIGN>(make_float2(s1 * t3.x + s2 * t4.x, s1 * t3.y + s2 * t4.y));  // SIGN i (s1 t3 + s2 t4)
    const float2 n2 = mul_i<SIGN>(make_float2(s2 * t3.x - s1 * t4.x, s2 * t3.y - s1 * t4.y));
    v[0] = make_float2(x0.x + t1.x + t2.x, x0.y + t1.y + t2.y);
    v[1] = cadd(m1, n1);
    v[4] = csub(m1, n1);
    v[2] = cadd(m2, n2);
    v[3] = csub(m2, n2);
  }
};

template <int SIGN>
struct Dft<8, SIGN> {
  static __device__ __forceinline__ void run(float2 (&v)[8]) {
    // even / odd samples: X_k = E_k + W8^k O_k, X_{k+4} = E_k - W8^k O_k
    dft4<SIGN>(v[0], v[2], v[4], v[6]);
    dft4<SIGN>(v[1], v[3], v[5], v[7]);
    constexpr float h = 0.70710678118654752f;
    // W8^k = e^{SIGN 2 pi i k / 8}
    const float2 o0 = v[1];
    const float2 o1 = make_float2(h * (v[3].x - SIGN * v[3].y), h * (v[3].y + SIGN * v[3].x));   // * (1 + SIGN i)/sqrt2
    const float2 o2 = mul_i<SIGN>(v[5]);
    const float2 o3 = make_float2(h * (-v[7].x - SIGN * v[7].y), h * (-v[7].y + SIGN * v[7].x)); // * (-1 + SIGN i)/sqrt2
    const float2 e0 = v[0], e1 = v[2], e2 = v[4], e3 = v[6];
    v[0] = cadd(e0, o0);
    v[4] = csub(e0, o0);
    v[1] = cadd(e1, o1);
    v[5] = csub(e1, o1);
    v[2] = cadd(e2, o2);
    v[6] = csub(e2, o2);
    v[3] = cadd(e3, o3);
    v[7] = csub(e3, o3);
  }
};

template <int SIGN>
struct Dft<16, SIGN> {
  static __device__ __forceinline__ void run(float2 (&v)[16]) {
    // n = 4 n' + s: A_s = DFT4(x_s, x_{s+4}, x_{s+8}, x_{s+12}); X_{k+4q} = sum_s W4^{sq} (W16^{sk} A_s[k])
#pragma unroll
    for (int s = 0; s < 4; ++s) dft4<SIGN>(v[s], v[s + 4], v[s + 8], v[s + 12]);  // A_s[k] now in v[s + 4k]
    constexpr float c1 = 0.92387953251128674f, s1 = 0.38268343236508977f, h = 0.70710678118654752f;
    // W16^j = cos(pi j / 8) + SIGN i sin(pi j / 8), j = s k in {1, 2, 3, 4, 6, 9}
    const float2 w1 = make_float2(c1, SIGN * s1), w2 = make_float2(h, SIGN * h), w3 = make_float2(s1, SIGN * c1);
    const float2 w6 = make_float2(-h, SIGN * h), w9 = make_float2(-c1, -SIGN * s1);
    v[1 + 4] = cmulx(v[1 + 4], w1);    // s = 1, k = 1
    v[1 + 8] = cmulx(v[1 + 8], w2);    // s = 1, k = 2
    v[1 + 12] = cmulx(v[1 + 12], w3);  // s = 1, k = 3
    v[2 + 4] = cmulx(v[2 + 4], w2);    // s = 2, k = 1
    v[2 + 8] = mul_i<SIGN>(v[2 + 8]);  // s = 2, k = 2: W16^4 = SIGN i
    v[2 + 12] = cmulx(v[2 + 12], w6);  // s = 2, k = 3
    v[3 + 4] = cmulx(v[3 + 4], w3);    // s = 3, k = 1
    v[3 + 8] = cmulx(v[3 + 8], w6);    // s = 3, k = 2
    v[3 + 12] = cmulx(v[3 + 12], w9);  // s = 3, k = 3
#pragma unroll
    for (int k = 0; k < 4; ++k) dft4<SIGN>(v[4 * k], v[4 * k + 1], v[4 * k + 2], v[4 * k + 3]);  // over s -> q
    // v[4k + q] = X_{k + 4q}: transpose to natural order
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
      for (int q = k + 1; q < 4; ++q) {
        const float2 t = v[4 * k + q];
        v[4 * k + q] = v[4 * q + k];
        v[4 * q + k] = t;
      }
  }
};

// ---- shared-memory line layout and the FFT stages -----------------------------------------------------------
// Element (x position p, column c) sits at float2 index p * XC + c + 8 * (p / 8): a row of 8 columns is half of
// the 32 banks; the padding puts rows p and p + 8 (last stage) in different halves, rows p and p + 1 are anyway.
__device__ __forceinline__ int sidx(int p, int c) { return 9 * p - (p & 7) + c; }  // = 8 p + c + 8 (p / 8), XC = 8
template <int N>
constexpr int xfft_smem_elems() { return N * XC + (N / 8) * 8; }

template <int N>
struct Radices;  // N = r0 * r1 * r2
template <> struct Radices<64>   { static constexpr int r0 = 8,  r1 = 8,  r2 = 1; };
template <> struct Radices<128>  { static constexpr int r0 = 16, r1 = 8,  r2 = 1; };
template <> struct Radices<256>  { static constexpr int r0 = 16, r1 = 16, r2 = 1; };
template <> struct Radices<512>  { static constexpr int r0 = 8,  r1 = 8,  r2 = 8; };
template <> struct Radices<1024> { static constexpr int r0 = 16, r1 = 8,  r2 = 8; };
template <> struct Radices<320>  { static constexpr int r0 = 5,  r1 = 8,  r2 = 8; };   // 5/4 * 256
template <> struct Radices<640>  { static constexpr int r0 = 5,  r1 = 16, r2 = 8; };   // 5/4 * 512

// One radix-R stage over sub-transforms of size S (M = S / R butterflies each).  tw[k] = e^{-2 pi i k / N}.
//   forward (DIF): y = DFT_R(x), y_q *= W_S^{jq};      inverse (DIT): x_r *= conj(W_S)^{jr}, y = IDFT_R(x)
// ld(p, c) / st(p, c, v) read and write element (position p, column c): the shared-memory line for the inner
// stages; the first load and the last store of a transform go straight from / to global memory or carry the
// pointwise k-space factors, which saves four of the nine passes over shared memory per transform (the kernel is
// bound by shared-memory bandwidth).  A thread's column c is the same in every stage.
template <int N, int R, int S, bool INV, class Ld, class St>
__device__ __forceinline__ void xfft_stage(const float2* __restrict__ tw, int tid, Ld ld, St st) {
  constexpr int M = S / R, NB = N * XC / R, NT = N * XC / XEPT;
#pragma unroll
  for (int b = tid; b < NB; b += NT) {
    const int c = b % XC, bf = b / XC, blk = bf / M, j = bf % M;
    const int p0 = blk * S + j;
    float2 v[R];
#pragma unroll
    for (int r = 0; r < R; ++r) v[r] = ld(p0 + r * M, c);
    // twiddles W^{j r}, r = 1 .. R-1: the powers of two are loaded, the others are products of two of them (one
    // rounding more, ~1e-7): 3 instead of 7 table loads per radix-8 butterfly -- the kernel is bound by the
    // load/store pipe (ncu: 64 % busy, a third of its instructions in these stages were twiddle loads).
    float2 w[R];
    if (M > 1) {  // M = 1: j = 0, every twiddle is 1
#pragma unroll
      for (int r = 1; r < R; r <<= 1) w[r] = __ldg(tw + (N / S) * j * r);
#if PMF_XTW_DERIVE
#pragma unroll
      for (int r = 3; r < R; ++r)
        if (r & (r - 1)) {  // not a power of two: highest set bit times the rest
          int hb = 1;
          while (hb * 2 <= r) hb *= 2;
          w[r] = cmulx(w[hb], w[r - hb]);
        }
#else
#pragma unroll
      for (int r = 3; r < R; ++r)
        if (r & (r - 1)) w[r] = __ldg(tw + (N / S) * j * r);
#endif
    }
    if (INV) {
      if (M > 1)
#pragma unroll
        for (int r = 1; r < R; ++r) v[r] = cmulc(v[r], w[r]);
      Dft<R, 1>::run(v);
    } else {
      Dft<R, -1>::run(v);
      if (M > 1)
#pragma unroll
        for (int q = 1; q < R; ++q) v[q] = cmulx(v[q], w[q]);
    }
#pragma unroll
    for (int q = 0; q < R; ++q) st(p0 + q * M, c, v[q]);
  }
  __syncthreads();
}

// A whole transform of the line in s: `first` loads the input of the first stage, `last` stores the output of
// the last stage (forward: element at position p holds frequency xfft_freq(p); inverse: natural order).
template <int N, bool INV, class Ld, class St>
__device__ __forceinline__ void xfft_line(float2* s, const float2* __restrict__ tw, int tid, Ld first, St last) {
  using Rd = Radices<N>;
  constexpr int S1 = N / Rd::r0, S2 = S1 / Rd::r1;
  constexpr bool three = Rd::r2 > 1;
  constexpr int R2 = three ? Rd::r2 : 8, S2e = three ? S2 : 8;  // (a valid, unused instantiation when r2 = 1)
  auto lds = [s](int p, int c) { return s[sidx(p, c)]; };
  auto sts = [s](int p, int c, float2 v) { s[sidx(p, c)] = v; };
  if (!INV) {
    xfft_stage<N, Rd::r0, N, false>(tw, tid, first, sts);
    if (three) {
      xfft_stage<N, Rd::r1, S1, false>(tw, tid, lds, sts);
      xfft_stage<N, R2, S2e, false>(tw, tid, lds, last);
    } else {
      xfft_stage<N, Rd::r1, S1, false>(tw, tid, lds, last);
    }
  } else {
    if (three) {
      xfft_stage<N, R2, S2e, true>(tw, tid, first, sts);
      xfft_stage<N, Rd::r1, S1, true>(tw, tid, lds, sts);
    } else {
      xfft_stage<N, Rd::r1, S1, true>(tw, tid, first, sts);
    }
    xfft_stage<N, Rd::r0, N, true>(tw, tid, lds, last);
  }
}

// frequency index held at position p after the forward (DIF) stages: p = q0 * (N/r0) + q1 * (N/(r0 r1)) + q2,
// k = q0 + r0 * (q1 + r1 * q2)
template <int N>
__device__ __forceinline__ int xfft_freq(int p) {
  using Rd = Radices<N>;
  constexpr int S1 = N / Rd::r0, S2 = S1 / Rd::r1;
  const int q0 = p / S1, rem = p - q0 * S1, q1 = rem / S2, q2 = rem - q1 * S2;
  return q0 + Rd::r0 * (q1 + Rd::r1 * q2);
}

struct XTabs {
  const double *grad, *lap, *win, *pc, *ps;  // per-axis symbol tables of pm_kspace.cu (column factors, once per thread)
  const float4* sym;                         // the same along the line, fp32: {lap, win, grad, 0} per index
  const float2* ph;                          // {pc, ps} per index
  const float2* tw;                          // e^{-2 pi i k / m}, k = 0 .. m-1
  int m, hz;
  int64_t ncol;                              // m * hz columns per x plane
};

// One CTA: XC consecutive columns q = iy * hz + iz of the (y,z) plane, all m values of x.
//   MODE 0 (force):     in0 (, in1 = second interlaced grid) -> out0..2 = x-inverse of S_a(n) dhat(n)
//   MODE 1 (transpose): in0..2 -> out0 (, out1) = x-inverse of sum_a conj(S_a) ghat_a
//   MODE 2 (potential): in0 (, in1) -> out0 = x-inverse of green(n) dhat(n): no gradient symbol -- the gradient is
//                       applied in real space (PM_FLAG_GRAD_REAL, pm_stencil.cu) or by the interpolation kernel
//                       (PM_FLAG_KERNEL_GRAD)
// Every input is the (y,z)-transformed, x-untransformed spectrum [x][y][hz]; every output likewise.
template <int N, int MODE>
__global__ void __launch_bounds__(N* XC / XEPT, N <= 512 ? (XEPT >= 16 ? 3 : 2) : 1) k_xfft_kspace(XTabs t, const float2* __restrict__ in0,
                                                               const float2* __restrict__ in1,
                                                               const float2* __restrict__ in2,
                                                               float2* __restrict__ out0, float2* __restrict__ out1,
                                                               float2* __restrict__ out2, double coeff_eff) {
  constexpr int SE = xfft_smem_elems<N>();
  extern __shared__ __align__(16) float2 s_x[];
  float2* s_w = s_x;        // work line: FFT in place
  float2* s_a = s_x + SE;   // MODE 0: green * dhat;  MODE 1: accumulated q
  const int tid = threadIdx.x;
  const int c = tid % XC;   // this thread's column in every pointwise loop (NT is a multiple of XC)
  const int64_t q = (int64_t)blockIdx.x * XC + c;
  const bool live = q < t.ncol;
  const int iy = live ? (int)(q / t.hz) : 0, iz = live ? (int)(q - (int64_t)iy * t.hz) : 0;
  const size_t plane = (size_t)t.ncol;

  // global memory as the first load / last store of a transform (64 contiguous bytes per x plane and CTA)
  auto gld = [&](const float2* __restrict__ src) {
    return [=](int p, int) { return live ? __ldcs(src + (size_t)p * plane + q) : make_float2(0.f, 0.f); };
  };
  auto gst = [&](float2* __restrict__ dst) {
    return [=](int p, int, float2 v) {
      if (live) dst[(size_t)p * plane + q] = v;
    };
  };

  // column factors
  const double lyz = t.lap[iy] + t.lap[iz], wyz = t.win[iy] * t.win[iz];
  const float dyv = (float)t.grad[iy], dzv = (float)t.grad[iz];
  const double pcyz = t.pc[iy] * t.pc[iz] - t.ps[iy] * t.ps[iz], psyz = t.pc[iy] * t.ps[iz] + t.ps[iy] * t.pc[iz];

  // NUFFT: the modes at or above the particle Nyquist are dropped (their window entry is 0, R8), which makes green_of
  // zero along the whole line.  A CTA whose columns are all dropped -- three quarters of them at sigma = 2 -- has
  // nothing to transform: its outputs are zero (cfg3: 7.5 -> 5.0 ms for this kernel).
  if (__syncthreads_and(!live || wyz == 0.0)) {
    constexpr int NT = N * XC / XEPT;
    const float2 zero = make_float2(0.f, 0.f);
    if (live)
      for (int p = tid / XC; p < N; p += NT / XC) {
        const size_t o = (size_t)p * plane + q;
        out0[o] = zero;
        if (MODE == 0) out1[o] = zero, out2[o] = zero;
        if (MODE == 1 && out1 != nullptr) out1[o] = zero;
      }
    return;
  }

  // coeff / (Lap * window); 0 at n = 0 and for dropped modes.  The column part of the symbols is summed in fp64
  // once per thread; along the line everything is fp32 (the result is an fp32 factor anyway; the fp64 adds,
  // multiplies and the divide per mode were a quarter of the kernel's stall samples).
  const float coeff_f = (float)coeff_eff, lyz_f = (float)lyz, wyz_f = (float)wyz;
  const float pcyz_f = (float)pcyz, psyz_f = (float)psyz;
  auto green_of = [&](int kx) -> float {
    const float4 sy = __ldg(t.sym + kx);
    const float den = (lyz_f + sy.x) * (wyz_f * sy.y);
    return den != 0.0f ? __fdiv_rn(coeff_f, den) : 0.0f;
  };
  auto phase_of = [&](int kx) -> float2 {  // interlace phase e^{-ik.s} (real part only on Nyquist planes, R9)
    const float2 e = __ldg(t.ph + kx);
    return make_float2(e.x * pcyz_f - e.y * psyz_f, e.x * psyz_f + e.y * pcyz_f);
  };
  auto grad_of = [&](int a, int kx) -> float { return a == 0 ? __ldg(&t.sym[kx].z) : (a == 1 ? dyv : dzv); };

  // In every transform the last forward stage and the first inverse stage give a thread the same elements
  // (same radix, same sub-transform size), so s_a is only ever touched by the thread that owns the element.
  if (MODE == 0) {
    const bool two = in1 != nullptr;
    if (two)  // second grid first: s_a = 1/2 phase * dhat2
      xfft_line<N, false>(s_w, t.tw, tid, gld(in1), [&](int p, int cc, float2 v) {
        const float2 e = cmulx(phase_of(xfft_freq<N>(p)), v);
        s_a[sidx(p, cc)] = make_float2(0.5f * e.x, 0.5f * e.y);
      });
    xfft_line<N, false>(s_w, t.tw, tid, gld(in0), [&](int p, int cc, float2 v) {  // s_a = green * dhat
      if (two) {
        const float2 e = s_a[sidx(p, cc)];
        v = make_float2(0.5f * v.x + e.x, 0.5f * v.y + e.y);
      }
      const float g = green_of(xfft_freq<N>(p));
      s_a[sidx(p, cc)] = make_float2(g * v.x, g * v.y);
    });
    // x component: the gradient symbol varies along the line
    xfft_line<N, true>(
        s_w, t.tw, tid,
        [&](int p, int cc) {  // -i D_x (re + i im) = D_x (im - i re)
          const float dm = grad_of(0, xfft_freq<N>(p));
          const float2 d = s_a[sidx(p, cc)];
          return make_float2(dm * d.y, -dm * d.x);
        },
        gst(out0));
    // y and z components: their gradient symbols are constant along x, so ONE inverse transform serves both
    // (x-inverse of -i D_y A = -i D_y x-inverse of A); the factor is applied to the output.
    xfft_line<N, true>(
        s_w, t.tw, tid, [&](int p, int cc) { return s_a[sidx(p, cc)]; },
        [&](int p, int, float2 v) {
          if (live) {
            out1[(size_t)p * plane + q] = make_float2(dyv * v.y, -dyv * v.x);
            out2[(size_t)p * plane + q] = make_float2(dzv * v.y, -dzv * v.x);
          }
        });
  } else if (MODE == 2) {
    const bool two = in1 != nullptr;
    if (two)
      xfft_line<N, false>(s_w, t.tw, tid, gld(in1), [&](int p, int cc, float2 v) {
        const float2 e = cmulx(phase_of(xfft_freq<N>(p)), v);
        s_a[sidx(p, cc)] = make_float2(0.5f * e.x, 0.5f * e.y);
      });
    xfft_line<N, false>(s_w, t.tw, tid, gld(in0), [&](int p, int cc, float2 v) {
      if (two) {
        const float2 e = s_a[sidx(p, cc)];
        v = make_float2(0.5f * v.x + e.x, 0.5f * v.y + e.y);
      }
      const float g = green_of(xfft_freq<N>(p));
      s_a[sidx(p, cc)] = make_float2(g * v.x, g * v.y);
    });
    xfft_line<N, true>(s_w, t.tw, tid, [&](int p, int cc) { return s_a[sidx(p, cc)]; }, gst(out0));
  } else {
    const bool two = out1 != nullptr;
    // conj(S_a) = +i D_a green:  q = i [D_x FFT_x(g_x) + FFT_x(D_y g_y + D_z g_z)]; green is applied on the way
    // out.  D_y, D_z are constant along x, so the y and z cotangents share one forward transform.
    xfft_line<N, false>(s_w, t.tw, tid, gld(in0), [&](int p, int cc, float2 v) {
      const float dm = grad_of(0, xfft_freq<N>(p));
      s_a[sidx(p, cc)] = make_float2(-dm * v.y, dm * v.x);
    });
    xfft_line<N, false>(
        s_w, t.tw, tid,
        [&](int p, int) {
          if (!live) return make_float2(0.f, 0.f);
          const float2 a = __ldcs(in1 + (size_t)p * plane + q), b = __ldcs(in2 + (size_t)p * plane + q);
          return make_float2(dyv * a.x + dzv * b.x, dyv * a.y + dzv * b.y);
        },
        [&](int p, int cc, float2 v) {
          float2 acc = s_a[sidx(p, cc)];
          acc.x -= v.y;
          acc.y += v.x;
          s_a[sidx(p, cc)] = acc;
        });
#pragma unroll 1
    for (int o = 0; o < (two ? 2 : 1); ++o) {
      xfft_line<N, true>(
          s_w, t.tw, tid,
          [&](int p, int cc) {
            const int kx = xfft_freq<N>(p);
            const float g = green_of(kx) * (two ? 0.5f : 1.0f);
            const float2 d = s_a[sidx(p, cc)];
            float2 v = make_float2(g * d.x, g * d.y);
            if (o == 1) v = cmulc(v, phase_of(kx));  // conj of the interlace phase
            return v;
          },
          gst(o == 0 ? out0 : out1));
    }
  }
}

// ---- host side -------------------------------------------------------------------------------------------
bool xfft_supported(int m) {
  return m == 64 || m == 128 || m == 256 || m == 512 || m == 1024 || m == 320 || m == 640;
}

int xfft_init(Ctx* c) {  // twiddle table and the batched 2-D (y,z) cuFFT plans; called from pm_create
  c->xfused = false;
  if (!xfft_supported(c->mg)) return PM_OK;
  if (c->p.flags & PM_FLAG_NO_XFUSE) return PM_OK;
  const int m = c->mg;
  std::vector<float2> tw(m);
  for (int k = 0; k < m; ++k) {
    const double a = -2.0 * M_PI * (double)k / (double)m;
    tw[k] = make_float2((float)cos(a), (float)sin(a));
  }
  PM_CUDA(c, cudaMalloc((void**)&c->xtw, sizeof(float2) * (size_t)m));
  PM_CUDA(c, cudaMemcpy(c->xtw, tw.data(), sizeof(float2) * (size_t)m, cudaMemcpyHostToDevice));
  {  // fp32 copies of the per-axis symbol tables, packed for one load per mode
    std::vector<double> g(m), l(m), w(m), pc(m), ps(m);
    const size_t nb = sizeof(double) * (size_t)m;
    PM_CUDA(c, cudaMemcpy(g.data(), c->tab_grad, nb, cudaMemcpyDeviceToHost));
    PM_CUDA(c, cudaMemcpy(l.data(), c->tab_lap, nb, cudaMemcpyDeviceToHost));
    PM_CUDA(c, cudaMemcpy(w.data(), c->tab_win, nb, cudaMemcpyDeviceToHost));
    PM_CUDA(c, cudaMemcpy(pc.data(), c->tab_cos, nb, cudaMemcpyDeviceToHost));
    PM_CUDA(c, cudaMemcpy(ps.data(), c->tab_sin, nb, cudaMemcpyDeviceToHost));
    std::vector<float4> sym(m);
    std::vector<float2> ph(m);
    for (int k = 0; k < m; ++k) {
      sym[k] = make_float4((float)l[k], (float)w[k], (float)g[k], 0.f);
      ph[k] = make_float2((float)pc[k], (float)ps[k]);
    }
    PM_CUDA(c, cudaMalloc((void**)&c->xsym, sizeof(float4) * (size_t)m));
    PM_CUDA(c, cudaMemcpy(c->xsym, sym.data(), sizeof(float4) * (size_t)m, cudaMemcpyHostToDevice));
    PM_CUDA(c, cudaMalloc((void**)&c->xph, sizeof(float2) * (size_t)m));
    PM_CUDA(c, cudaMemcpy(c->xph, ph.data(), sizeof(float2) * (size_t)m, cudaMemcpyHostToDevice));
  }
  int n2[2] = {m, m};
  size_t ws1 = 0, ws2 = 0;
  PM_CUFFT(c, cufftCreate(&c->plan2_r2c));
  PM_CUFFT(c, cufftCreate(&c->plan2_c2r));
  c->plans2_ok = true;
  PM_CUFFT(c, cufftSetAutoAllocation(c->plan2_r2c, 0));
  PM_CUFFT(c, cufftSetAutoAllocation(c->plan2_c2r, 0));
  PM_CUFFT(c, cufftMakePlanMany(c->plan2_r2c, 2, n2, nullptr, 1, 0, nullptr, 1, 0, CUFFT_R2C, m, &ws1));
  PM_CUFFT(c, cufftMakePlanMany(c->plan2_c2r, 2, n2, nullptr, 1, 0, nullptr, 1, 0, CUFFT_C2R, m, &ws2));
  c->fft2_work_bytes = ws1 > ws2 ? ws1 : ws2;
  c->xfused = true;
  return PM_OK;
}

int fft2_r2c(Ctx* c, const float* in, float2* out, cudaStream_t st) {
  PM_CUFFT(c, cufftSetStream(c->plan2_r2c, st));
  PM_CUFFT(c, cufftExecR2C(c->plan2_r2c, const_cast<float*>(in), reinterpret_cast<cufftComplex*>(out)));
  return PM_OK;
}
int fft2_c2r(Ctx* c, float2* in, float* out, cudaStream_t st) {
  PM_CUFFT(c, cufftSetStream(c->plan2_c2r, st));
  PM_CUFFT(c, cufftExecC2R(c->plan2_c2r, reinterpret_cast<cufftComplex*>(in), out));
  return PM_OK;
}

template <int N, int MODE>
static int xfft_launch_n(Ctx* c, const XTabs& t, const float2* i0, const float2* i1, const float2* i2, float2* o0,
                         float2* o1, float2* o2, double coeff_eff, cudaStream_t st) {
  constexpr int NT = N * XC / XEPT;
  constexpr size_t smem = sizeof(float2) * 2 * (size_t)xfft_smem_elems<N>();
  auto kern = k_xfft_kspace<N, MODE>;
  int occ = 0;
  PM_TRY(kernel_occupancy(c, (const void*)kern, NT, smem, &occ));
  const int64_t grid = (t.ncol + XC - 1) / XC;
  kern<<<(unsigned)grid, NT, smem, st>>>(t, i0, i1, i2, o0, o1, o2, coeff_eff);
  count_launch(c);
  PM_CUDA(c, cudaGetLastError());
  return PM_OK;
}

template <int MODE>
static int xfft_launch(Ctx* c, const float2* i0, const float2* i1, const float2* i2, float2* o0, float2* o1,
                       float2* o2, double coeff_eff, cudaStream_t st) {
  XTabs t;
  t.grad = c->tab_grad;
  t.lap = c->tab_lap;
  t.win = c->tab_win;
  t.pc = c->tab_cos;
  t.ps = c->tab_sin;
  t.tw = c->xtw;
  t.sym = c->xsym;
  t.ph = c->xph;
  t.m = c->mg;
  t.hz = c->mg / 2 + 1;
  t.ncol = (int64_t)t.m * t.hz;
  switch (c->mg) {
    case 64: return xfft_launch_n<64, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 128: return xfft_launch_n<128, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 256: return xfft_launch_n<256, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 512: return xfft_launch_n<512, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 1024: return xfft_launch_n<1024, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 320: return xfft_launch_n<320, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
    case 640: return xfft_launch_n<640, MODE>(c, t, i0, i1, i2, o0, o1, o2, coeff_eff, st);
  }
  return fail(c, PM_ESTATE, "fused x-FFT not built for m = %d", c->mg);
}

// d1 (, d2): (y,z)-transformed density spectra -> gh[a]: x-inverse-transformed force spectra
int launch_xfft_forward(Ctx* c, const float2* d1, const float2* d2, float2* const gh[3], double coeff_eff,
                        cudaStream_t st) {
  return xfft_launch<0>(c, d1, d2, nullptr, gh[0], gh[1], gh[2], coeff_eff, st);
}
// gh[a]: (y,z)-transformed cotangent spectra -> q1 (, q2): x-inverse-transformed density cotangent spectra
int launch_xfft_transpose(Ctx* c, const float2* const gh[3], float2* q1, float2* q2, double coeff_eff,
                          cudaStream_t st) {
  return xfft_launch<1>(c, gh[0], gh[1], gh[2], q1, q2, nullptr, coeff_eff, st);
}

// potential: d1 (, d2) -> phi spectrum
int launch_xfft_potential(Ctx* c, const float2* d1, const float2* d2, float2* phi, double coeff_eff, cudaStream_t st) {
  return xfft_launch<2>(c, d1, d2, nullptr, phi, nullptr, nullptr, coeff_eff, st);
}

// ---- the spectral operator on real meshes, fused or not ------------------------------------------------------
int spectral_forward(Ctx* c, const float* d1, const float* d2, float* const g[3], double coeff_eff, bool stages,
                     cudaStream_t st) {
  const bool fused = c->xfused;
  if (stages) stage_begin(c, PM_STAGE_FFT_FWD, st);
  PM_TRY(fused ? fft2_r2c(c, d1, c->dhat[0], st) : fft_r2c(c, d1, c->dhat[0], st));
  if (d2) PM_TRY(fused ? fft2_r2c(c, d2, c->dhat[1], st) : fft_r2c(c, d2, c->dhat[1], st));
  if (stages) stage_end(c, PM_STAGE_FFT_FWD, st);
  if (c->p.flags & PM_FLAG_GRAD_REAL) {  // one inverse transform of the potential, gradient by the Table 2 stencil
    PM_TRY(ensure_phi(c));
    if (stages) stage_begin(c, PM_STAGE_KSPACE, st);
    PM_TRY(spectral_potential_hat(c, d2 != nullptr, c->ghat[0], coeff_eff, st));
    if (stages) stage_end(c, PM_STAGE_KSPACE, st);
    if (stages) stage_begin(c, PM_STAGE_FFT_INV, st);
    PM_TRY(fused ? fft2_c2r(c, c->ghat[0], c->phi, st) : fft_c2r(c, c->ghat[0], c->phi, st));
    if (stages) stage_end(c, PM_STAGE_FFT_INV, st);
    if (stages) stage_begin(c, PM_STAGE_GRADIENT, st);
    PM_TRY(launch_fd_gradient(c, c->phi, g, st));
    if (stages) stage_end(c, PM_STAGE_GRADIENT, st);
    return PM_OK;
  }
  if (stages) stage_begin(c, PM_STAGE_KSPACE, st);
  if (fused)
    PM_TRY(launch_xfft_forward(c, c->dhat[0], d2 ? c->dhat[1] : nullptr, c->ghat, coeff_eff, st));
  else
    PM_TRY(launch_kspace_forward(c, c->dhat[0], d2 ? c->dhat[1] : nullptr, c->ghat, coeff_eff, st));
  if (stages) stage_end(c, PM_STAGE_KSPACE, st);
  if (stages) stage_begin(c, PM_STAGE_FFT_INV, st);
  for (int a = 0; a < 3; ++a) PM_TRY(fused ? fft2_c2r(c, c->ghat[a], g[a], st) : fft_c2r(c, c->ghat[a], g[a], st));
  if (stages) stage_end(c, PM_STAGE_FFT_INV, st);
  return PM_OK;
}

// dhat[0] (, dhat[1]) -> out = green * (combined) density spectrum (x-inverse-transformed on the fused path)
int spectral_potential_hat(Ctx* c, bool two, float2* out, double coeff_eff, cudaStream_t st) {
  if (c->xfused) return launch_xfft_potential(c, c->dhat[0], two ? c->dhat[1] : nullptr, out, coeff_eff, st);
  return launch_kspace_scalar(c, c->dhat[0], two ? c->dhat[1] : nullptr, out, coeff_eff, st);
}

// The potential mesh of the spread / assigned density: d1 (, d2) -> phi (real space).  Used by the NUFFT
// kernel-gradient force (PM_FLAG_KERNEL_GRAD).
int spectral_potential(Ctx* c, const float* d1, const float* d2, float* phi, double coeff_eff, bool stages,
                       cudaStream_t st) {
  const bool fused = c->xfused;
  if (stages) stage_begin(c, PM_STAGE_FFT_FWD, st);
  PM_TRY(fused ? fft2_r2c(c, d1, c->dhat[0], st) : fft_r2c(c, d1, c->dhat[0], st));
  if (d2) PM_TRY(fused ? fft2_r2c(c, d2, c->dhat[1], st) : fft_r2c(c, d2, c->dhat[1], st));
  if (stages) stage_end(c, PM_STAGE_FFT_FWD, st);
  if (stages) stage_begin(c, PM_STAGE_KSPACE, st);
  PM_TRY(spectral_potential_hat(c, d2 != nullptr, c->ghat[0], coeff_eff, st));
  if (stages) stage_end(c, PM_STAGE_KSPACE, st);
  if (stages) stage_begin(c, PM_STAGE_FFT_INV, st);
  PM_TRY(fused ? fft2_c2r(c, c->ghat[0], phi, st) : fft_c2r(c, c->ghat[0], phi, st));
  if (stages) stage_end(c, PM_STAGE_FFT_INV, st);
  return PM_OK;
}

// The transposed operator always works in Fourier space, also for a PM_FLAG_GRAD_REAL ctx (same linear operator;
// see pm_stencil.cu for why its real-space form is not used).
int spectral_transpose(Ctx* c, const float* const gb[3], float* q1, float* q2, double coeff_eff, cudaStream_t st) {
  const bool fused = c->xfused;
  for (int a = 0; a < 3; ++a) PM_TRY(fused ? fft2_r2c(c, gb[a], c->ghat[a], st) : fft_r2c(c, gb[a], c->ghat[a], st));
  if (fused)
    PM_TRY(launch_xfft_transpose(c, c->ghat, c->dhat[0], q2 ? c->dhat[1] : nullptr, coeff_eff, st));
  else
    PM_TRY(launch_kspace_transpose(c, c->ghat, c->dhat[0], q2 ? c->dhat[1] : nullptr, coeff_eff, st));
  PM_TRY(fused ? fft2_c2r(c, c->dhat[0], q1, st) : fft_c2r(c, c->dhat[0], q1, st));
  if (q2) PM_TRY(fused ? fft2_c2r(c, c->dhat[1], q2, st) : fft_c2r(c, c->dhat[1], q2, st));
  return PM_OK;
}

}  // namespace pmf
