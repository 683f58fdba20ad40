// jerk_fft64.cuh — two-pass 64 x 64 register FFT for seg_len 4096.
//
// One length-4096 complex FFT is computed by 64 threads (two warps) holding 64 points each, in TWO passes of radix 64
// with ONE shared-memory exchange (the three-pass radix-16 scheme of jerk_fft.cuh needs two).  The fused search kernel
// is bound by the L1TEX/shared-memory data stage (profiles/r1_02: 76.8 % busy against 61.9 % for the FMA pipe), and a
// 64-point register transform halves the exchange traffic per point, needs no shared-memory twiddle table, and has a
// quarter of the barriers per flop.  PAPER.md:31 (shared-memory FFT inside the convolution kernel) is the prior art.
//
//   k = 64*k1 + k0 (input),   n = n0 + 64*n1 (output),   w_L^{kn} = w_64^{k1 n0} * w_L^{k0 n0} * w_64^{k0 n1}
//
//   pass 1: thread k0 holds x[64 k1 + k0], k1 = 0..63: DFT_64 over k1 -> B[k0][n0]
//   exchange: element (k0, n0) at float2 slot kS64*n0 + k0 (row stride 66: 64-bit stores and 128-bit loads conflict-free)
//   pass 2: thread n0 holds B[k0][n0], k0 = 0..63: twiddle w_L^{k0 n0} folded into the first radix-4 layer, DFT_64 over k0
//           -> X[n0 + 64 n1]
//
// DFT_64 = 4 x 16: radix-4 butterflies over x[16 a + b], then four DFT_16 whose input twiddles w_64^{b k} are compile-time
// constants split into a quarter turn (free operand modifier) and a residual angle |rho| <= pi/4 applied as
// c * (v + tan(rho) * i v) with c folded into the following fused multiply-adds.
// Register order of a DFT_64 result: output index a + 4 b sits in register 16 a + b  (dft64_out_index).
#pragma once
#include "jerk_fft.cuh"

namespace jerk {

constexpr int kS64 = 66;              // exchange row stride in float2
constexpr int kEx64 = 64 * kS64;      // float2 slots of one exchange buffer (>= 4096: doubles as a plain staging array)

// cos and tan of 2 pi m / 64, m = 0..8
__device__ __forceinline__ constexpr float cos64(int m) {
  return m == 0 ? 1.0f
       : m == 1 ? 0.99518472667219688624f
       : m == 2 ? 0.98078528040323044913f
       : m == 3 ? 0.95694033573220886494f
       : m == 4 ? 0.92387953251128675613f
       : m == 5 ? 0.88192126434835502971f
       : m == 6 ? 0.83146961230254523708f
       : m == 7 ? 0.77301045336273696081f
       : 0.70710678118654752440f;
}
__device__ __forceinline__ constexpr float tan64(int m) {
  return m == 0 ? 0.0f
       : m == 1 ? 0.09849140335716425308f
       : m == 2 ? 0.19891236737965800691f
       : m == 3 ? 0.30334668360734239167f
       : m == 4 ? 0.41421356237309504880f
       : m == 5 ? 0.53451113595079164680f
       : m == 6 ? 0.66817863791929891999f
       : m == 7 ? 0.82067879082866033098f
       : 1.0f;
}

// (SIGN i)^Q * a
template <int SIGN, int Q>
__device__ __forceinline__ float2 rotq(float2 a) {
  constexpr int q = ((Q % 4) + 4) % 4;
  if (q == 0) return a;
  if (q == 1) return rot90<SIGN>(a);
  if (q == 2) return cneg(a);
  return rot90<-SIGN>(a);
}

// w = exp(SIGN 2 pi i E / 64) = (SIGN i)^quad * c * (1 + SIGN i t),  residual r = E - 16 quad in [-8, 7]
template <int E>
struct Tw64 {
  static constexpr int e = ((E % 64) + 64) % 64;
  static constexpr int quad = ((e + 8) / 16) % 4;
  static constexpr int r = e - 16 * ((e + 8) / 16);
  static constexpr float c = cos64(r < 0 ? -r : r);
  static constexpr float t = r < 0 ? -tan64(-r) : tan64(r);
};

// w x / c : one fused multiply-add, or nothing for a pure quarter turn
template <int SIGN, int E>
__device__ __forceinline__ float2 tw64_u(float2 x) {
  using T = Tw64<E>;
  if (T::r == 0) return rotq<SIGN, T::quad>(x);
  return fma_s(rotq<SIGN, T::quad + 1>(x), T::t, rotq<SIGN, T::quad>(x));
}

// radix-4 butterfly over inputs carrying the constant twiddles w_64^{E0..E3}: x_k <- sum_a (SIGN i)^{a k} w^{E_a} x_a
template <int SIGN, int E0, int E1, int E2, int E3>
__device__ __forceinline__ void bfly4_ct(float2& x0, float2& x1, float2& x2, float2& x3) {
  constexpr float c0 = Tw64<E0>::c, c1 = Tw64<E1>::c, c2 = Tw64<E2>::c, c3 = Tw64<E3>::c;
  float2 a0 = tw64_u<SIGN, E0>(x0);
  if (Tw64<E0>::r != 0) a0 = __fmul2_rn(a0, bc(c0));
  const float2 u1 = tw64_u<SIGN, E1>(x1), u2 = tw64_u<SIGN, E2>(x2), u3 = tw64_u<SIGN, E3>(x3);
  float2 t0, t1, t2, t3;
  if (Tw64<E2>::r == 0) {
    t0 = cadd(a0, u2);
    t1 = csub(a0, u2);
  } else {
    t0 = fma_s(u2, c2, a0);
    t1 = fma_s(cneg(u2), c2, a0);
  }
  if (Tw64<E1>::r == 0 && Tw64<E3>::r == 0) {
    t2 = cadd(u1, u3);
    t3 = csub(u1, u3);
    const float2 r3 = rot90<SIGN>(t3);
    x0 = cadd(t0, t2);
    x2 = csub(t0, t2);
    x1 = cadd(t1, r3);
    x3 = csub(t1, r3);
  } else {
    t2 = fma_s(u3, c3 / c1, u1);
    t3 = fma_s(cneg(u3), c3 / c1, u1);
    bfly4_tail<SIGN>(t0, t1, t2, t3, c1, x0, x1, x2, x3);
  }
}

// x[q] *= w_64^{K q}, q = 0..15, then DFT_16 (natural output order)
template <int SIGN, int K>
__device__ __forceinline__ void dft16_ct(float2 (&x)[16]) {
  bfly4_ct<SIGN, 0, 4 * K, 8 * K, 12 * K>(x[0], x[4], x[8], x[12]);
  bfly4_ct<SIGN, K, 5 * K, 9 * K, 13 * K>(x[1], x[5], x[9], x[13]);
  bfly4_ct<SIGN, 2 * K, 6 * K, 10 * K, 14 * K>(x[2], x[6], x[10], x[14]);
  bfly4_ct<SIGN, 3 * K, 7 * K, 11 * K, 15 * K>(x[3], x[7], x[11], x[15]);
  dft16_layerB<SIGN>(x);
}

// second half of DFT_64: x[16 a + b] (a = radix-4 output, b = 0..15) -> X[a + 4 k2] at x[16 a + k2]
template <int SIGN>
__device__ __forceinline__ void dft64_stage2(float2 (&x)[64]) {
#define JERK_DFT64_COL(A)                                   \
  {                                                         \
    float2 y[16];                                           \
    _Pragma("unroll") for (int b = 0; b < 16; b++) y[b] = x[16 * A + b]; \
    dft16_ct<SIGN, A>(y);                                   \
    _Pragma("unroll") for (int b = 0; b < 16; b++) x[16 * A + b] = y[b]; \
  }
  JERK_DFT64_COL(0)
  JERK_DFT64_COL(1)
  JERK_DFT64_COL(2)
  JERK_DFT64_COL(3)
#undef JERK_DFT64_COL
}

// DFT_64 of x[0..63] (input index = register index); output index a + 4 b is left in register 16 a + b
template <int SIGN>
__device__ __forceinline__ void dft64(float2 (&x)[64]) {
#pragma unroll
  for (int b = 0; b < 16; b++) {
    float2 t[4] = {x[b], x[16 + b], x[32 + b], x[48 + b]};
    Dft<4, SIGN>::run(t);
    x[b] = t[0]; x[16 + b] = t[1]; x[32 + b] = t[2]; x[48 + b] = t[3];
  }
  dft64_stage2<SIGN>(x);
}
__device__ __forceinline__ constexpr int dft64_out_index(int reg) { return (reg >> 4) + 4 * (reg & 15); }

// First layer of a DFT_64 whose inputs carry runtime twiddles in mixed form (dft16_layerA_tw): tw(c, w) returns table
// entries 16c..16c+15, entry 4 b + a belongs to input register 16 a + b.  SIGN < 0 conjugates the (inverse-sign) table.
template <int SIGN, class TW>
__device__ __forceinline__ void dft64_tw_stage1(float2 (&x)[64], const TW& tw) {
#pragma unroll
  for (int c = 0; c < 4; c++) {
    float2 w16[16];
    tw.load16(c, w16);
#pragma unroll
    for (int m = 0; m < 4; m++) {
      const int b = 4 * c + m;
      const float2 w[4] = {w16[4 * m], w16[4 * m + 1], w16[4 * m + 2], w16[4 * m + 3]};
      if (b == 0) dft16_layerA_tw<SIGN, true>(x[0], x[16], x[32], x[48], w);
      else dft16_layerA_tw<SIGN, false>(x[b], x[16 + b], x[32 + b], x[48 + b], w);
    }
  }
}
#ifdef __CUDACC__
// The same with the table in tensor memory, double-buffered: the load of chunk c+1 is in flight while chunk c is used.
template <int SIGN>
__device__ __forceinline__ void dft64_tw_stage1(float2 (&x)[64], const TmemArray<4096>& tw) {
  float wa[32], wb[32];
  tw.issue16(0, wa);
#pragma unroll
  for (int c = 0; c < 4; c++) {
    float(&cur)[32] = (c & 1) ? wb : wa;
    float(&nxt)[32] = (c & 1) ? wa : wb;
    tmem_ld32_wait(cur);
    if (c < 3) tw.issue16(c + 1, nxt);
#pragma unroll
    for (int m = 0; m < 4; m++) {
      const int b = 4 * c + m;
      const float2 w[4] = {make_float2(cur[8 * m], cur[8 * m + 1]), make_float2(cur[8 * m + 2], cur[8 * m + 3]),
                           make_float2(cur[8 * m + 4], cur[8 * m + 5]), make_float2(cur[8 * m + 6], cur[8 * m + 7])};
      if (b == 0) dft16_layerA_tw<SIGN, true>(x[0], x[16], x[32], x[48], w);
      else dft16_layerA_tw<SIGN, false>(x[b], x[16 + b], x[32 + b], x[48 + b], w);
    }
  }
}
#endif
template <int SIGN, class TW>
__device__ __forceinline__ void dft64_tw(float2 (&x)[64], const TW& tw) {
  dft64_tw_stage1<SIGN>(x, tw);
  dft64_stage2<SIGN>(x);
}
// column A (0..3) of the second stage alone: x[16 A + b] -> X[A + 4 k2] at x[16 A + k2]
template <int SIGN, int A>
__device__ __forceinline__ void dft64_stage2_col(float2 (&x)[64]) {
  float2 y[16];
#pragma unroll
  for (int b = 0; b < 16; b++) y[b] = x[16 * A + b];
  dft16_ct<SIGN, A>(y);
#pragma unroll
  for (int b = 0; b < 16; b++) x[16 * A + b] = y[b];
}

// Pass-2 twiddle table entry pos = 4 b + a of thread n0 (inverse sign): mixed form of w_4096^{(16 a + b) n0}
__device__ __forceinline__ float2 tw64_mixed(int pos, int n0) {
  const int a = pos & 3, b = pos >> 2;
  const float2 w = unit_root((16 * a + b) * n0, 4096);
  if (a == 0) return w;
  const float c = tw_cos_safe(w.x);
  const float t = w.y / c;
  if (a == 3) return make_float2(c / tw_cos_safe(unit_root((16 + b) * n0, 4096).x), t);
  return make_float2(c, t);
}

#ifdef __CUDACC__
__device__ __forceinline__ void bar_sync_named(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

// Both passes on the 64 points of thread t (0..63) of one FFT group.  On entry v[k1] = x[64 k1 + t]; on exit register r
// holds X[t + 64 * dft64_out_index(r)].  ex: the group's exchange buffer (kEx64 float2); barid: its named barrier.
// mid() runs between the two layers of pass 1 (a cheap place to start a barrier probe whose answer before_store() needs),
// before_store() before the first write to ex (the caller's write-after-read protection of ex), after_load() right
// after the last read of ex.
// The exchange is spread over the arithmetic: each of the four second-layer columns of pass 1 is stored as soon as it is
// done (the stores of column A issue under the butterflies of column A + 1), and the pass-2 loads are issued in the order
// the first radix-4 layer consumes them (registers b, 16 + b, 32 + b, 48 + b), so that layer starts after four loads
// instead of thirty-two.
// FIRST_DONE: the caller has already run the first radix-4 layer of pass 1 (the search kernel fuses it with the
// multiplication by G: dft16_layerA_tw on F and the mixed-form filter).
template <int SIGN, bool FIRST_DONE = false, class TW, class MID, class PRE, class POST>
__device__ __forceinline__ void fft64_passes(float2 (&v)[64], const TW& tw, float2* ex, int t, int barid, MID mid, PRE before_store,
                                             POST after_load) {
  if (!FIRST_DONE) {
#pragma unroll
    for (int b = 0; b < 16; b++) {
      float2 q[4] = {v[b], v[16 + b], v[32 + b], v[48 + b]};
      Dft<4, SIGN>::run(q);
      v[b] = q[0]; v[16 + b] = q[1]; v[32 + b] = q[2]; v[48 + b] = q[3];
    }
  }
  mid();
  float2* w = ex + t;
#define JERK_FFT64_COL(A)                                                                  \
  dft64_stage2_col<SIGN, A>(v);                                                            \
  if (A == 0) before_store();                                                              \
  _Pragma("unroll") for (int k2 = 0; k2 < 16; k2++) w[kS64 * (A + 4 * k2)] = v[16 * A + k2];   /* element (k0 = t, n0 = A + 4 k2) */
  JERK_FFT64_COL(0)
  JERK_FFT64_COL(1)
  JERK_FFT64_COL(2)
  JERK_FFT64_COL(3)
#undef JERK_FFT64_COL
  bar_sync_named(barid, 64);
  {
    const float4* rd = reinterpret_cast<const float4*>(ex + kS64 * t);
#pragma unroll
    for (int p = 0; p < 8; p++)
#pragma unroll
      for (int a = 0; a < 4; a++) {
        const int q = 8 * a + p;
        const float4 x = rd[q];
        v[2 * q] = make_float2(x.x, x.y);
        v[2 * q + 1] = make_float2(x.z, x.w);
      }
  }
  after_load();
  dft64_tw<SIGN>(v, tw);
}
#endif

}  // namespace jerk
