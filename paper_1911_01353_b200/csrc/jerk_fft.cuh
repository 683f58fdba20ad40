// jerk_fft.cuh — register/shared-memory radix FFT used by the template-bank and fused search kernels.
//
// One length-L complex FFT is computed by NT = L/P threads holding P = max(16, L/256) points each, in three
// passes of radices R1 = L/256, 16, 16 with two shared-memory exchanges (
// PAPER.md:31 "shared memory implementation of the FFT").  Index algebra:
//
//   k = 256*k2 + 16*k1 + k0   (input),      n = n0 + R1*n1 + 16*R1*n2   (output)
//   w_L^{kn} = w_R1^{k2 n0} * w_L^{(16 k1 + k0) n0} * w_16^{k1 n1} * w_256^{k0 n1} * w_16^{k0 n2}
//
//   pass 1: butterfly b1 = 16*k1 + k0  : DFT_R1 over k2,  then twiddle T1 = w_L^{b1*n0}   (per-thread registers)
//   pass 2: butterfly b2 = 16*n0 + k0  : DFT_16 over k1;  twiddle T2 = w_256^{k0*n1} (16x16 smem table) is applied when pass 3 loads
//   pass 3: butterfly b3 = n0 + R1*n1  : DFT_16 over k0,  output n = b3 + 16*R1*n2
//
// SIGN = +1 is the unnormalised inverse transform (e^{+2 pi i kn/L}), SIGN = -1 the forward one.
#pragma once
#include <cuda_runtime.h>

namespace jerk {

// Complex arithmetic on (re, im) register pairs with Blackwell's packed FP32 instructions (FADD2 / FMUL2 / FFMA2):
// one issue slot does both halves; the half-swap, negate and scalar-broadcast operand forms are free SASS modifiers
// (R.F32x2.LO_HI, -R.F32x2.LO_HI.NP, R.F32), so multiplying by +-i costs nothing and a complex multiply is 2 instructions.
__device__ __forceinline__ float2 bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
// a * b = a*(b.x,b.x) + (i a)*(b.y,b.y)
__device__ __forceinline__ float2 cmul(float2 a, float2 b) {
  return __ffma2_rn(make_float2(-a.y, a.x), bc(b.y), __fmul2_rn(a, bc(b.x)));
}
// a * conj(b) = a*(b.x,b.x) + (-i a)*(b.y,b.y)
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 b) {
  return __ffma2_rn(make_float2(a.y, -a.x), bc(b.y), __fmul2_rn(a, bc(b.x)));
}

// multiply by SIGN * i (folds into the operand modifier of the consuming packed instruction)
template <int SIGN>
__device__ __forceinline__ float2 rot90(float2 a) {
  return SIGN > 0 ? make_float2(-a.y, a.x) : make_float2(a.y, -a.x);
}

// cos(2 pi m / 32), m = 0..8
__device__ __forceinline__ constexpr float cos32(int m) {
  return m == 0 ? 1.0f
       : m == 1 ? 0.98078528040323044913f
       : m == 2 ? 0.92387953251128675613f
       : m == 3 ? 0.83146961230254523708f
       : m == 4 ? 0.70710678118654752440f
       : m == 5 ? 0.55557023301960222474f
       : m == 6 ? 0.38268343236508977173f
       : m == 7 ? 0.19509032201612826785f
       : 0.0f;
}

// v * w_N^{m} with w_N = exp(SIGN * 2 pi i / N), N in {4,8,16,32}, m a compile-time constant after unrolling.
template <int SIGN, int N>
__device__ __forceinline__ float2 mul_tw(float2 v, int m) {
  int k = ((m % N) + N) % N * (32 / N);   // in 32nds of a turn, 0..31
  int quad = k >> 3;                       // quarter turns
  int r = k & 7;                           // remainder, 0..7
  float2 t = v;
  if (r != 0) {
    if (r == 4) {                          // (1 + SIGN i)/sqrt(2) * v = (v + SIGN i v)/sqrt(2)
      t = __fmul2_rn(__fadd2_rn(v, rot90<SIGN>(v)), bc(cos32(4)));
    } else {                               // (c + SIGN i s) * v = c v + s (SIGN i v)
      t = __ffma2_rn(rot90<SIGN>(v), bc(cos32(8 - r)), __fmul2_rn(v, bc(cos32(r))));
    }
  }
  // apply quarter turns: multiply by (SIGN i)^quad
  if (quad == 1) t = rot90<SIGN>(t);
  else if (quad == 2) t = make_float2(-t.x, -t.y);
  else if (quad == 3) t = rot90<-SIGN>(t);
  return t;
}

template <int R, int SIGN>
struct Dft;

template <int SIGN>
struct Dft<2, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[2]) {
    float2 a = x[0], b = x[1];
    x[0] = cadd(a, b);
    x[1] = csub(a, b);
  }
};

template <int SIGN>
struct Dft<4, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[4]) {
    float2 t0 = cadd(x[0], x[2]), t1 = csub(x[0], x[2]);
    float2 t2 = cadd(x[1], x[3]), t3 = rot90<SIGN>(csub(x[1], x[3]));
    x[0] = cadd(t0, t2);
    x[2] = csub(t0, t2);
    x[1] = cadd(t1, t3);
    x[3] = csub(t1, t3);
  }
};

// Cooley-Tukey step R = P*Q in registers:  X[k1 + P k2] = sum_{n2<Q} w_R^{n2 k1} w_Q^{n2 k2} sum_{n1<P} x[Q n1 + n2] w_P^{n1 k1}
template <int P, int Q, int SIGN>
__device__ __forceinline__ void dft_pq(float2 (&x)[P * Q]) {
  float2 y[Q][P];
#pragma unroll
  for (int n2 = 0; n2 < Q; n2++) {
    float2 t[P];
#pragma unroll
    for (int n1 = 0; n1 < P; n1++) t[n1] = x[Q * n1 + n2];
    Dft<P, SIGN>::run(t);
#pragma unroll
    for (int k1 = 0; k1 < P; k1++) y[n2][k1] = mul_tw<SIGN, P * Q>(t[k1], n2 * k1);
  }
#pragma unroll
  for (int k1 = 0; k1 < P; k1++) {
    float2 t[Q];
#pragma unroll
    for (int n2 = 0; n2 < Q; n2++) t[n2] = y[n2][k1];
    Dft<Q, SIGN>::run(t);
#pragma unroll
    for (int k2 = 0; k2 < Q; k2++) x[k1 + P * k2] = t[k2];
  }
}

template <int SIGN>
struct Dft<8, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[8]) { dft_pq<2, 4, SIGN>(x); }
};
template <int SIGN>
struct Dft<16, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[16]) { dft_pq<4, 4, SIGN>(x); }
};
template <int SIGN>
struct Dft<32, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[32]) { dft_pq<2, 16, SIGN>(x); }
};

// ---------------------------------------------------------------------------------------------------------
template <int L_>
struct FftGeom {
  static constexpr int L = L_;
  static constexpr int R1 = L / 256;                 // 4, 8, 16, 32
  static constexpr int P = R1 > 16 ? R1 : 16;        // points per thread
  static constexpr int NT = L / P;                   // threads per FFT
  static constexpr int NB1 = P / R1;                 // pass-1 butterflies per thread
  static constexpr int NB2 = P / 16;                 // pass-2/3 butterflies per thread
  static constexpr int LOG2L = L == 1024 ? 10 : L == 2048 ? 11 : L == 4096 ? 12 : 13;
  static_assert(L == 1024 || L == 2048 || L == 4096 || L == 8192, "seg_len");
};

// exp(SIGN * 2 pi i * num / den), den a power of two, num reduced exactly in integers
__device__ __forceinline__ float2 unit_root(int num, int den) {
  int r = num & (den - 1);
  float s, c;
  sincospif(2.0f * (float)r / (float)den, &s, &c);
  return make_float2(c, s);
}

// Per-thread T1 twiddles for the INVERSE transform: tw1[u*R1 + n0] = w_L^{b1*n0}, b1 = t + NT*u.
template <int L>
__device__ __forceinline__ void make_tw1(float2 (&tw1)[FftGeom<L>::P], int t) {
  using G = FftGeom<L>;
#pragma unroll
  for (int u = 0; u < G::NB1; u++) {
    int b1 = t + G::NT * u;
#pragma unroll
    for (int n0 = 0; n0 < G::R1; n0++) tw1[u * G::R1 + n0] = unit_root(b1 * n0, L);
  }
}

// T2 table (inverse sign) in shared memory: tw2[n1*kTw2Stride + k0] = w_256^{k0*n1}.  It is read in pass 3, where the
// row n1 = b3 / R1 is uniform over R1 consecutive lanes (broadcast loads); rows are padded to 18 float2 so that the
// rows touched by one 128-bit load instruction fall in different banks.
constexpr int kTw2Stride = 18;
constexpr int kTw2Floats2 = 16 * kTw2Stride;
__device__ __forceinline__ void fill_tw2(float2* tw2, int t, int nthreads) {
  for (int i = t; i < 256; i += nthreads) tw2[(i >> 4) * kTw2Stride + (i & 15)] = unit_root((i >> 4) * (i & 15), 256);
}

// Passes 1..3 on the P points in v[].  On entry v[u*R1 + k2] = x[256*k2 + b1], b1 = t + NT*u.
// On exit v[u3*16 + n2] = X[b3 + 16*R1*n2], b3 = t + NT*u3.  exA/exB: two exchange buffers of L float2 each.
// tw1: inverse-sign per-thread twiddles (conjugated here when SIGN < 0).  Two barriers (bar id, NT threads).
template <int L, int SIGN>
__device__ __forceinline__ void fft_passes(float2 (&v)[FftGeom<L>::P], const float2 (&tw1)[FftGeom<L>::P],
                                           const float2* __restrict__ tw2, float2* exA, float2* exB, int t) {
  using G = FftGeom<L>;
  // ---- pass 1
#pragma unroll
  for (int u = 0; u < G::NB1; u++) {
    float2 a[G::R1];
#pragma unroll
    for (int i = 0; i < G::R1; i++) a[i] = v[u * G::R1 + i];
    Dft<G::R1, SIGN>::run(a);
    int b1 = t + G::NT * u;
#pragma unroll
    for (int n0 = 0; n0 < G::R1; n0++) {
      float2 r = n0 == 0 ? a[0] : (SIGN > 0 ? cmul(a[n0], tw1[u * G::R1 + n0]) : cmul_conj(a[n0], tw1[u * G::R1 + n0]));
      exA[n0 * 256 + b1] = r;
    }
  }
  __syncthreads();
  // ---- pass 2
  const int k0 = t & 15;
#pragma unroll
  for (int u = 0; u < G::NB2; u++) {
    int b2 = t + G::NT * u;
    int n0 = b2 >> 4;
    float2 a[16];
#pragma unroll
    for (int k1 = 0; k1 < 16; k1++) a[k1] = exA[n0 * 256 + k1 * 16 + k0];
    Dft<16, SIGN>::run(a);
#pragma unroll
    for (int n1 = 0; n1 < 16; n1++) {
      int b3 = n0 + G::R1 * n1;
      exB[16 * b3 + ((k0 + b3) & 15)] = a[n1];
    }
  }
  __syncthreads();
  // ---- pass 3 (the T2 twiddle w_256^{k0*n1} is applied here, on the read side: its row n1 is lane-uniform)
#pragma unroll
  for (int u = 0; u < G::NB2; u++) {
    int b3 = t + G::NT * u;
    const float2* trow = tw2 + (b3 / G::R1) * kTw2Stride;
    float2 a[16];
#pragma unroll
    for (int q = 0; q < 16; q++) {
      float2 x = exB[16 * b3 + ((q + b3) & 15)];
      a[q] = q == 0 ? x : (SIGN > 0 ? cmul(x, trow[q]) : cmul_conj(x, trow[q]));
    }
    Dft<16, SIGN>::run(a);
#pragma unroll
    for (int n2 = 0; n2 < 16; n2++) v[u * 16 + n2] = a[n2];
  }
}

}  // namespace jerk
