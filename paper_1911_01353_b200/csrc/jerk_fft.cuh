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
#include <stdint.h>

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
// ---- DFT_16 = 4 x 4 with every twiddle absorbed into fused multiply-adds.
// A twiddle w = c + i s applied to v is written c * (v + t * (i v)), t = s / c (one FFMA2), and the factor c is applied by
// the FFMA2 that adds the result to its butterfly partner; when both partners carry a factor, one is divided out
// (c_b / c_a) and c_a is applied one level later.  A twiddled radix-4 butterfly costs 11 packed instructions instead of 14.
__device__ __forceinline__ float2 cneg(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 fma_s(float2 a, float s, float2 c) { return __ffma2_rn(a, bc(s), c); }   // a*s + c

constexpr float kC1 = 0.92387953251128675613f;   // cos(pi/8)
constexpr float kC2 = 0.70710678118654752440f;   // cos(pi/4)
constexpr float kC3 = 0.38268343236508977173f;   // cos(3pi/8)
constexpr float kT1 = 0.41421356237309504880f;   // tan(pi/8) = cos(3pi/8)/cos(pi/8)
constexpr float kT3 = 2.41421356237309504880f;   // tan(3pi/8) = cos(pi/8)/cos(3pi/8)

// second half of a radix-4 butterfly whose odd half (t2, t3) still carries the real factor c:
//   o0 = t0 + c t2, o2 = t0 - c t2, o1 = t1 + c (SIGN i) t3, o3 = t1 - c (SIGN i) t3
template <int SIGN>
__device__ __forceinline__ void bfly4_tail(float2 t0, float2 t1, float2 t2, float2 t3, float c, float2& o0, float2& o1,
                                           float2& o2, float2& o3) {
  const float2 r3 = rot90<SIGN>(t3);
  o0 = fma_s(t2, c, t0);
  o2 = fma_s(cneg(t2), c, t0);
  o1 = fma_s(r3, c, t1);
  o3 = fma_s(cneg(r3), c, t1);
}

// Second layer of DFT_16: column k1 holds v[n2] = x[4 k1 + n2]; out X[k1 + 4 k2] = sum_n2 v[n2] w16^{n2 k1} i^{SIGN n2 k2}
template <int SIGN>
__device__ __forceinline__ void dft16_layerB(float2 (&x)[16]) {
  float2 y[16];
  {  // k1 = 0: plain radix-4
    float2 t[4] = {x[0], x[1], x[2], x[3]};
    Dft<4, SIGN>::run(t);
    y[0] = t[0]; y[4] = t[1]; y[8] = t[2]; y[12] = t[3];
  }
  {  // k1 = 1: twiddles w16^1, w16^2, w16^3
    const float2 v0 = x[4], v1 = x[5], v2 = x[6], v3 = x[7];
    const float2 u2 = cadd(v2, rot90<SIGN>(v2));
    const float2 t0 = fma_s(u2, kC2, v0), t1 = fma_s(cneg(u2), kC2, v0);
    const float2 u1 = fma_s(rot90<SIGN>(v1), kT1, v1), u3 = fma_s(rot90<SIGN>(v3), kT3, v3);
    const float2 t2 = fma_s(u3, kT1, u1), t3 = fma_s(cneg(u3), kT1, u1);           // c3/c1 = tan(pi/8)
    bfly4_tail<SIGN>(t0, t1, t2, t3, kC1, y[1], y[5], y[9], y[13]);
  }
  {  // k1 = 2: twiddles w16^2, w16^4 = SIGN i, w16^6 = c2 (-1 + SIGN i)
    const float2 v0 = x[8], v1 = x[9], v2 = x[10], v3 = x[11];
    const float2 r2 = rot90<SIGN>(v2);
    const float2 t0 = cadd(v0, r2), t1 = csub(v0, r2);
    const float2 u1 = cadd(v1, rot90<SIGN>(v1)), u3 = csub(rot90<SIGN>(v3), v3);
    const float2 t2 = cadd(u1, u3), t3 = csub(u1, u3);
    bfly4_tail<SIGN>(t0, t1, t2, t3, kC2, y[2], y[6], y[10], y[14]);
  }
  {  // k1 = 3: twiddles w16^3, w16^6, w16^9 = -c1 (1 + SIGN i tan(pi/8))
    const float2 v0 = x[12], v1 = x[13], v2 = x[14], v3 = x[15];
    const float2 u2 = csub(rot90<SIGN>(v2), v2);
    const float2 t0 = fma_s(u2, kC2, v0), t1 = fma_s(cneg(u2), kC2, v0);
    const float2 u1 = fma_s(rot90<SIGN>(v1), kT3, v1), u3 = fma_s(rot90<SIGN>(v3), kT1, v3);
    const float2 t2 = fma_s(cneg(u3), kT3, u1), t3 = fma_s(u3, kT3, u1);           // -c1/c3 = -tan(3pi/8)
    bfly4_tail<SIGN>(t0, t1, t2, t3, kC3, y[3], y[7], y[11], y[15]);
  }
#pragma unroll
  for (int i = 0; i < 16; i++) x[i] = y[i];
}

template <int SIGN>
struct Dft<16, SIGN> {
  static __device__ __forceinline__ void run(float2 (&x)[16]) {
#pragma unroll
    for (int n2 = 0; n2 < 4; n2++) {          // first layer: radix-4 over n1 on x[4 n1 + n2], result k1 left at x[4 k1 + n2]
      float2 t[4] = {x[n2], x[4 + n2], x[8 + n2], x[12 + n2]};
      Dft<4, SIGN>::run(t);
      x[n2] = t[0]; x[4 + n2] = t[1]; x[8 + n2] = t[2]; x[12 + n2] = t[3];
    }
    dft16_layerB<SIGN>(x);
  }
};

// First layer of a DFT_16 whose inputs carry the twiddles w_q (q = 4 n1 + n2), for one n2.  The four twiddles arrive in
// "mixed form" (tw_mixed below), in the order n1 = 0..3:
//   w[0] = (c, s)            full complex multiply (skipped when n2 == 0: w_0 = 1)
//   w[1] = (c_a, t_a)        q = 4+n2      t = s/c
//   w[2] = (c_b, t_b)        q = 8+n2
//   w[3] = (c_d / c_a, t_d)  q = 12+n2
// 13 packed instructions (11 for n2 = 0) against 16 for multiply-then-butterfly.  SIGN = -1 conjugates the twiddles.
template <int SIGN, bool FIRST_TRIVIAL>
__device__ __forceinline__ void dft16_layerA_tw(float2& x0, float2& x1, float2& x2, float2& x3, const float2 (&w)[4]) {
  const float2 a0 = FIRST_TRIVIAL ? x0 : (SIGN > 0 ? cmul(x0, w[0]) : cmul_conj(x0, w[0]));
  const float2 u2 = fma_s(rot90<SIGN>(x2), w[2].y, x2);
  const float2 t0 = fma_s(u2, w[2].x, a0), t1 = fma_s(cneg(u2), w[2].x, a0);
  const float2 u1 = fma_s(rot90<SIGN>(x1), w[1].y, x1), u3 = fma_s(rot90<SIGN>(x3), w[3].y, x3);
  const float2 t2 = fma_s(u3, w[3].x, u1), t3 = fma_s(cneg(u3), w[3].x, u1);
  bfly4_tail<SIGN>(t0, t1, t2, t3, w[1].x, x0, x1, x2, x3);
}
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
  static constexpr int GS = NT / 16;                 // threads that share one k0 (they exchange among themselves after pass 1)
  static constexpr int NW = NT / 32;                 // warps
  static constexpr int LOG2L = L == 1024 ? 10 : L == 2048 ? 11 : L == 4096 ? 12 : 13;
  static_assert(L == 1024 || L == 2048 || L == 4096 || L == 8192, "seg_len");
  static_assert(NB2 * GS == R1, "pass-2 butterflies per k0 group");
  // Thread roles.  Pass 1: thread t owns k0 = t / GS and k1 = t % GS + GS*u.  Pass 2 works on the same k0 values inside
  // the same warp (exchange 1 never leaves the warp: __syncwarp only).  For GS = 16 the two k0 groups of a warp are
  // interleaved over the lanes in pass 2 (lane l: k0 = 2*warp + (l & 1), n0 = l >> 1), which is what makes the padded
  // exchange-2 layout conflict-free for 64-bit stores AND 128-bit loads; for GS < 16 the natural mapping already is.
  static constexpr bool INTERLEAVE = GS == 16;
  static __device__ __forceinline__ int k0_of(int t) { return t / GS; }
  static __device__ __forceinline__ int b1_of(int t, int u) { return 16 * ((t % GS) + GS * u) + t / GS; }   // 16*k1 + k0
  static __device__ __forceinline__ int k1_of(int t, int u) { return (t % GS) + GS * u; }
  static __device__ __forceinline__ int k0_p2(int t) { return INTERLEAVE ? 2 * (t >> 5) + (t & 1) : t / GS; }
  static __device__ __forceinline__ int n0_p2(int t) { return INTERLEAVE ? (t & 31) >> 1 : t % GS; }        // + GS*u
  static __device__ __forceinline__ int b3_of(int t, int u) { return t + NT * u; }                           // n0 + R1*n1
  // Padded shared-memory exchange layouts (float2 index); every loop-variable term is a compile-time offset, so each
  // access is base register + immediate.  Constants found by exhaustive bank-conflict search:
  //   exchange 1: element (k0, n0, k1) at A1*k0 + B1*n0 + k1      (pass 1 stores n0 = 0..R1-1, pass 2 loads k1 = 0..15)
  //   exchange 2: element (n0 + R1*n1, k0) at B2*n0 + C2*n1 + k0  (pass 2 stores n1 = 0..15, pass 3 loads k0 = 0..15)
  // Even strides allow 128-bit loads of (k, k+1) pairs.  All four accesses are conflict-free for every L.
  static constexpr int A1 = L == 1024 ? 68 : L == 2048 ? 152 : L == 4096 ? 280 : 584;
  static constexpr int B1 = L == 1024 ? 17 : L == 2048 ? 18 : L == 4096 ? 17 : 18;
  static constexpr int B2 = L == 1024 ? 20 : 18;
  static constexpr int C2 = L == 1024 ? 78 : L == 2048 ? 142 : L == 4096 ? 286 : 576;
  static constexpr bool WIDE1 = (A1 % 2 == 0) && (B1 % 2 == 0);
  static constexpr bool WIDE2 = (B2 % 2 == 0) && (C2 % 2 == 0);
  static constexpr int EX1 = (A1 * 15 + B1 * (R1 - 1) + 16 + 1) / 2 * 2;    // float2 slots of exchange buffer A (>= L)
  static constexpr int EX2 = (B2 * (R1 - 1) + C2 * 15 + 16 + 1) / 2 * 2;    // float2 slots of exchange buffer B
  static_assert(EX1 >= L && EX2 >= L, "exchange buffers double as plain L-point staging arrays");
};

// exp(2 pi i * num / den), den a power of two, num reduced exactly in integers
__device__ __forceinline__ float2 unit_root(int num, int den) {
  int r = num & (den - 1);
  float s, c;
  sincospif(2.0f * (float)r / (float)den, &s, &c);
  return make_float2(c, s);
}

// Mixed-form twiddle (see dft16_layerA_tw) at table position pos = 4*n2 + n1 for the 16 input twiddles
// w_q = exp(2 pi i * e * q / den), q = 4*n1 + n2, of one DFT_16 (inverse sign).  An exactly vanishing cosine (quarter
// turns) is replaced by 1e-9: c * (v + (s/c) i v) then equals i s v up to 1e-9 |v|, far below fp32 rounding.
__device__ __forceinline__ float tw_cos_safe(float c) { return c == 0.0f ? 1e-9f : c; }
__device__ __forceinline__ float2 tw_mixed(int pos, int e, int den) {
  const int n1 = pos & 3, q = 4 * n1 + (pos >> 2);
  const float2 w = unit_root(e * q, den);
  if (n1 == 0) return w;
  const float c = tw_cos_safe(w.x);
  const float t = w.y / c;
  if (n1 == 3) return make_float2(c / tw_cos_safe(unit_root(e * (q - 8), den).x), t);
  return make_float2(c, t);
}

// Per-thread pass-3 twiddles (inverse sign): tw3[16*u + pos] = mixed form of w_L^{k0 * b3_of(t,u)}, k0 = q(pos).
template <int L>
__device__ __forceinline__ void make_tw3(float2 (&tw3)[FftGeom<L>::P], int t) {
  using G = FftGeom<L>;
#pragma unroll
  for (int u = 0; u < G::NB2; u++)
#pragma unroll
    for (int pos = 0; pos < 16; pos++) tw3[16 * u + pos] = tw_mixed(pos, G::b3_of(t, u), L);
}

// Pass-3 twiddle providers: load8(i, w) returns entries 8i..8i+7 of the thread's tw3[] array.
template <int L>
struct Tw3Regs {                                    // kept in registers (template-bank kernel)
  float2 w[FftGeom<L>::P];
  __device__ __forceinline__ void load8(int i, float2 (&o)[8]) const {
#pragma unroll
    for (int k = 0; k < 8; k++) o[k] = w[8 * i + k];
  }
};

// ---- tensor memory as a per-thread register extension (32x32b shape: thread i of warp w <-> TMEM lane 32*(w%4)+i).
// The load and its wait are ONE asm statement: tcgen05.ld fills its destination registers asynchronously, so the
// compiler must not be able to move or spill them between the two instructions.
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]), "=f"(r[9]),
        "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15]), "=f"(r[16]), "=f"(r[17]), "=f"(r[18]),
        "=f"(r[19]), "=f"(r[20]), "=f"(r[21]), "=f"(r[22]), "=f"(r[23]), "=f"(r[24]), "=f"(r[25]), "=f"(r[26]), "=f"(r[27]),
        "=f"(r[28]), "=f"(r[29]), "=f"(r[30]), "=f"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const float (&r)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
      "{%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};\n\t"
      "tcgen05.wait::st.sync.aligned;"
      :: "r"(taddr), "f"(r[0]), "f"(r[1]), "f"(r[2]), "f"(r[3]), "f"(r[4]), "f"(r[5]), "f"(r[6]), "f"(r[7]), "f"(r[8]), "f"(r[9]),
        "f"(r[10]), "f"(r[11]), "f"(r[12]), "f"(r[13]), "f"(r[14]), "f"(r[15]), "f"(r[16]), "f"(r[17]), "f"(r[18]),
        "f"(r[19]), "f"(r[20]), "f"(r[21]), "f"(r[22]), "f"(r[23]), "f"(r[24]), "f"(r[25]), "f"(r[26]), "f"(r[27]),
        "f"(r[28]), "f"(r[29]), "f"(r[30]), "f"(r[31])
      : "memory");
}

// Split form: tmem_ld32_issue starts the load, tmem_ld32_wait completes it.  The wait names the 32 registers as
// read-write operands so that no use of them can be scheduled before it (and no copy of them after the issue).
__device__ __forceinline__ void tmem_ld32_issue(uint32_t taddr, float (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]), "=f"(r[9]),
        "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15]), "=f"(r[16]), "=f"(r[17]), "=f"(r[18]),
        "=f"(r[19]), "=f"(r[20]), "=f"(r[21]), "=f"(r[22]), "=f"(r[23]), "=f"(r[24]), "=f"(r[25]), "=f"(r[26]), "=f"(r[27]),
        "=f"(r[28]), "=f"(r[29]), "=f"(r[30]), "=f"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld32_wait(float (&r)[32]) {
  asm volatile("tcgen05.wait::ld.sync.aligned;"
               : "+f"(r[0]), "+f"(r[1]), "+f"(r[2]), "+f"(r[3]), "+f"(r[4]), "+f"(r[5]), "+f"(r[6]), "+f"(r[7]), "+f"(r[8]), "+f"(r[9]),
                 "+f"(r[10]), "+f"(r[11]), "+f"(r[12]), "+f"(r[13]), "+f"(r[14]), "+f"(r[15]), "+f"(r[16]), "+f"(r[17]), "+f"(r[18]),
                 "+f"(r[19]), "+f"(r[20]), "+f"(r[21]), "+f"(r[22]), "+f"(r[23]), "+f"(r[24]), "+f"(r[25]), "+f"(r[26]), "+f"(r[27]),
                 "+f"(r[28]), "+f"(r[29]), "+f"(r[30]), "+f"(r[31])
               :
               : "memory");
}

__device__ __forceinline__ void tmem_ld16(uint32_t taddr, float (&r)[16]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3]), "=f"(r[4]), "=f"(r[5]), "=f"(r[6]), "=f"(r[7]), "=f"(r[8]), "=f"(r[9]),
        "=f"(r[10]), "=f"(r[11]), "=f"(r[12]), "=f"(r[13]), "=f"(r[14]), "=f"(r[15])
      : "r"(taddr)
      : "memory");
}

__device__ __forceinline__ void tmem_ld4(uint32_t taddr, float (&r)[4]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x4.b32 {%0,%1,%2,%3}, [%4];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3])
      : "r"(taddr)
      : "memory");
}

// four single columns taddr, taddr + 16, taddr + 32, taddr + 48 of the thread's lane
__device__ __forceinline__ void tmem_ld1x4(uint32_t taddr, float (&r)[4]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x1.b32 {%0}, [%4];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x1.b32 {%1}, [%5];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x1.b32 {%2}, [%6];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x1.b32 {%3}, [%7];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=f"(r[0]), "=f"(r[1]), "=f"(r[2]), "=f"(r[3])
      : "r"(taddr), "r"(taddr + 16), "r"(taddr + 32), "r"(taddr + 48)
      : "memory");
}

// A thread-private array of P complex values (P = 16 or 32) held in TMEM columns [addr, addr + 2P) of the thread's lane.
// load16(h, o) / store16(h, o) move entries 16h .. 16h+15; load8(i, o) entries 8i .. 8i+7.
template <int L>
struct TmemArray {
  uint32_t addr;
  __device__ __forceinline__ void load8(int i, float2 (&o)[8]) const {
    float r[16];
    tmem_ld16(addr + 16 * i, r);
#pragma unroll
    for (int k = 0; k < 8; k++) o[k] = make_float2(r[2 * k], r[2 * k + 1]);
  }
  __device__ __forceinline__ void load16(int h, float2 (&o)[16]) const {
    float r[32];
    tmem_ld32(addr + 32 * h, r);
#pragma unroll
    for (int i = 0; i < 16; i++) o[i] = make_float2(r[2 * i], r[2 * i + 1]);
  }
  __device__ __forceinline__ void issue16(int h, float (&r)[32]) const { tmem_ld32_issue(addr + 32 * h, r); }
  __device__ __forceinline__ void store16(int h, const float2 (&o)[16]) const {
    float r[32];
#pragma unroll
    for (int i = 0; i < 16; i++) {
      r[2 * i] = o[i].x;
      r[2 * i + 1] = o[i].y;
    }
    tmem_st32(addr + 32 * h, r);
  }
};

// T2 table (inverse sign) in shared memory: tw2[n1*kTw2Stride + k0] = w_256^{k0*n1}.  It is read in pass 3, where the
// row n1 = b3 / R1 is uniform over R1 consecutive lanes (broadcast loads); rows are padded to 18 float2 so that the
// rows touched by one 128-bit load instruction fall in different banks.
constexpr int kTw2Stride = 18;
// Pass-2 table (inverse sign) in shared memory: row n0 (R1 rows, padded to 18 float2) holds the 16 mixed-form input
// twiddles w_{16 R1}^{k1 n0} of the pass-2 DFT_16 over k1, in position order (pos = 4*n2 + n1, k1 = 4*n1 + n2).  The rows
// read by the 8 lanes of one 128-bit load phase are 4 (or 8) consecutive n0: bank group 4*n0 + const, conflict-free.
template <int L>
struct Tw2Table {
  static constexpr int FLOATS2 = FftGeom<L>::R1 * kTw2Stride;
};
template <int L>
__device__ __forceinline__ void fill_tw2(float2* tw2, int t, int nthreads) {
  for (int i = t; i < 16 * FftGeom<L>::R1; i += nthreads)
    tw2[(i >> 4) * kTw2Stride + (i & 15)] = tw_mixed(i & 15, i >> 4, 16 * FftGeom<L>::R1);
}

// Non-blocking barrier that protects exchange buffer B against the next transform's writes: every thread arrives when
// its pass-3 loads are done and waits (normally already complete) just before it writes B again.
struct WarBarrier {
  uint32_t bar;     // shared-memory address of an mbarrier initialised with count NT
  uint32_t parity;  // phase the next wait() must see completed
  __device__ __forceinline__ void arrive() const {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
  }
  __device__ __forceinline__ void wait() {
    uint32_t done = 0;
    while (!done) {
      asm volatile(
          "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
          : "=r"(done)
          : "r"(bar), "r"(parity)
          : "memory");
    }
    parity ^= 1u;
  }
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// mbarrier for the split write-after-read barrier of exchange buffer B: count NT, primed so that the first wait passes
template <int NT>
__device__ __forceinline__ WarBarrier war_init(unsigned long long* bar, int t) {
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(NT));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  WarBarrier w;
  w.bar = smem_u32(bar);
  w.parity = 0;
  w.arrive();
  return w;
}

// Passes 1..3 on the P points in v[].  On entry v[u*R1 + k2] = x[256*k2 + b1_of(t,u)].
// On exit v[u3*16 + n2] = X[b3_of(t,u3) + 16*R1*n2].  exA/exB: exchange buffers of FftGeom::EX1 / EX2 float2.
// All twiddles sit on the input side of a DFT_16 (decimation in time) so that they fold into its first layer:
//   pass 1: DFT_R1 over k2, no twiddle;
//   pass 2: input twiddle w_{16 R1}^{k1 n0} (shared-memory table tw2, row n0), DFT_16 over k1;
//   pass 3: input twiddle w_L^{k0 b3} (per-thread table tw3: tensor memory or registers), DFT_16 over k0.
// Tables hold the inverse-sign twiddles; SIGN < 0 conjugates them on the fly.  One __syncthreads per call; `war` must
// have been arrived at by every thread after its previous use of exB (the first call after init needs a primed barrier).
template <int L, int SIGN, class TW3>
__device__ __forceinline__ void fft_passes(float2 (&v)[FftGeom<L>::P], const TW3& tw3, const float2* __restrict__ tw2,
                                           float2* exA, float2* exB, WarBarrier& war, int t) {
  using G = FftGeom<L>;
  // ---- pass 1: DFT_R1 over k2, exchange 1 (inside the warp)
  float2* const w1 = exA + G::A1 * G::k0_of(t) + (t % G::GS);
#pragma unroll
  for (int u = 0; u < G::NB1; u++) {
    float2 a[G::R1];
#pragma unroll
    for (int i = 0; i < G::R1; i++) a[i] = v[u * G::R1 + i];
    Dft<G::R1, SIGN>::run(a);
#pragma unroll
    for (int n0 = 0; n0 < G::R1; n0++) w1[G::B1 * n0 + G::GS * u] = a[n0];   // element (k0, n0, k1 = t%GS + GS*u)
  }
  __syncwarp();
  // ---- pass 2: twiddle + DFT_16 over k1, exchange 2
  float2 b[G::NB2][16];
  const int k0p = G::k0_p2(t), n0p = G::n0_p2(t);
  {
    const float2* r1 = exA + G::A1 * k0p + G::B1 * n0p;
#pragma unroll
    for (int u = 0; u < G::NB2; u++) {
      if constexpr (G::WIDE1) {
#pragma unroll
        for (int k1 = 0; k1 < 16; k1 += 2) {
          const float4 x = *reinterpret_cast<const float4*>(r1 + G::B1 * G::GS * u + k1);
          b[u][k1] = make_float2(x.x, x.y);
          b[u][k1 + 1] = make_float2(x.z, x.w);
        }
      } else {
#pragma unroll
        for (int k1 = 0; k1 < 16; k1++) b[u][k1] = r1[G::B1 * G::GS * u + k1];
      }
    }
  }
  __syncwarp();                       // exA may be rewritten by this warp's next transform
#pragma unroll
  for (int u = 0; u < G::NB2; u++) {
    const float4* trow = reinterpret_cast<const float4*>(tw2 + (n0p + G::GS * u) * kTw2Stride);
#pragma unroll
    for (int n2 = 0; n2 < 4; n2++) {
      const float4 wa = trow[2 * n2], wb = trow[2 * n2 + 1];
      const float2 w[4] = {make_float2(wa.x, wa.y), make_float2(wa.z, wa.w), make_float2(wb.x, wb.y), make_float2(wb.z, wb.w)};
      if (n2 == 0) dft16_layerA_tw<SIGN, true>(b[u][0], b[u][4], b[u][8], b[u][12], w);
      else dft16_layerA_tw<SIGN, false>(b[u][n2], b[u][4 + n2], b[u][8 + n2], b[u][12 + n2], w);
    }
    dft16_layerB<SIGN>(b[u]);
  }
  war.wait();                         // every thread has finished reading exB from the previous transform
  {
    float2* w2 = exB + G::B2 * n0p + k0p;
#pragma unroll
    for (int u = 0; u < G::NB2; u++)
#pragma unroll
      for (int n1 = 0; n1 < 16; n1++) w2[G::B2 * G::GS * u + G::C2 * n1] = b[u][n1];   // element (n0 + R1*n1, k0)
  }
  __syncthreads();
  // ---- pass 3: twiddle + DFT_16 over k0
  {
    const float2* r2 = exB + G::B2 * (t % G::R1) + G::C2 * (t / G::R1);              // b3 = t + NT*u: n0 = t % R1, n1 = t / R1 + (NT/R1)*u
#pragma unroll
    for (int u = 0; u < G::NB2; u++) {
      if constexpr (G::WIDE2) {
#pragma unroll
        for (int q = 0; q < 16; q += 2) {
          const float4 x = *reinterpret_cast<const float4*>(r2 + G::C2 * (G::NT / G::R1) * u + q);
          b[u][q] = make_float2(x.x, x.y);
          b[u][q + 1] = make_float2(x.z, x.w);
        }
      } else {
#pragma unroll
        for (int q = 0; q < 16; q++) b[u][q] = r2[G::C2 * (G::NT / G::R1) * u + q];
      }
    }
  }
  war.arrive();
#pragma unroll
  for (int u = 0; u < G::NB2; u++) {
#pragma unroll
    for (int half = 0; half < 2; half++) {
      float2 w8[8];
      tw3.load8(2 * u + half, w8);
#pragma unroll
      for (int m = 0; m < 2; m++) {
        const int n2 = 2 * half + m;
        const float2 w[4] = {w8[4 * m], w8[4 * m + 1], w8[4 * m + 2], w8[4 * m + 3]};
        if (n2 == 0) dft16_layerA_tw<SIGN, true>(b[u][0], b[u][4], b[u][8], b[u][12], w);
        else dft16_layerA_tw<SIGN, false>(b[u][n2], b[u][4 + n2], b[u][8 + n2], b[u][12 + n2], w);
      }
    }
    dft16_layerB<SIGN>(b[u]);
#pragma unroll
    for (int n2 = 0; n2 < 16; n2++) v[u * 16 + n2] = b[u][n2];
  }
}

}  // namespace jerk
