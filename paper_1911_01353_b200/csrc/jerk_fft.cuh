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

// Per-thread T1 twiddles for the INVERSE transform: tw1[u*R1 + n0] = w_L^{b1*n0}, b1 = b1_of(t, u).
template <int L>
__device__ __forceinline__ void make_tw1(float2 (&tw1)[FftGeom<L>::P], int t) {
  using G = FftGeom<L>;
#pragma unroll
  for (int u = 0; u < G::NB1; u++) {
    int b1 = G::b1_of(t, u);
#pragma unroll
    for (int n0 = 0; n0 < G::R1; n0++) tw1[u * G::R1 + n0] = unit_root(b1 * n0, L);
  }
}

// T1 twiddle providers: load16(h, w) returns entries 16h..16h+15 of the thread's tw1[] array.
template <int L>
struct Tw1Regs {                                    // kept in registers (template-bank kernel)
  float2 w[FftGeom<L>::P];
  __device__ __forceinline__ void load16(int h, float2 (&o)[16]) const {
#pragma unroll
    for (int i = 0; i < 16; i++) o[i] = w[16 * h + i];
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

// A thread-private array of P complex values (P = 16 or 32) held in TMEM columns [addr, addr + 2P) of the thread's lane.
// load16(h, o) / store16(h, o) move entries 16h .. 16h+15.
template <int L>
struct TmemArray {
  uint32_t addr;
  __device__ __forceinline__ void load16(int h, float2 (&o)[16]) const {
    float r[32];
    tmem_ld32(addr + 32 * h, r);
#pragma unroll
    for (int i = 0; i < 16; i++) o[i] = make_float2(r[2 * i], r[2 * i + 1]);
  }
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
constexpr int kTw2Floats2 = 16 * kTw2Stride;
__device__ __forceinline__ void fill_tw2(float2* tw2, int t, int nthreads) {
  for (int i = t; i < 256; i += nthreads) tw2[(i >> 4) * kTw2Stride + (i & 15)] = unit_root((i >> 4) * (i & 15), 256);
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

// Passes 1..3 on the P points in v[].  On entry v[u*R1 + k2] = x[256*k2 + b1_of(t,u)].
// On exit v[u3*16 + n2] = X[b3_of(t,u3) + 16*R1*n2].  exA/exB: exchange buffers of FftGeom::EX1 / EX2 float2.
// tw1: inverse-sign per-thread T1 twiddles (conjugated here when SIGN < 0).  One __syncthreads per call; `war` must have
// been arrived at by every thread after its previous use of exB (the first call after init needs a primed barrier).
template <int L, int SIGN, class TW1>
__device__ __forceinline__ void fft_passes(float2 (&v)[FftGeom<L>::P], const TW1& tw1, const float2* __restrict__ tw2,
                                           float2* exA, float2* exB, WarBarrier& war, int t) {
  using G = FftGeom<L>;
  // ---- pass 1: DFT_R1 over k2, twiddle T1, exchange 1 (inside the warp); 16 array entries (16/R1 butterflies) at a time
  float2* const w1 = exA + G::A1 * G::k0_of(t) + (t % G::GS);
#pragma unroll
  for (int h = 0; h < G::P / 16; h++) {
    constexpr int BPH = 16 / G::R1 > 0 ? 16 / G::R1 : 1;     // butterflies per block of 16 entries (R1 = 32: handled below)
    if constexpr (G::R1 <= 16) {
#pragma unroll
      for (int ub = 0; ub < BPH; ub++) {
        float2 a[G::R1];
#pragma unroll
        for (int i = 0; i < G::R1; i++) a[i] = v[16 * h + ub * G::R1 + i];
        Dft<G::R1, SIGN>::run(a);
#pragma unroll
        for (int i = 0; i < G::R1; i++) v[16 * h + ub * G::R1 + i] = a[i];
      }
    } else if (h == 0) {
      Dft<G::R1, SIGN>::run(v);                                // R1 = 32 = P: one butterfly over the whole array
    }
    float2 w[16];
    tw1.load16(h, w);
#pragma unroll
    for (int i = 0; i < 16; i++) {
      const int e = 16 * h + i, u = e / G::R1, n0 = e % G::R1;
      float2 r = n0 == 0 ? v[e] : (SIGN > 0 ? cmul(v[e], w[i]) : cmul_conj(v[e], w[i]));
      w1[G::B1 * n0 + G::GS * u] = r;                          // element (k0, n0, k1 = t%GS + GS*u)
    }
  }
  __syncwarp();
  // ---- pass 2: DFT_16 over k1, exchange 2
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
  for (int u = 0; u < G::NB2; u++) Dft<16, SIGN>::run(b[u]);
  war.wait();                         // every thread has finished reading exB from the previous transform
  {
    float2* w2 = exB + G::B2 * n0p + k0p;
#pragma unroll
    for (int u = 0; u < G::NB2; u++)
#pragma unroll
      for (int n1 = 0; n1 < 16; n1++) w2[G::B2 * G::GS * u + G::C2 * n1] = b[u][n1];   // element (n0 + R1*n1, k0)
  }
  __syncthreads();
  // ---- pass 3 (the T2 twiddle w_256^{k0*n1} is applied here, on the read side: its row n1 is lane-uniform)
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
    const int b3 = G::b3_of(t, u);
    const float2* trow = tw2 + (b3 / G::R1) * kTw2Stride;
#pragma unroll
    for (int q = 1; q < 16; q++) b[u][q] = SIGN > 0 ? cmul(b[u][q], trow[q]) : cmul_conj(b[u][q], trow[q]);
    Dft<16, SIGN>::run(b[u]);
#pragma unroll
    for (int n2 = 0; n2 < 16; n2++) v[u * 16 + n2] = b[u][n2];
  }
}

}  // namespace jerk
