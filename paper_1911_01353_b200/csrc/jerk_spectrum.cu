// jerk_spectrum.cu — spectrum preparation upstream of the jerk search (BASELINE.json configs[0]:
// "The real FFT gives 32768 complex bins, normalised to unit mean power per 1000-bin block"; reading S15).
//
//   X[k] = sum_n x[n] exp(-2 pi i k n / N), k = 0 .. N/2-1 (DC kept, Nyquist dropped);  every `block`-bin block / sqrt(mean |X|^2)
//
// The real series of N = 2^m samples is read as M = N/2 complex points z[j] = x[2j] + i x[2j+1]; FFT_M(z) is a four-step
// transform M = M1 x M2 built from the register/shared-memory FFT of jerk_fft.cuh (three launches, each one read and
// one write of the 8M-byte array, HBM-bound):
//   k_fft_strided (A)  for every n2 < M2: Y[k1][n2] = w_M^{n2 k1} * DFT_M1 over n1 of z[M2 n1 + n2]          (columns)
//   k_fft_strided (B)  for every k1 < M1: Z[k1 + M1 k2] = DFT_M2 over n2 of Y[k1][n2]                          (rows)
//   k_untangle_norm    X[k] = (Z[k] + conj Z[M-k])/2 - i exp(-i pi k / M) (Z[k] - conj Z[M-k])/2, block power, scale
// M2 = 4096 for M >= 2^22, else 1024; M1 = M / M2 in {1 .. 4096}; lengths below 1024 use a direct DFT (tiny inputs only).
// Both FFT launches stage their transforms through a shared-memory tile so that the strided side moves whole sectors.
#include <cuda_runtime.h>
#include <stdint.h>

#include <mutex>

#include "../../include/jerk.h"
#include "jerk_fft.cuh"

namespace jerk {

struct StridedFft {
  const float2* in;
  float2* out;
  long long in_sb, in_se, out_sb, out_se;  // strides in float2 units: batch b, element e at in[b*in_sb + e*in_se]
  int nbatch;                              // number of transforms
  int per_cta;                             // consecutive batches handled by one CTA (sector reuse of the strided side)
  int tw_den;                              // 0: none; else output k of batch b is multiplied by exp(-2 pi i b k / tw_den)
};

// C transforms (consecutive batch indices) per CTA, staged through a shared-memory tile so that every global access moves
// whole 32-byte sectors whichever of the two index directions is contiguous in memory: when the elements of a transform
// are contiguous (stride 1) a thread moves 16 bytes of one transform, when the batches are contiguous it moves the C
// neighbouring values of one element index (C * 8 bytes).  The tile is padded by one slot per 16 so that the FFT's
// register layout (stride-16 gathers) reads it without bank conflicts.
template <int L>
struct TileGeom {
  static constexpr int C = L <= 2048 ? 4 : 2;            // transforms per CTA
  static constexpr int ROW = L + L / 16;                 // padded row length in float2
  static __device__ __forceinline__ int at(int e) { return e + (e >> 4); }
};

template <int L>
__global__ void __launch_bounds__(FftGeom<L>::NT) k_fft_strided(StridedFft a) {
  using Gm = FftGeom<L>;
  using Tg = TileGeom<L>;
  constexpr int C = Tg::C, NT = Gm::NT;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* exA = reinterpret_cast<float2*>(smem_raw);
  float2* exB = exA + Gm::EX1;
  float2* tw2 = exB + Gm::EX2;
  float2* tile = tw2 + Tw2Table<L>::FLOATS2;             // [C][ROW]
  __shared__ unsigned long long s_war;
  const int t = threadIdx.x;
  fill_tw2<L>(tw2, t, NT);
  Tw3Regs<L> tw3;
  make_tw3<L>(tw3.w, t);
  WarBarrier war = war_init<NT>(&s_war, t);
  const int b0 = blockIdx.x * C;                          // nbatch is a multiple of C (host checks)
  // ---- load
  if (a.in_se == 1) {
    for (int c = 0; c < C; c++) {
      const float4* src = reinterpret_cast<const float4*>(a.in + (long long)(b0 + c) * a.in_sb);
      for (int e2 = t; e2 < L / 2; e2 += NT) {
        const float4 x = src[e2];
        tile[c * Tg::ROW + Tg::at(2 * e2)] = make_float2(x.x, x.y);
        tile[c * Tg::ROW + Tg::at(2 * e2 + 1)] = make_float2(x.z, x.w);
      }
    }
  } else {                                                // in_sb == 1
    for (int e = t; e < L; e += NT) {
      const float4* src = reinterpret_cast<const float4*>(a.in + b0 + (long long)e * a.in_se);
#pragma unroll
      for (int h = 0; h < C / 2; h++) {
        const float4 x = src[h];
        tile[(2 * h) * Tg::ROW + Tg::at(e)] = make_float2(x.x, x.y);
        tile[(2 * h + 1) * Tg::ROW + Tg::at(e)] = make_float2(x.z, x.w);
      }
    }
  }
  __syncthreads();
  // ---- transforms, in place in the tile
  for (int c = 0; c < C; c++) {
    float2* row = tile + c * Tg::ROW;
    float2 v[Gm::P];
#pragma unroll
    for (int u = 0; u < Gm::NB1; u++)
#pragma unroll
      for (int k2 = 0; k2 < Gm::R1; k2++) v[u * Gm::R1 + k2] = row[Tg::at(256 * k2 + Gm::b1_of(t, u))];
    fft_passes<L, -1>(v, tw3, tw2, exA, exB, war, t);     // its block barrier orders every read of `row` before the writes below
    const int b = b0 + c;
#pragma unroll
    for (int u = 0; u < Gm::NB2; u++)
#pragma unroll
      for (int n2 = 0; n2 < 16; n2++) {
        const int k = Gm::b3_of(t, u) + 16 * Gm::R1 * n2;
        float2 x = v[u * 16 + n2];
        if (a.tw_den) x = cmul(x, unit_root(-(b * k), a.tw_den));
        row[Tg::at(k)] = x;
      }
  }
  __syncthreads();
  // ---- store
  if (a.out_se == 1) {
    for (int c = 0; c < C; c++) {
      float4* dst = reinterpret_cast<float4*>(a.out + (long long)(b0 + c) * a.out_sb);
      for (int e2 = t; e2 < L / 2; e2 += NT) {
        const float2 p = tile[c * Tg::ROW + Tg::at(2 * e2)], q = tile[c * Tg::ROW + Tg::at(2 * e2 + 1)];
        dst[e2] = make_float4(p.x, p.y, q.x, q.y);
      }
    }
  } else {                                                // out_sb == 1
    for (int e = t; e < L; e += NT) {
      float4* dst = reinterpret_cast<float4*>(a.out + b0 + (long long)e * a.out_se);
#pragma unroll
      for (int h = 0; h < C / 2; h++) {
        const float2 p = tile[(2 * h) * Tg::ROW + Tg::at(e)], q = tile[(2 * h + 1) * Tg::ROW + Tg::at(e)];
        dst[h] = make_float4(p.x, p.y, q.x, q.y);
      }
    }
  }
}

// Direct DFT for lengths below 1024 (time series shorter than 2^21 samples): one thread per output.
__global__ void __launch_bounds__(256) k_dft_direct(StridedFft a, int L) {
  const long long idx = (long long)blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= (long long)a.nbatch * L) return;
  const int b = (int)(idx % a.nbatch), k = (int)(idx / a.nbatch);   // batch fastest: neighbouring threads read neighbouring columns
  const float2* src = a.in + (long long)b * a.in_sb;
  double re = 0.0, im = 0.0;
  for (int e = 0; e < L; e++) {
    const float2 x = src[(long long)e * a.in_se];
    const float2 w = unit_root(-(e * k), L);
    re += (double)x.x * w.x - (double)x.y * w.y;
    im += (double)x.x * w.y + (double)x.y * w.x;
  }
  float2 r = make_float2((float)re, (float)im);
  if (a.tw_den) r = cmul(r, unit_root(-(b * k), a.tw_den));
  a.out[(long long)b * a.out_sb + (long long)k * a.out_se] = r;
}

// untangled real-input spectrum bin k from the half-length transform Z (M points)
__device__ __forceinline__ float2 untangle_bin(const float2* __restrict__ Z, int M, int k) {
  if (k == 0) {
    const float2 z0 = Z[0];
    return make_float2(z0.x + z0.y, 0.f);
  }
  const float2 zk = Z[k], zm = Z[M - k];
  const float2 e = make_float2(0.5f * (zk.x + zm.x), 0.5f * (zk.y - zm.y));   // (Z[k] + conj Z[M-k]) / 2
  const float2 o = make_float2(0.5f * (zk.x - zm.x), 0.5f * (zk.y + zm.y));   // (Z[k] - conj Z[M-k]) / 2
  float s, c;
  sincospif((float)k / (float)M, &s, &c);                                     // exp(-i pi k/M) = (c, -s)
  return make_float2(e.x + (-s * o.x + c * o.y), e.y + (-c * o.x - s * o.y));  // e - i exp(-i pi k/M) o
}

// One CTA per normalisation block: untangle the half-length transform into the real-input spectrum, reduce the block's
// power in a fixed order (deterministic), scale.  Every thread re-reads only what it wrote itself.
__global__ void __launch_bounds__(256) k_untangle_norm(const float2* __restrict__ Z, float2* __restrict__ X, int M, int block) {
  const int k_lo = blockIdx.x * block, k_hi = min(M, k_lo + block);
  double acc = 0.0;
  for (int k = k_lo + threadIdx.x; k < k_hi; k += 256) {
    const float2 x = untangle_bin(Z, M, k);
    X[k] = x;
    acc += (double)x.x * x.x + (double)x.y * x.y;
  }
  __shared__ double s_part[8];
  __shared__ float s_scale;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
  if ((threadIdx.x & 31) == 0) s_part[threadIdx.x >> 5] = acc;
  __syncthreads();
  if (threadIdx.x == 0) {
    double tot = 0.0;
    for (int w = 0; w < 8; w++) tot += s_part[w];
    const double mean = tot / (double)(k_hi - k_lo);
    s_scale = mean > 0.0 ? (float)(1.0 / sqrt(mean)) : 1.0f;
  }
  __syncthreads();
  const float sc = s_scale;
  for (int k = k_lo + threadIdx.x; k < k_hi; k += 256) {
    const float2 x = X[k];
    X[k] = make_float2(x.x * sc, x.y * sc);
  }
}

// Block starts of the red-noise variant (N1 reading): lengths 6, 7, 8, ... growing by len / 8 (at least 1) up
// to `block`; bounds[0 .. nblk] with bounds[nblk] = M, nblk stored in bounds[-1 + cap] ... by one thread (a few hundred
// steps at most before the lengths saturate, then M / block more).
__global__ void k_rednoise_bounds(int* bounds, int cap, int M, int block) {
  if (blockIdx.x || threadIdx.x) return;
  int n = 0, k = 0, len = 6;
  bounds[0] = 0;
  while (k + len < M && n + 2 < cap) {
    k += len;
    bounds[++n] = k;
    const int g = len / 8;
    len = min(block, len + (g > 1 ? g : 1));
  }
  bounds[++n] = M;
  bounds[cap] = n;        // number of blocks
}

// Median variants (SURVEY.md 8(f) N1 "median-based and red-noise variants"): one CTA per normalisation block
// [lo, hi): untangle, powers into shared memory, bitonic sort, median (mean of the two middle values for an even
// count), scale by 1 / sqrt(median / ln 2).  bounds == nullptr: uniform blocks of `block` bins.
__global__ void __launch_bounds__(256) k_untangle_norm_median(const float2* __restrict__ Z, float2* __restrict__ X, int M, int block,
                                                              const int* __restrict__ bounds, int cap) {
  extern __shared__ float s_pow[];      // next power of two >= block
  __shared__ float s_scale;
  int k_lo, k_hi;
  if (bounds) {
    if ((int)blockIdx.x >= bounds[cap]) return;
    k_lo = bounds[blockIdx.x];
    k_hi = bounds[blockIdx.x + 1];
  } else {
    k_lo = blockIdx.x * block;
    k_hi = min(M, k_lo + block);
  }
  const int n = k_hi - k_lo;
  int np2 = 1;
  while (np2 < n) np2 <<= 1;
  for (int i = threadIdx.x; i < np2; i += 256) {
    float pw = INFINITY;                 // padding sorts to the end
    if (i < n) {
      const float2 x = untangle_bin(Z, M, k_lo + i);
      X[k_lo + i] = x;
      pw = fmaf(x.x, x.x, x.y * x.y);
    }
    s_pow[i] = pw;
  }
  __syncthreads();
  for (int size = 2; size <= np2; size <<= 1)
    for (int stride = size >> 1; stride > 0; stride >>= 1) {
      for (int i = threadIdx.x; i < np2 / 2; i += 256) {
        const int lo = 2 * i - (i & (stride - 1));          // element whose bit `stride` is 0
        const int hi = lo + stride;
        const bool up = (lo & size) == 0;
        const float a = s_pow[lo], b = s_pow[hi];
        if ((a > b) == up) {
          s_pow[lo] = b;
          s_pow[hi] = a;
        }
      }
      __syncthreads();
    }
  if (threadIdx.x == 0) {
    const float med = (n & 1) ? s_pow[n / 2] : 0.5f * (s_pow[n / 2 - 1] + s_pow[n / 2]);
    s_scale = med > 0.f ? (float)(1.0 / sqrt((double)med / 0.69314718055994530942)) : 1.0f;
  }
  __syncthreads();
  const float sc = s_scale;
  for (int k = k_lo + threadIdx.x; k < k_hi; k += 256) {   // every thread re-reads only what it wrote itself
    const float2 x = X[k];
    X[k] = make_float2(x.x * sc, x.y * sc);
  }
}

template <int L>
static cudaError_t launch_strided(const StridedFft& a, cudaStream_t st) {
  using Gm = FftGeom<L>;
  using Tg = TileGeom<L>;
  if (a.nbatch % Tg::C) return cudaErrorInvalidValue;
  if (!((a.in_se == 1 || a.in_sb == 1) && (a.out_se == 1 || a.out_sb == 1))) return cudaErrorInvalidValue;
  const size_t smem = (size_t)(Gm::EX1 + Gm::EX2 + Tw2Table<L>::FLOATS2 + Tg::C * Tg::ROW) * sizeof(float2);
  cudaError_t e = cudaFuncSetAttribute(k_fft_strided<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_fft_strided<L><<<a.nbatch / Tg::C, Gm::NT, smem, st>>>(a);
  return cudaGetLastError();
}

static cudaError_t run_fft(const StridedFft& a, int L, cudaStream_t st) {
  const bool tiled = (L == 1024 && a.nbatch % TileGeom<1024>::C == 0) || (L == 2048 && a.nbatch % TileGeom<2048>::C == 0) ||
                     (L == 4096 && a.nbatch % TileGeom<4096>::C == 0);   // one or two transforms only (2^11, 2^12 samples): direct DFT
  switch (tiled ? L : 0) {
    case 1024: return launch_strided<1024>(a, st);
    case 2048: return launch_strided<2048>(a, st);
    case 4096: return launch_strided<4096>(a, st);
  }
  const long long n = (long long)a.nbatch * L;
  k_dft_direct<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(a, L);
  return cudaGetLastError();
}

}  // namespace jerk

using namespace jerk;

// ---------------------------------------------------------------------------------------------------------------------
// jerk_prepare_spectrum_static: spectrum preparation for callers that cannot hand the library a scratch buffer
// (include/jerk.h has the user-facing text).  The intermediate array Z of the four-step transform lives in the
// file-scope device array below instead of in caller memory.  8 MiB per GPU that loads the library, held until the
// process exits, which is why the limit is 2^21 samples and not the 2^25 of the caller-scratch entry points.
//
// g_static_scratch is a device symbol: in host code its name is only a handle (a host-side shadow variable), never
// a device address, so nothing in this file passes `g_static_scratch` or `&g_static_scratch[0]` to a kernel.  The
// address a kernel can use comes from cudaGetSymbolAddress, asked once per device with that device current; every
// device has its own copy of the array at its own address, hence the table indexed by device ordinal.
constexpr int64_t kStaticMaxSamples = JERK_STATIC_SPECTRUM_MAX_SAMPLES;
constexpr uint64_t kStaticScratchBytes = (uint64_t)(kStaticMaxSamples / 2) * sizeof(float2);
constexpr int kStaticMaxDevices = 64;
static __device__ __align__(256) unsigned char g_static_scratch[kStaticScratchBytes];
static void* g_static_scratch_addr[kStaticMaxDevices];   // [device ordinal] -> device address of that device's copy (null: not asked yet)
static std::mutex g_static_scratch_mutex;

// Device address of the current device's copy of g_static_scratch (looked up on the first call per device).
static int static_scratch_for_current_device(void** out) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) return JERK_ENODEV;
  if (dev < 0 || dev >= kStaticMaxDevices) return JERK_ENODEV;
  std::lock_guard<std::mutex> lock(g_static_scratch_mutex);
  if (!g_static_scratch_addr[dev]) {
    void* ptr = nullptr;
    if (cudaGetSymbolAddress((void**)&ptr, g_static_scratch) != cudaSuccess || !ptr) {
      (void)cudaGetLastError();   // leave no sticky "last error" behind for the caller's next launch check
      return JERK_ECUDA;
    }
    g_static_scratch_addr[dev] = ptr;
  }
  *out = g_static_scratch_addr[dev];
  return JERK_OK;
}

extern "C" {

// blocks of the red-noise schedule are at least 6 bins long: M / 6 + 2 starts at most, + the count
static uint64_t bounds_cap(int64_t nsamples) { return (uint64_t)(nsamples / 2) / 6 + 4; }

uint64_t jerk_spectrum_scratch_bytes(int64_t nsamples) {
  if (nsamples < 2) return 0;
  return (uint64_t)(nsamples / 2) * sizeof(float2) + (bounds_cap(nsamples) + 1) * sizeof(int);
}

int jerk_prepare_spectrum(const float* d_series, int64_t nsamples, int block, void* d_spec, void* d_scratch, uint64_t scratch_bytes,
                          void* stream) {
  return jerk_prepare_spectrum_mode(d_series, nsamples, block, JERK_NORM_MEAN, d_spec, d_scratch, scratch_bytes, stream);
}

int jerk_prepare_spectrum_mode(const float* d_series, int64_t nsamples, int block, int mode, void* d_spec, void* d_scratch,
                               uint64_t scratch_bytes, void* stream) {
  if (!d_series || !d_spec || !d_scratch || block < 1) return JERK_EINVAL;
  if (mode != JERK_NORM_MEAN && mode != JERK_NORM_MEDIAN && mode != JERK_NORM_REDNOISE) return JERK_EINVAL;
  if (mode != JERK_NORM_MEAN && block > 4096) return JERK_EINVAL;      // the block is sorted in shared memory
  if (mode == JERK_NORM_REDNOISE && block < 8) return JERK_EINVAL;
  if (nsamples < (1 << 11) || nsamples > (1 << 25) || (nsamples & (nsamples - 1))) return JERK_EINVAL;   // 2^11 .. 2^25 samples
  // the red-noise block table sits behind the transform scratch; the other modes need the transform scratch only
  if (scratch_bytes < (mode == JERK_NORM_REDNOISE ? jerk_spectrum_scratch_bytes(nsamples) : (uint64_t)(nsamples / 2) * sizeof(float2))) return JERK_ENOMEM;
  if ((uintptr_t)d_series % 16 || (uintptr_t)d_spec % 16 || (uintptr_t)d_scratch % 16) return JERK_EINVAL;   // 128-bit accesses
  int dev = 0, major = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess ||
      major != 10)
    return JERK_ENODEV;   // sm_100 only: this library has no other code path
  cudaStream_t st = (cudaStream_t)stream;
  const int M = (int)(nsamples / 2);
  const int M2 = M >= (1 << 22) ? 4096 : 1024;
  const int M1 = M / M2;
  float2* Y = (float2*)d_spec;       // step A output lives in the result buffer; step B writes the scratch buffer
  float2* Z = (float2*)d_scratch;
  StridedFft a;
  a.in = (const float2*)d_series;
  a.out = Y;
  a.in_sb = 1;
  a.in_se = M2;
  a.out_sb = 1;
  a.out_se = M2;
  a.nbatch = M2;
  a.per_cta = 4;
  a.tw_den = M;
  if (run_fft(a, M1, st) != cudaSuccess) return JERK_ECUDA;
  StridedFft b;
  b.in = Y;
  b.out = Z;
  b.in_sb = M2;
  b.in_se = 1;
  b.out_sb = 1;
  b.out_se = M1;
  b.nbatch = M1;
  b.per_cta = M1 >= 4 ? 4 : 1;
  b.tw_den = 0;
  if (run_fft(b, M2, st) != cudaSuccess) return JERK_ECUDA;
  if (mode == JERK_NORM_MEAN) {
    k_untangle_norm<<<(M + block - 1) / block, 256, 0, st>>>(Z, (float2*)d_spec, M, block);
  } else {
    int np2 = 1;
    while (np2 < block) np2 <<= 1;
    const size_t smem = (size_t)np2 * sizeof(float);
    if (mode == JERK_NORM_MEDIAN) {
      k_untangle_norm_median<<<(M + block - 1) / block, 256, smem, st>>>(Z, (float2*)d_spec, M, block, nullptr, 0);
    } else {
      int* bounds = (int*)((unsigned char*)d_scratch + (size_t)M * sizeof(float2));
      const int cap = (int)bounds_cap(nsamples);
      k_rednoise_bounds<<<1, 32, 0, st>>>(bounds, cap, M, block);
      // an upper bound on the number of blocks (the growth phase has fewer than 64): surplus CTAs leave at once
      k_untangle_norm_median<<<M / block + 66, 256, smem, st>>>(Z, (float2*)d_spec, M, block, bounds, cap);
    }
  }
  if (cudaGetLastError() != cudaSuccess) return JERK_ECUDA;
  return JERK_OK;
}

int jerk_prepare_spectrum_static(const float* d_series, int64_t nsamples, int block, void* d_spec, void* stream) {
  if (!d_series || !d_spec || block < 1) return JERK_EINVAL;
  if (nsamples > kStaticMaxSamples) return JERK_ELIMIT;   // before anything else looks at the size: the array cannot grow
  void* scratch = nullptr;
  const int rc = static_scratch_for_current_device(&scratch);
  if (rc != JERK_OK) return rc;
  // Same three launches as jerk_prepare_spectrum, with Z in the static array.  Launch B writes all nsamples/2 elements
  // of Z before the third launch reads them, so whatever an earlier call left in the array is never read and nothing
  // has to be cleared.  No cudaMalloc / cudaFree / allocating library call on this path.
  return jerk_prepare_spectrum_mode(d_series, nsamples, block, JERK_NORM_MEAN, d_spec, scratch, kStaticScratchBytes, stream);
}

}  // extern "C"
