// bench_probes.cu -- measurement aids of bench.py, NOT part of the library (libjerk_b200.so / include/jerk.h).
// Built by bench.py (and __graft_entry__.build) into bench_probes.so beside it:
//   nvcc -gencode arch=compute_100a,code=sm_100a -O3 -lineinfo -Xcompiler -fPIC -shared -o bench_probes.so bench_probes.cu
//
//   bench_probe_fma    roofline denominator check ("the bench must also run a pure-FFMA micro-kernel"):
//                      launches a kernel of nothing but independent FP32 fused multiply-add chains (2048 threads per SM,
//                      16 chains per thread, `iters` iterations) on `stream` and returns in *flops (HOST) the number of
//                      floating-point operations it executes; the caller times it.  d_out: DEVICE, >= 4 bytes.
//   bench_probe_issue  issue-slot model of the search kernel: six short kernels at the occupancy of
//                      k_search64 (8 warps per SM, two per scheduler); every round of a warp is 8 independent packed FP32
//                      fused multiply-adds followed by 4 companion instructions of one kind: [0] none, [1] integer
//                      byte-permute, [2] 128-bit shared-memory load, [3] three-input FP32 maximum with |.| operands,
//                      [4] scalar FP32 fused multiply-add, [5] warp shuffle.  h_cycles_per_round (HOST, 6 doubles)
//                      receives the scheduler cycles one round takes.  Synchronises `stream`.  d_scratch: DEVICE, >= 256
//                      bytes, 8-byte aligned.
// Both return 0 or a negative status (-1 bad argument, -5 no device, -3 CUDA error).
#include <cuda_runtime.h>
#include <stdint.h>

enum { PROBE_OK = 0, PROBE_EINVAL = -1, PROBE_ECUDA = -3, PROBE_ENODEV = -5 };

namespace {

// Measurement aid ("the bench must also run a pure-FFMA micro-kernel"): 16 independent fused multiply-add
// chains per thread, nothing else; flops = threads * iters * 16 * 2.
__global__ void __launch_bounds__(256) k_ffma_probe(float* out, int iters) {
  float a[16];
#pragma unroll
  for (int i = 0; i < 16; i++) a[i] = 1.0f + 1e-3f * (float)(threadIdx.x + i);
  const float m = 0.999f + 1e-6f * (float)(blockIdx.x & 7), c = 1e-3f;
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 16; i++) a[i] = fmaf(a[i], m, c);
  }
  float s = 0.f;
#pragma unroll
  for (int i = 0; i < 16; i++) s += a[i];
  if (s == 12345.678f) out[0] = s;   // never true: keeps the chains alive without memory traffic
}

// ---- issue-slot probe (measurement aid): packed FP32 instructions with companions of another kind
__device__ __forceinline__ float2 probe_ffma2(float2 a, float2 b, float2 c) {
  float2 d;
  asm volatile("fma.rn.f32x2 %0, %1, %2, %3;"
               : "=l"(*reinterpret_cast<unsigned long long*>(&d))
               : "l"(*reinterpret_cast<unsigned long long*>(&a)), "l"(*reinterpret_cast<unsigned long long*>(&b)),
                 "l"(*reinterpret_cast<unsigned long long*>(&c)));
  return d;
}
// 8 warps per SM (two per scheduler, as in k_search64).  Every round: 8 independent packed FMAs, then 4 companions
// chosen by KIND: 0 none, 1 integer byte-permute (ALU pipe), 2 128-bit shared-memory load, 3 three-input FP32 maximum
// with |.| operands, 4 scalar FP32 FMA, 5 warp shuffle.  cycles[KIND] = clock64 cycles of warp 0 of CTA 0.
template <int KIND>
__global__ void __launch_bounds__(256, 1) k_issue_probe(float* out, int iters, long long* cycles) {
  extern __shared__ float4 probe_sm[];
  float2 a[8];
#pragma unroll
  for (int i = 0; i < 8; i++) a[i] = make_float2(threadIdx.x * 0.001f + i, i * 0.5f);
  const float2 b = make_float2(1.0001f, 0.9999f), c = make_float2(1e-6f, -1e-6f);
  for (int i = threadIdx.x; i < 4096; i += blockDim.x) probe_sm[i] = make_float4((float)i, 1.f, 2.f, 3.f);
  __syncthreads();
  float m0 = 0.f, m1 = 0.f, m2 = 0.f, m3 = 0.f, s0 = 1.f, s1 = 2.f, s2 = 3.f, s3 = 4.f;
  int ia = threadIdx.x, ib = 1;
  const unsigned p = (unsigned)__cvta_generic_to_shared(probe_sm + threadIdx.x);
  const long long t0 = clock64();
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 16; r++) {
#pragma unroll
      for (int i = 0; i < 8; i++) a[i] = probe_ffma2(a[i], b, c);
      if (KIND == 1) {
        asm volatile("prmt.b32 %0, %0, %1, 0x3210;" : "+r"(ia) : "r"(ib));
        asm volatile("prmt.b32 %0, %0, %1, 0x3210;" : "+r"(ib) : "r"(ia));
        asm volatile("prmt.b32 %0, %0, %1, 0x3210;" : "+r"(ia) : "r"(ib));
        asm volatile("prmt.b32 %0, %0, %1, 0x3210;" : "+r"(ib) : "r"(ia));
      } else if (KIND == 2) {
#pragma unroll
        for (int q = 0; q < 4; q++) {
          float4 x;
          asm volatile("ld.shared.v4.f32 {%0,%1,%2,%3}, [%4];" : "=f"(x.x), "=f"(x.y), "=f"(x.z), "=f"(x.w) : "r"(p + 4096 * ((r + q) & 3) + 16384 * q));
          s0 += x.x;
        }
      } else if (KIND == 3) {
        asm volatile("max.f32 %0, %1, %2, %0;" : "+f"(m0) : "f"(fabsf(a[0].x)), "f"(fabsf(a[0].y)));
        asm volatile("max.f32 %0, %1, %2, %0;" : "+f"(m1) : "f"(fabsf(a[1].x)), "f"(fabsf(a[1].y)));
        asm volatile("max.f32 %0, %1, %2, %0;" : "+f"(m2) : "f"(fabsf(a[2].x)), "f"(fabsf(a[2].y)));
        asm volatile("max.f32 %0, %1, %2, %0;" : "+f"(m3) : "f"(fabsf(a[3].x)), "f"(fabsf(a[3].y)));
      } else if (KIND == 4) {
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(s0) : "f"(1.0001f), "f"(1e-7f));
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(s1) : "f"(1.0001f), "f"(1e-7f));
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(s2) : "f"(1.0001f), "f"(1e-7f));
        asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(s3) : "f"(1.0001f), "f"(1e-7f));
      } else if (KIND == 5) {
#pragma unroll
        for (int q = 0; q < 4; q++) s0 += __shfl_xor_sync(0xffffffffu, a[q].x, 1);
      }
    }
  }
  const long long t1 = clock64();
  float s = m0 + m1 + m2 + m3 + s0 + s1 + s2 + s3 + (float)(ia + ib);
#pragma unroll
  for (int i = 0; i < 8; i++) s += a[i].x + a[i].y;
  if (s == 123.456f) out[0] = s;
  if (threadIdx.x == 0 && blockIdx.x == 0) cycles[KIND] = t1 - t0;
}

template <int KIND>
static cudaError_t launch_issue_probe(float* out, int iters, long long* cycles, int sms, cudaStream_t st) {
  cudaError_t e = cudaFuncSetAttribute(k_issue_probe<KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, 160 * 1024);
  if (e != cudaSuccess) return e;
  k_issue_probe<KIND><<<sms, 256, 160 * 1024, st>>>(out, iters, cycles);   // 160 KB of shared memory: one CTA per SM
  return cudaGetLastError();
}

}  // namespace

extern "C" {

int bench_probe_issue(void* d_scratch, int iters, double* h_cycles_per_round, void* stream) {
  if (!d_scratch || iters < 1 || !h_cycles_per_round) return PROBE_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PROBE_ENODEV;
  cudaStream_t st = (cudaStream_t)stream;
  float* out = (float*)d_scratch;
  long long* cyc = (long long*)((unsigned char*)d_scratch + 64);
  cudaError_t e = launch_issue_probe<0>(out, iters, cyc, sms, st);
  if (e == cudaSuccess) e = launch_issue_probe<1>(out, iters, cyc, sms, st);
  if (e == cudaSuccess) e = launch_issue_probe<2>(out, iters, cyc, sms, st);
  if (e == cudaSuccess) e = launch_issue_probe<3>(out, iters, cyc, sms, st);
  if (e == cudaSuccess) e = launch_issue_probe<4>(out, iters, cyc, sms, st);
  if (e == cudaSuccess) e = launch_issue_probe<5>(out, iters, cyc, sms, st);
  long long h[6];
  if (e == cudaSuccess) e = cudaMemcpyAsync(h, cyc, sizeof(h), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return PROBE_ECUDA;
  // per scheduler: two resident warps share it, so one round of one warp takes half of the warp's own cycle count
  for (int k = 0; k < 6; k++) h_cycles_per_round[k] = (double)h[k] / ((double)iters * 16.0) / 2.0;
  return PROBE_OK;
}

int bench_probe_fma(void* d_out, int iters, double* flops, void* stream) {
  if (!d_out || iters < 1 || !flops) return PROBE_EINVAL;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return PROBE_ENODEV;
  const int blocks = sms * 8;   // 2048 threads per SM
  k_ffma_probe<<<blocks, 256, 0, (cudaStream_t)stream>>>((float*)d_out, iters);
  if (cudaGetLastError() != cudaSuccess) return PROBE_ECUDA;
  *flops = (double)blocks * 256.0 * (double)iters * 16.0 * 2.0;
  return PROBE_OK;
}

}  // extern "C"
