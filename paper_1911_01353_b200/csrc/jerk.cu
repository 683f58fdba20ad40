// jerk.cu — C-ABI (include/jerk.h) and sm_100a kernels of the Fourier-domain jerk-search hot path.
//
// Kernels:
//   k_bank     a-1  template bank: fp64 Gauss-Legendre response on the half-bin lattice -> taps -> FFT_L -> conj/L -> HBM
//   k_search   a-2..a-5  persistent fused kernel: bulk-copy (TMA) segment -> forward FFT (F stays in registers) ->
//              for each template-phase: F*G -> inverse FFT -> overlap discard -> |.|^2 -> plane store | threshold + local max
//   k_resolve  a-5  settles the few candidates that sit on a warp/segment seam (neighbour owned by another warp/segment)
#include <cuda_runtime.h>
#include <math.h>
#include <stdint.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <string>
#include <type_traits>
#include <vector>

#include "../../include/jerk.h"
#include "jerk_fft.cuh"
#include "jerk_fft64.cuh"

namespace jerk {

// ------------------------------------------------------------------------------------------------- plan
struct TemplateGeom {
  int32_t c;
  int32_t hw;
};

constexpr int kChunkTP = 256;          // template-phases per work item (G chunk = kChunkTP * L * 8 bytes, L2-resident; 128..1024 measured equal)
constexpr uint64_t kWorkHeader = 256;  // bytes: counters
constexpr uint64_t kBankAlign = 256;
// d_work = header | stash | seam records.  The stash gives every resident FFT group (k_search64: 64 threads) or CTA
// (k_search<L>) room for the phase-0 and phase-1 powers of one segment (rare path of the candidate test); launches never
// use more groups than slots, so the constant only has to cover sm_count * 4 groups (148 * 4 on B200, twice that here).
constexpr int kStashSlots = 1184;
constexpr uint64_t kStashSlotBytes = 2ull * 4096 * sizeof(float);
constexpr uint64_t kStashBytes = (uint64_t)kStashSlots * kStashSlotBytes;
constexpr uint64_t kSeamCapDefault = 1ull << 20;   // seam records jerk_plan_info's work_bytes leaves room for (a larger d_work holds more)

}  // namespace jerk

struct jerk_plan {
  int64_t nbins;
  double zmax, dz, wmax, dw;
  int numbetween, L;
  int nz, nw, T;
  int hw_max, c_max, step;
  int64_t seg_base, nseg;
  std::vector<jerk::TemplateGeom> geom;  // [T]
  uint64_t geom_bytes, bank_bytes, work_bytes, stash_bytes, order_bytes;   // d_work = header | order list | stash | seam records
  void* d_bank;
  int bank_ti_lo, bank_ti_cnt;   // templates [bank_ti_lo, bank_ti_lo + bank_ti_cnt) are in d_bank (jerk_templates: all T)
  int sm_count;
  // overlap classes of the candidate searches (add_class_jobs): class of a template = (hw - cls_lo) / cls_width,
  // cls_hw[k] = largest half-width of the grid's templates in class k (0: empty); ncls = 1: one segmentation for all
  int ncls, cls_lo, cls_width, cls_hw[16];
  std::string err;
};

namespace jerk {

static int fail(jerk_plan* p, int code, const std::string& msg) {
  if (p) p->err = msg;
  return code;
}

static int round_half_away(double v) { return (int)copysign(floor(fabs(v) + 0.5), v); }

// c(z,w): rounded midpoint of the excursion of g(u) = z u + w u^2/2 on [0,1]; hw = ceil(|z|/2+|w|/4)+8 (readings S3-S5)
static TemplateGeom template_geom(double z, double w) {
  double lo = 0.0, hi = 0.0;
  double e = z + w / 2.0;
  lo = fmin(lo, e);
  hi = fmax(hi, e);
  if (w != 0.0) {
    double us = -z / w;
    if (us > 0.0 && us < 1.0) {
      double v = -z * z / (2.0 * w);
      lo = fmin(lo, v);
      hi = fmax(hi, v);
    }
  }
  TemplateGeom g;
  g.c = round_half_away((lo + hi) / 2.0);
  g.hw = (int)ceil(fabs(z) / 2.0 + fabs(w) / 4.0) + 8;
  return g;
}

// ------------------------------------------------------------------------------------------------- bank kernel
// 8-node Gauss-Legendre on [-1,1]
__constant__ double c_gl_x[8] = {-0.96028985649753623168, -0.79666647741362673959, -0.52553240991632898582,
                                 -0.18343464249564980494, 0.18343464249564980494,  0.52553240991632898582,
                                 0.79666647741362673959,  0.96028985649753623168};
__constant__ double c_gl_w[8] = {0.10122853629037625915, 0.22238103445337447054, 0.31370664587788728734,
                                 0.36268378337836198297, 0.36268378337836198297, 0.31370664587788728734,
                                 0.22238103445337447054, 0.10122853629037625915};

// R_{z,w}(q) = int_0^1 exp(2 pi i (z u^2/2 + w u^3/6 - q u)) du  (BASELINE.json north_star item (1)).
// `panels` panels of at most ~one phase cycle each; phase in fp64, reduced mod 1, then fp32 sincospi.
__device__ float2 response_quadrature(double z, double w, double q, int panels) {
  const double h = 1.0 / (double)panels;
  const double a2 = 0.5 * z, a3 = w / 6.0;
  double sr = 0.0, si = 0.0;
  for (int pnl = 0; pnl < panels; pnl++) {
    double um = ((double)pnl + 0.5) * h;
    double pr = 0.0, pi = 0.0;
#pragma unroll
    for (int i = 0; i < 8; i++) {
      double u = fma(c_gl_x[i], 0.5 * h, um);
      double ph = u * (u * fma(a3, u, a2) - q);
      ph -= rint(ph);
      float s, c;
      sincospif(2.0f * (float)ph, &s, &c);
      pr = fma(c_gl_w[i], (double)c, pr);
      pi = fma(c_gl_w[i], (double)s, pi);
    }
    sr += pr;
    si += pi;
  }
  return make_float2((float)(sr * 0.5 * h), (float)(si * 0.5 * h));
}

__device__ __forceinline__ int quad_panels(double z, double w, int c, int hw) {
  // |d phase/du| <= max |g(u) - q| <= |excursion|/2 + hw + 1 cycles per unit u (q within hw of the excursion midpoint)
  double ex = fabs(z) + fabs(w) / 2.0;
  (void)c;
  return (int)ceil(0.5 * ex + (double)hw + 1.0) + 4;
}

struct BankParams {
  double zmax, dz, wmax, dw;
  int nz, nw;
  int nb;                    // numbetween: phases per template
  int ti_lo;                 // first template of the range being built (block b builds template ti_lo + b)
  const TemplateGeom* geom;  // device, [T]
  float2* G;                 // device, [ti - ti_lo][nb][L] in kernel element order
};

// element order of G inside one (template, phase): thread t of the search kernel reads float4 #(u*R1/2 + k2/2)*NT + t,
// which holds elements k = 256*k2 + b1_of(t,u) for k2 = 2h, 2h+1
template <int L>
__device__ __forceinline__ int bank_slot(int k) {
  using Gm = FftGeom<L>;
  int k2 = k >> 8, b1 = k & 255;
  int k1 = b1 >> 4, k0 = b1 & 15;
  int u = k1 / Gm::GS, t = k0 * Gm::GS + (k1 % Gm::GS);
  return (((u * (Gm::R1 / 2) + (k2 >> 1)) * Gm::NT + t) << 1) + (k2 & 1);
}

// seg_len 4096 is searched by k_search64 (64 threads x 64 points per FFT), which fuses the multiplication by G with the
// first radix-4 layer of the inverse transform (butterfly b of thread t combines elements k = 64 (16 a + b) + t, a = 0..3).
// Thread t reads float4 #((2 b + a / 2) * 64 + t): float2 slot of element (a, b, t); the values are stored in the mixed
// form of dft16_layerA_tw (bank_mixed_store below).
template <>
__device__ __forceinline__ int bank_slot<4096>(int k) {
  const int k1 = k >> 6, t = k & 63;
  const int a = k1 >> 4, b = k1 & 15;
  return ((((2 * b + (a >> 1)) << 6) + t) << 1) + (a & 1);
}
// g = c (1 + i t) with a real part kept away from zero (relative 1e-8: below fp32 rounding of the product; |t| <= 1e8
// keeps t * F far from overflow for any sensible spectrum)
__device__ __forceinline__ float2 bank_mixed(float2 g) {
  float c = g.x;
  const float lim = fmaxf(1e-8f * fabsf(g.y), 1e-30f);
  if (fabsf(c) < lim) c = copysignf(lim, c);
  return make_float2(c, g.y / c);
}

template <int L>
__global__ void __launch_bounds__(FftGeom<L>::NT) k_bank(BankParams bp) {
  using Gm = FftGeom<L>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* exA = reinterpret_cast<float2*>(smem_raw);
  float2* exB = exA + Gm::EX1;
  float2* tw2 = exB + Gm::EX2;
  float2* lat = tw2 + Tw2Table<L>::FLOATS2;  // 4*hw_max+1 lattice values
  __shared__ unsigned long long s_war;
  const int t = threadIdx.x;
  const int ti = bp.ti_lo + blockIdx.x;
  const int iz = ti % bp.nz, iw = ti / bp.nz;
  const double z = -bp.zmax + iz * bp.dz, w = -bp.wmax + iw * bp.dw;
  const TemplateGeom g = bp.geom[ti];
  const int panels = quad_panels(z, w, g.c, g.hw);
  for (int i = t; i < 4 * g.hw + 1; i += Gm::NT) lat[i] = response_quadrature(z, w, (double)(g.c - g.hw) + 0.5 * i, panels);
  fill_tw2<L>(tw2, t, Gm::NT);
  Tw3Regs<L> tw1;
  make_tw3<L>(tw1.w, t);
  WarBarrier war = war_init<Gm::NT>(&s_war, t);
  for (int p = 0; p < bp.nb; p++) {
    // taps h~_p[m'] = R(c + m' - p/2) at index (m' mod L): lattice index i = 2*(m'+hw) - p
    for (int k = t; k < L; k += Gm::NT) {
      int mp = k < L / 2 ? k : k - L;  // m' in [-L/2, L/2)
      float2 v = make_float2(0.f, 0.f);
      int lo = p ? -g.hw + 1 : -g.hw;
      if (mp >= lo && mp <= g.hw) v = lat[2 * (mp + g.hw) - p];
      exA[k] = v;
    }
    __syncthreads();
    float2 v[Gm::P];
#pragma unroll
    for (int u = 0; u < Gm::NB1; u++)
#pragma unroll
      for (int k2 = 0; k2 < Gm::R1; k2++) v[u * Gm::R1 + k2] = exA[256 * k2 + Gm::b1_of(t, u)];
    __syncthreads();
    fft_passes<L, -1>(v, tw1, tw2, exA, exB, war, t);
    float2* out = bp.G + ((size_t)blockIdx.x * bp.nb + p) * L;
    const float sc = 1.0f / (float)L;
#pragma unroll
    for (int u = 0; u < Gm::NB2; u++)
#pragma unroll
      for (int n2 = 0; n2 < 16; n2++) {
        int k = Gm::b3_of(t, u) + 16 * Gm::R1 * n2;
        float2 x = v[u * 16 + n2];
        const float2 gk = make_float2(x.x * sc, -x.y * sc);       // conj(FFT)/L
        if (L == 4096) exA[k] = gk;                                // staged in natural order, converted below
        else out[bank_slot<L>(k)] = gk;
      }
    __syncthreads();
    if (L == 4096) {
      // mixed form per radix-4 butterfly (a = 0..3 at k = 64 (16 a + b) + t64): plain, (c1, t1), (c2, t2), (c3 / c1, t3)
      for (int q = t; q < 1024; q += Gm::NT) {
        const int b = q >> 6, t64 = q & 63;
        const float2 g0 = exA[64 * b + t64], m1 = bank_mixed(exA[64 * (16 + b) + t64]), m2 = bank_mixed(exA[64 * (32 + b) + t64]),
                     m3 = bank_mixed(exA[64 * (48 + b) + t64]);
        float4* o4 = reinterpret_cast<float4*>(out) + (2 * b) * 64 + t64;
        o4[0] = make_float4(g0.x, g0.y, m1.x, m1.y);
        o4[64] = make_float4(m2.x, m2.y, m3.x / m1.x, m3.y);
      }
      __syncthreads();
    }
  }
}

__global__ void k_taps(double z, double w, int c, int hw, float2* out) {
  int panels = quad_panels(z, w, c, hw);
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < 4 * hw + 1; i += gridDim.x * blockDim.x)
    out[i] = response_quadrature(z, w, (double)(c - hw) + 0.5 * i, panels);
}

// ------------------------------------------------------------------------------------------------- search kernel
// One (r, iz, iw) box of the volume handled by a launch.  Candidate mode has one job (the whole grid); the harmonic
// stage submits up to eight plane-mode boxes (one per fraction k/8) in a single launch so that small boxes share the GPU.
struct SearchJob {
  int64_t seg_first, seg_count;  // segments [seg_first, seg_first+seg_count)
  int64_t r_lo, r_cnt;           // plane mode: bins [r_lo, r_lo+r_cnt) are written
  int iz_lo, iz_cnt, iw_lo, iw_cnt;
  int ntp;                       // template-phases selected = nb*iz_cnt*iw_cnt (box) or nb*(templates of the class)
  int chunk_tp;                  // template-phases per work item (even)
  // Overlap of this job's segments: outputs n in [hw, hw + step) of a segment are kept, step = L - 2 hw, segment s starts
  // at bin seg_base + s*step.  A box job uses the plan's hw_max; an overlap class (candidate modes) the largest
  // half-width of ITS templates, so that narrow templates are not charged the overlap of the widest one.
  int hw, step;
  int64_t seg_base;
  const int* order;              // overlap class: its template indices ti (the job's templates in walk order); nullptr: row-major box
  float* plane;                  // plane mode: P[iw_rel][iz_rel][j - 2*r_lo]
  float* bmax;                   // plane mode, optional: block maxima of every (row, segment) unit, [row][seg - seg_first][kBmaxBlocks][2] (harmonic stage)
  long long item_end;            // work items of jobs 0..this one (exclusive prefix sum of nchunks*seg_count)
};
constexpr int kMaxJobs = 16;
// Block maxima of a plane-mode unit (the bounds of the harmonic stage): outputs n of a unit fall into six blocks by
// n >> 9 -> {0,1 | 2 | 3 | 4 | 5 | 6,7} (the first and last merged: the valid window [hw_max, hw_max + step) cuts them
// short) and two halves by bit 5 of n (which warp of the FFT group owns the output).
constexpr int kBmaxBlocks = 6;
__host__ __device__ __forceinline__ int bmax_block(int n) {
  const int g = (n >> 9) - 1;
  return g < 0 ? 0 : (g > kBmaxBlocks - 1 ? kBmaxBlocks - 1 : g);
}

// Harmonic stage fused into the top-harmonic search (row a-6): sub-plane of fraction e/8, e = 1..7, as written by the
// plane-mode kernel: P_e[iw_rel][iz_rel][j - j0], row length nj.
struct HarmGather {
  const float* base[7];
  long long j0[7], nj[7];
  int iz_lo[7], iz_cnt[7], iw_lo[7];
  int cz, cw;                // centre indices (nz-1)/2, (nw-1)/2
  const float* bmax[7];      // arg-max mode: block maxima of sub-plane e (SearchJob::bmax of the launch that stored it)
  int seg_first[7], seg_count[7];
  float thr[4];              // arg-max mode: only sums above thr[log2 h] can be reported
  jerk_cand* warpbest;       // arg-max mode: [4][gridDim.x * warps per CTA] best record of every warp, h = 1,2,4,8
  float* out;                // store mode: S_h of the box, out[iw - out_iw_lo][iz - out_iz_lo][j - 2 r_lo]
  int out_stage;             // store mode: log2 h
  int out_iz_lo, out_iz_cnt, out_iw_lo;
};

constexpr int kMaxBatch = 32;   // spectra per launch of the batched candidate search

struct SearchParams {
  const float2* spec[kMaxBatch];  // X_b[nbins], b < nspec (one spectrum everywhere but in jerk_search_candidates_batch)
  int nspec;
  int nb;              // numbetween: 2 (half-bin phases 0 and 1) or 1 (phase 0 only)
  int64_t nbins;
  const float2* G;
  const TemplateGeom* geom;
  int nz, nw_grid;     // grid size (nw_grid = nw of the plan)
  int hw_max, step;
  int64_t seg_base;
  int njobs;
  long long nitems;
  SearchJob jobs[kMaxJobs];
  // candidate mode
  float threshold;
  jerk_cand* cands;
  int64_t max_cands;
  unsigned long long* count;
  // scratch
  unsigned long long* work;  // [0] item counter, [1] seam count, [2] seam overflow, [3] provisional
  jerk_cand* seams;
  unsigned long long seam_cap;   // seam records that fit in d_work
  float* stash;              // one slot of 2 L floats per resident FFT group / CTA: powers of the current template, written only on the rare path
  double* rowstats;          // MODE_CAND_STATS: [T][2] running sum of P and of P^2 over the valid points of every (z,w) row
  HarmGather hg;             // MODE_HARM / MODE_HARM_STORE: the seven sub-planes the top-harmonic pass gathers from
};

// spectrum b of a batch owns cands[b*max_cands ..) and count[b]; its seam records carry b in flags bits 8..31
__device__ __forceinline__ void emit_cand(const SearchParams& sp, int b, int j, int iz, int iw, float pw) {
  unsigned long long slot = atomicAdd(sp.count + b, 1ULL);
  if ((int64_t)slot < sp.max_cands) {
    jerk_cand c;
    c.j = j;
    c.iz = (int16_t)iz;
    c.iw = (int16_t)iw;
    c.power = pw;
    c.flags = 0;
    sp.cands[(size_t)b * sp.max_cands + slot] = c;
  }
}
__device__ __forceinline__ void emit_seam(const SearchParams& sp, int b, int j, int iz, int iw, float pw, uint32_t flags) {
  unsigned long long slot = atomicAdd(sp.work + 1, 1ULL);
  if (slot < sp.seam_cap) {
    jerk_cand c;
    c.j = j;
    c.iz = (int16_t)iz;
    c.iw = (int16_t)iw;
    c.power = pw;
    c.flags = flags | ((uint32_t)b << 8);
    sp.seams[slot] = c;
  } else {
    sp.work[2] = 1ULL;
  }
}

enum { SEAM_LEFT = 1u, SEAM_RIGHT = 2u, SEAM_WITNESS = 4u };

// One work item = (job, chunk of template-phases, spectrum of the batch, segment), chunk-major so that every resident
// FFT group streams the same chunk of the bank through L2 at the same time, for all segments of all spectra.
struct WorkItem {
  int q, chunk, b;
  int64_t seg;
};
__device__ __forceinline__ WorkItem decode_item(const SearchParams& sp, long long item) {
  WorkItem w;
  w.q = 0;
  while (w.q + 1 < sp.njobs && item >= sp.jobs[w.q].item_end) w.q++;
  const SearchJob& jb = sp.jobs[w.q];
  const long long jitem = item - (w.q ? sp.jobs[w.q - 1].item_end : 0LL);
  const long long per_chunk = jb.seg_count * sp.nspec;
  w.chunk = (int)(jitem / per_chunk);
  const long long rem = jitem % per_chunk;
  w.b = (int)(rem / jb.seg_count);
  w.seg = jb.seg_first + rem % jb.seg_count;
  return w;
}

// Candidate test of one valid point in the rare path (P > thr, P > P[j-1], P >= P[j+1]).  `left` /
// `right` are the neighbours' powers when this warp holds them; a neighbour across a warp or segment seam is unknown
// (seamL / seamR) and the point becomes a seam record, flagged SEAM_WITNESS when it already lost on a known side (it
// is then only evidence for its neighbour).  At the spectrum ends the missing neighbour is -inf (known).
__device__ __forceinline__ void test_point(const SearchParams& sp, int b, int j, int iz, int iw, float p, float left, float right,
                                           bool seamL, bool seamR) {
  if (!(p > sp.threshold)) return;
  const bool pass = (seamL || p > left) && (seamR || p >= right);
  if (seamL || seamR) emit_seam(sp, b, j, iz, iw, p, (seamL ? SEAM_LEFT : 0u) | (seamR ? SEAM_RIGHT : 0u) | (pass ? 0u : SEAM_WITNESS));
  else if (pass) emit_cand(sp, b, j, iz, iw, p);
}

// 2: candidate mode + per-row power statistics; 3 / 4: top-harmonic pass of the harmonic stage (arg-max / S_h store), seg_len 4096
enum { MODE_PLANE = 0, MODE_CAND = 1, MODE_CAND_STATS = 2, MODE_HARM = 3, MODE_HARM_STORE = 4 };

// TMEM columns per CTA: two thread-private arrays (F and T1) of 2P floats per thread, NW/4 warp groups side by side
template <int L>
struct TmemCols {
  static constexpr int value = 2 * ((FftGeom<L>::NW + 3) / 4) * 2 * FftGeom<L>::P;
};

template <int L, int MODE>
__global__ void __launch_bounds__(FftGeom<L>::NT, 1)
k_search(const __grid_constant__ SearchParams sp) {
  using Gm = FftGeom<L>;
  constexpr int NT = Gm::NT, P = Gm::P, R1 = Gm::R1;
  constexpr int TCOLS = TmemCols<L>::value;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* exA = reinterpret_cast<float2*>(smem_raw);
  float2* exB = exA + Gm::EX1;
  float2* tw2 = exB + Gm::EX2;
  unsigned long long* mbar = reinterpret_cast<unsigned long long*>(tw2 + Tw2Table<L>::FLOATS2);  // [0] segment copy, [1] exB WAR
  __shared__ long long s_item;
  __shared__ uint32_t s_tmem;
  const int t = threadIdx.x, lane = t & 31, warp = t >> 5;

  // ---- tensor memory: per-thread homes for F (forward-transformed segment) and the T1 twiddles
  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TCOLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  fill_tw2<L>(tw2, t, NT);
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(smem_u32(mbar)));
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  WarBarrier war = war_init<NT>(mbar + 1, t);   // contains the __syncthreads that publishes s_tmem, tw2 and mbar[0]
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tbase = s_tmem + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)(warp >> 2) * (2 * P);
  TmemArray<L> tmF, tmT;
  tmF.addr = tbase;
  tmT.addr = tbase + TCOLS / 2;
  {
    float2 w[P];
    make_tw3<L>(w, t);
#pragma unroll
    for (int h = 0; h < P / 16; h++) {
      float2 q[16];
#pragma unroll
      for (int i = 0; i < 16; i++) q[i] = w[16 * h + i];
      tmT.store16(h, q);
    }
  }
  uint32_t mphase = 0;
  const long long nitems = sp.nitems;
  float* gstash = sp.stash + (size_t)blockIdx.x * (2 * L);   // [2][P][NT] powers of the current template (rare path)

  for (;;) {
    if (t == 0) s_item = (long long)atomicAdd(sp.work, 1ULL);
    __syncthreads();
    const long long item = s_item;
    if (item >= nitems) break;
    const WorkItem wi = decode_item(sp, item);
    const SearchJob& jb = sp.jobs[wi.q];
    const float2* spec = sp.spec[wi.b];
    const int iz_cnt = jb.iz_cnt, iz_lo = jb.iz_lo, iw_lo = jb.iw_lo;
    const int hw_j = jb.hw, step_j = jb.step;                    // this job's overlap (SearchJob)
    const int64_t s0 = jb.seg_base + wi.seg * (int64_t)step_j;   // first bin of the segment (even)

    // ---- a-2: stage the segment in shared memory (exA): TMA bulk copy when fully inside the spectrum, guarded loads at the edges
    const bool interior = (s0 >= 0) && (s0 + L <= sp.nbins);
    if (interior) {
      if (t == 0) {
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");  // order earlier generic accesses to exA before the async write
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(mbar)), "r"((uint32_t)(L * 8)) : "memory");
        asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(exA)),
                     "l"(spec + s0), "r"((uint32_t)(L * 8)), "r"(smem_u32(mbar))
                     : "memory");
      }
      uint32_t done = 0;
      while (!done) {
        asm volatile(
            "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
            : "=r"(done)
            : "r"(smem_u32(mbar)), "r"(mphase)
            : "memory");
      }
      mphase ^= 1u;
    } else {
      for (int k = t; k < L; k += NT) {
        int64_t b = s0 + k;
        exA[k] = (b >= 0 && b < sp.nbins) ? spec[b] : make_float2(0.f, 0.f);
      }
      __syncthreads();
    }
    // ---- forward FFT; F goes to TMEM in the pass-1 layout F[256*k2 + b1_of(t,u)] at array index u*R1 + k2
    {
      float2 v[P];
#pragma unroll
      for (int u = 0; u < Gm::NB1; u++)
#pragma unroll
        for (int k2 = 0; k2 < R1; k2++) v[u * R1 + k2] = exA[256 * k2 + Gm::b1_of(t, u)];
      __syncthreads();                                   // exA is about to be reused as exchange buffer 1
      fft_passes<L, -1>(v, tmT, tw2, exA, exB, war, t);
      __syncthreads();                                   // all pass-2 reads of exA done (they precede the barrier inside)
#pragma unroll
      for (int u = 0; u < Gm::NB2; u++)
#pragma unroll
        for (int n2 = 0; n2 < 16; n2++) exA[Gm::b3_of(t, u) + 16 * R1 * n2] = v[u * 16 + n2];
      __syncthreads();
#pragma unroll
      for (int h = 0; h < P / 16; h++) {
        float2 q[16];
#pragma unroll
        for (int i = 0; i < 16; i++) {
          const int e = 16 * h + i, u = e / R1, k2 = e % R1;
          q[i] = exA[256 * k2 + Gm::b1_of(t, u)];
        }
        tmF.store16(h, q);
      }
      __syncthreads();
    }

    // ---- loop over the template-phases of this chunk (numbetween = 1: one phase per template)
    const int nb = sp.nb;
    const int tp_lo = wi.chunk * jb.chunk_tp;
    const int tp_hi = min(jb.ntp, tp_lo + jb.chunk_tp);
    float p0v[P];  // phase-0 powers (plane mode keeps them to store float2 pairs)
    int any0 = 0;  // candidate mode: phase-0 powers of this warp exceeded the threshold and were stashed
    int izr = (tp_lo / nb) % iz_cnt, iwr = (tp_lo / nb) / iz_cnt;
    const int* order = jb.order;
    for (int tp = tp_lo; tp < tp_hi; tp++) {
      const int ph = nb == 2 ? (tp & 1) : 0;
      if (ph == 0 && tp != tp_lo && ++izr == iz_cnt) {
        izr = 0;
        ++iwr;
      }
      const int ti = order ? __ldg(order + tp / nb) : (iw_lo + iwr) * sp.nz + iz_lo + izr;
      const int iz = ti % sp.nz, iw = ti / sp.nz;
      const int c = sp.geom[ti].c;
      // ---- a-3: Y = F .* G (G straight from L2/HBM, F from TMEM), inverse FFT
      float2 v[P];
      __syncwarp();   // tcgen05.ld is .sync.aligned: the warp must be converged (the store / candidate paths below diverge)
      {
        const float4* g4 = reinterpret_cast<const float4*>(sp.G + ((size_t)ti * nb + ph) * L) + t;
        float4 g[P / 2];
#pragma unroll
        for (int e = 0; e < P / 2; e++) g[e] = __ldg(g4 + e * NT);
#pragma unroll
        for (int h = 0; h < P / 16; h++) {
          float2 fq[16];
          tmF.load16(h, fq);
#pragma unroll
          for (int i = 0; i < 8; i++) {
            v[16 * h + 2 * i] = cmul(fq[2 * i], make_float2(g[8 * h + i].x, g[8 * h + i].y));
            v[16 * h + 2 * i + 1] = cmul(fq[2 * i + 1], make_float2(g[8 * h + i].z, g[8 * h + i].w));
          }
        }
      }
      fft_passes<L, 1>(v, tmT, tw2, exA, exB, war, t);
      // ---- a-4: overlap discard + power.  n = b3 + 16*R1*n2 ; b = s0 + n - c ; j = nb*b + ph.
      // valid outputs: n in [n_lo, n_hi) = window [hw_max, hw_max+step) clipped to the bins this call covers
      int n_lo, n_hi;
      {
        long long blo = MODE == MODE_PLANE ? jb.r_lo : 0, bhi = MODE == MODE_PLANE ? jb.r_lo + jb.r_cnt : sp.nbins;
        long long lo = blo + c - s0, hi = bhi + c - s0;
        n_lo = (int)max((long long)hw_j, min(lo, (long long)L));
        n_hi = (int)min((long long)(hw_j + step_j), max(hi, 0LL));
      }
      float pw[P];
#pragma unroll
      for (int i = 0; i < P; i++) pw[i] = fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
      if (MODE == MODE_PLANE) {
        float* row = jb.plane + ((size_t)iwr * iz_cnt + izr) * (size_t)(nb * jb.r_cnt);
        const long long boff = s0 - c - jb.r_lo;
        if (nb == 1) {
#pragma unroll
          for (int u = 0; u < Gm::NB2; u++)
#pragma unroll
            for (int n2 = 0; n2 < 16; n2++) {
              const int n = Gm::b3_of(t, u) + 16 * R1 * n2;
              if (n >= n_lo && n < n_hi) row[boff + n] = pw[u * 16 + n2];
            }
        } else if (ph == 0) {
#pragma unroll
          for (int i = 0; i < P; i++) p0v[i] = pw[i];
        } else {
#pragma unroll
          for (int u = 0; u < Gm::NB2; u++)
#pragma unroll
            for (int n2 = 0; n2 < 16; n2++) {
              const int n = Gm::b3_of(t, u) + 16 * R1 * n2;
              if (n >= n_lo && n < n_hi)
                *reinterpret_cast<float2*>(row + 2 * (boff + n)) = make_float2(p0v[u * 16 + n2], pw[u * 16 + n2]);
            }
        }
      } else {
        if (MODE == MODE_CAND_STATS) {
          // sum of P and P^2 over the valid points of this unit, one fp64 atomic pair per warp
          float a1[4] = {0.f, 0.f, 0.f, 0.f}, a2[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
          for (int i = 0; i < P; i++) {
            const int n = Gm::b3_of(t, i >> 4) + 16 * R1 * (i & 15);
            const float p = (n >= n_lo && n < n_hi) ? pw[i] : 0.f;
            a1[i & 3] += p;
            a2[i & 3] = fmaf(p, p, a2[i & 3]);
          }
          float s1 = (a1[0] + a1[1]) + (a1[2] + a1[3]), s2 = (a2[0] + a2[1]) + (a2[2] + a2[3]);
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
          }
          if (lane == 0) {
            atomicAdd(sp.rowstats + 2 * (size_t)ti, (double)s1);
            atomicAdd(sp.rowstats + 2 * (size_t)ti + 1, (double)s2);
          }
        }
        // ---- a-5: threshold + local max.  Hot path: one max-reduction and a vote; everything else only when some
        // power of this warp (valid or not) exceeds the threshold.
        float mx = pw[0];
#pragma unroll
        for (int i = 1; i < P; i++) mx = fmaxf(mx, pw[i]);
        const int anyhit = __any_sync(0xffffffffu, mx > sp.threshold);
        float* st0 = gstash;            // [P][NT]: element i of thread t at i*NT + t (written and read by the same thread)
        float* st1 = gstash + L;
        const float NEG = -INFINITY;
        if (nb == 1) {
          if (anyhit) {
#pragma unroll
            for (int i = 0; i < P; i++) st0[i * NT + t] = pw[i];
            __syncwarp();
#pragma unroll 1
            for (int i = 0; i < P; i++) {
              const int n = Gm::b3_of(t, i >> 4) + 16 * R1 * (i & 15);
              const bool valid = (n >= n_lo) && (n < n_hi);
              const float p = valid ? st0[i * NT + t] : NEG;
              const float l = __shfl_up_sync(0xffffffffu, p, 1);      // P[b-1]
              const float r = __shfl_down_sync(0xffffffffu, p, 1);    // P[b+1]
              if (!valid) continue;
              const long long b = s0 + n - c;
              const bool seamL = (lane == 0 || n == hw_j) && (b > 0);
              const bool seamR = (lane == 31 || n == hw_j + step_j - 1) && (b < sp.nbins - 1);
              test_point(sp, wi.b, (int)b, iz, iw, p, b > 0 ? l : NEG, b < sp.nbins - 1 ? r : NEG, seamL, seamR);
            }
            __syncwarp();
          }
        } else if (ph == 0) {
          any0 = anyhit;
          if (anyhit) {
#pragma unroll
            for (int i = 0; i < P; i++) st0[i * NT + t] = pw[i];
          }
        } else if (anyhit | any0) {
#pragma unroll
          for (int i = 0; i < P; i++) st1[i * NT + t] = pw[i];
          __syncwarp();
#pragma unroll 1
          for (int i = 0; i < P; i++) {
            const int n = Gm::b3_of(t, i >> 4) + 16 * R1 * (i & 15);
            const bool valid = (n >= n_lo) && (n < n_hi);
            const float p1 = valid ? st1[i * NT + t] : NEG;
            const float p0 = (valid && any0) ? st0[i * NT + t] : NEG;
            const float l1 = __shfl_up_sync(0xffffffffu, p1, 1);    // P1[n-1]
            const float r0 = __shfl_down_sync(0xffffffffu, p0, 1);  // P0[n+1]
            if (!valid) continue;
            const long long b = s0 + n - c;
            // phase-0 point j = 2b: left neighbour (b-1, phase 1), right neighbour (b, phase 1)
            test_point(sp, wi.b, (int)(2 * b), iz, iw, p0, b > 0 ? l1 : NEG, p1, (lane == 0 || n == hw_j) && (b > 0), false);
            // phase-1 point j = 2b+1: left neighbour (b, phase 0), right neighbour (b+1, phase 0)
            test_point(sp, wi.b, (int)(2 * b + 1), iz, iw, p1, p0, b < sp.nbins - 1 ? r0 : NEG, false,
                       (lane == 31 || n == hw_j + step_j - 1) && (b < sp.nbins - 1));
          }
          __syncwarp();
        }
      }
    }
    __syncthreads();
  }
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "n"(TCOLS));
}

// ------------------------------------------------------------------------------------------------- search kernel, seg_len 4096
// k_search64: the same fused path (rows a-2..a-5) on the two-pass 64 x 64 FFT of jerk_fft64.cuh.  A CTA holds two
// independent FFT groups of 64 threads (two warps each); every group takes its own work items from the global counter,
// has its own exchange buffer, named barrier and mbarriers, and shares only the CTA's tensor-memory allocation:
// F (the transformed segment, 64 complex per thread) in columns [0,128) and the pass-2 twiddles in [128,256) of the
// thread's own TMEM lane.  Two CTAs per SM (TMEM 2 x 256 columns, up to 255 registers per thread).
//
// G never passes through registers before it is used: while pass 2 of the current template-phase runs, one thread
// bulk-copies (TMA) the 32 KB of the NEXT template-phase into the group's exchange buffer, which is idle from the
// pass-2 loads of one transform to the pass-1 stores of the next; the multiply F .* G then reads G with 128-bit
// shared-memory loads (30 cycles instead of an exposed L2 round trip with only two warps per scheduler to hide it).
// Hazards on the buffer, per group: [1] G landed (TMA tx) -> G reads; [2] G reads done (count 64) -> pass-1 stores;
// named barrier: stores -> loads; [3] loads done (count 64) -> next TMA.
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
// one probe of the barrier (the answer takes ~90 cycles: start it early, use it late): 1 iff phase `parity` is complete
__device__ __forceinline__ uint32_t mbar_probe(uint32_t bar, uint32_t parity) {
  uint32_t done;
  asm volatile(
      "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
      : "=r"(done)
      : "r"(bar), "r"(parity)
      : "memory");
  return done;
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  uint32_t done = 0;
  while (!done) {
    asm volatile(
        "{\n\t.reg .pred p;\n\tmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\tselp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(done)
        : "r"(bar), "r"(parity)
        : "memory");
  }
}
__device__ __forceinline__ void bulk_copy_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // earlier generic accesses to dst before the async write
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst), "l"(src),
               "r"(bytes), "r"(bar)
               : "memory");
}
// ---- harmonic stage, fused into the top-harmonic pass (row a-6; BASELINE.json configs[4]; reading S13)
//   S_h(j,iz',iw') = sum_{k=1..h} P[rnd(j k/h); rnd(iz' k/h), rnd(iw' k/h)],  signed grid indices, rnd = round half away from zero.
// Every fraction k/h of h in {1,2,4,8} is e/8:  S1 = P8;  S2 = S1 + P4;  S4 = S2 + P2 + P6;  S8 = S4 + P1 + P3 + P5 + P7,
// Pe = the sub-plane of fraction e/8.  P8 is the search itself: the top-harmonic pass holds it in registers (phase 1) and
// tensor memory (phase 0) and gathers P1..P7 from the sub-planes that an earlier plane-mode launch left in scratch, so
// the largest sub-plane never exists in memory and no separate summing pass reads it back.
struct HarmRecord {   // running arg-max of one warp and one stage
  float s;            // best sum so far (initially the stage threshold: only sums above it count)
  int j, ti;          // its position (j = -1: none yet)
};

__device__ __forceinline__ int rnd_eighths(int a, int e) {          // round-half-away-from-zero of a*e/8
  const int m = (abs(a) * e + 4) >> 3;
  return a < 0 ? -m : m;
}

// a beats b as the arg-max: larger sum, ties -> smallest (iw, iz, j) in row-major order (ti = iw*nz + iz)
__device__ __forceinline__ bool harm_better_ti(float sa, int ja, int tia, float sb, int jb, int tib) {
  if (sa != sb) return sa > sb;
  if (tia != tib) return tia < tib;
  return ja < jb;
}

// the four stage sums of one point from its own power p8 and the seven gathered sub-harmonic powers g[e-1]
__device__ __forceinline__ void harm_stage_sums(float p8, const float (&g)[7], float (&sv)[4]) {
  sv[0] = p8;
  sv[1] = sv[0] + g[3];
  sv[2] = sv[1] + g[1] + g[5];
  sv[3] = sv[2] + g[0] + g[2] + g[4] + g[6];
}

// Seven read-only loads (one per fraction e = 1..7) at byte offsets KOFF * e from the seven pointers: one register of
// one phase.  Unpredicated: a register outside the unit's valid window (the box may be much shorter than a segment) reads
// up to (4096 + c_max) e / 4 floats before or after its sub-plane row -- still inside the scratch buffer, which carries a
// guard band at both ends (kHarmGuard) -- and its sums are discarded.  volatile: the loads of a batch keep their place before the fence.
template <int KOFF>
__device__ __forceinline__ void ld_gather7(float (&g)[7], const float* const (&q)[7]) {
  asm volatile(
      "ld.global.nc.f32 %0, [%7+%14];\n\tld.global.nc.f32 %1, [%8+%15];\n\tld.global.nc.f32 %2, [%9+%16];\n\t"
      "ld.global.nc.f32 %3, [%10+%17];\n\tld.global.nc.f32 %4, [%11+%18];\n\tld.global.nc.f32 %5, [%12+%19];\n\t"
      "ld.global.nc.f32 %6, [%13+%20];"
      : "=f"(g[0]), "=f"(g[1]), "=f"(g[2]), "=f"(g[3]), "=f"(g[4]), "=f"(g[5]), "=f"(g[6])
      : "l"(q[0]), "l"(q[1]), "l"(q[2]), "l"(q[3]), "l"(q[4]), "l"(q[5]), "l"(q[6]), "n"(KOFF * 1), "n"(KOFF * 2), "n"(KOFF * 3),
        "n"(KOFF * 4), "n"(KOFF * 5), "n"(KOFF * 6), "n"(KOFF * 7));
}

// row pointers of the seven sub-planes for template ti, positioned at the source of point j = jt + 128 n1 + ph for
// n1 = n1_first (see harm_unit)
__device__ __forceinline__ void harm_pointers(const SearchParams& sp, int ti, long long jt, int n1_first, const float* (&q0)[7],
                                              const float* (&q1)[7]) {
  const HarmGather& hg = sp.hg;
  const int az = ti % sp.nz - hg.cz, aw = ti / sp.nz - hg.cw;
#pragma unroll
  for (int e = 1; e <= 7; e++) {
    const int ize = rnd_eighths(az, e) + hg.cz, iwe = rnd_eighths(aw, e) + hg.cw;
    const float* row = hg.base[e - 1] + ((long long)(iwe - hg.iw_lo[e - 1]) * hg.iz_cnt[e - 1] + (ize - hg.iz_lo[e - 1])) * hg.nj[e - 1] -
                       hg.j0[e - 1] + 16 * n1_first * e;
    q0[e - 1] = row + ((jt * e + 4) >> 3);
    q1[e - 1] = row + (((jt + 1) * e + 4) >> 3);
  }
}

// One batch of the gathers of harm_unit: the four registers 16 a + k (a = 0..3) of one k, i.e. n1 = 4 k + a: 256 contiguous
// bins, both phases: 56 loads, all issued before the first sum.  q0 / q1 point at n1 = 4 k.
template <bool STORE>
__device__ __forceinline__ void harm_batch(const HarmGather& hg, const float* const (&q0)[7], const float* const (&q1)[7], uint32_t tmP,
                                           const float* p1s, int k, int t, int n_lo, int n_hi, bool inner_valid, float2* dst,
                                           float (&mx)[4]) {
  float g0[4][7], g1[4][7];
  bool ok[4];
#pragma unroll
  for (int a = 0; a < 4; a++) {
    const int n1 = 4 * k + a;
    const int n = t + 64 * n1;
    ok[a] = (inner_valid && n1 >= 8 && n1 < 56) || (n >= n_lo && n < n_hi);
  }
  ld_gather7<64 * 0>(g0[0], q0); ld_gather7<64 * 0>(g1[0], q1);
  ld_gather7<64 * 1>(g0[1], q0); ld_gather7<64 * 1>(g1[1], q1);
  ld_gather7<64 * 2>(g0[2], q0); ld_gather7<64 * 2>(g1[2], q1);
  ld_gather7<64 * 3>(g0[3], q0); ld_gather7<64 * 3>(g1[3], q1);
  // Scheduling fence: the sums sit behind a branch the compiler cannot resolve (cz >= 0 always), i.e. in another basic
  // block, so that every load of the batch is issued before the first sum waits for one (ptxas otherwise pulls each
  // sum up next to its own loads, which serialises the round trips).
  if (hg.cz < 0) return;
  float p0c[4];
  tmem_ld1x4(tmP + k, p0c);   // the powers of this batch: phase 0 from tensor memory (columns 16 a + k), phase 1 from shared memory
#pragma unroll
  for (int a = 0; a < 4; a++) {
    float sa[4], sb[4];
    harm_stage_sums(p0c[a], g0[a], sa);
    harm_stage_sums(p1s[(16 * a + k) * 64 + t], g1[a], sb);
    if (STORE) {
      if (ok[a]) dst[64 * (4 * k + a)] = make_float2(sa[hg.out_stage], sb[hg.out_stage]);
    } else if (ok[a]) {
#pragma unroll
      for (int q = 0; q < 4; q++) mx[q] = fmaxf(mx[q], fmaxf(sa[q], sb[q]));
    }
  }
}

// Which pairs of batches (top bins n in [256 kp, 256 kp + 512), kp = KLO, KLO + 2, ...) can hold a sum that reaches the
// warp's record?  Upper bound of S_h over a pair: the thread's own largest power there (pms) plus, per fraction e, the
// largest stored power its sources can come from.  The <= 449 + 1 source bins of a fraction lie in at most two blocks of
// the producer's block maxima (each block is at least 512 outputs long, SearchJob::bmax), those of the first and of the
// last source bin, times two halves: four values per fraction, fetched by 28 lanes in parallel, for all pairs at once
// (one round trip per template instead of one per pair); the four are folded with two shuffles, and lane i then
// evaluates pair i (its seven bounds come through shared memory, the warp's own maxima from a warp reduction), so the
// whole test has no loop over the pairs.  Exact pruning: a pair is skipped only if every stage's bound stays below the
// record (initially the stage threshold), so no arg-max or tie can be lost.  Bit i of the result: pair i.
template <int KLO, int KHI>
__device__ __forceinline__ uint32_t harm_bounds_mask(const SearchParams& sp, int s0, int c, int ti, int n_lo, int n_hi, int lane, int t,
                                                     const float* pms, const float (&pw)[64], float* scr, const HarmRecord* rec) {
  constexpr int NP = (KHI - KLO) / 2;
  const HarmGather& hg = sp.hg;
  // scratch: be[pair][8] in this warp's own slots of the group's buffer (scr[r * 64 + t] belongs to thread t): pairs
  // 0..3 in its 32 floats of row 0, pairs 4..7 in those of row 1
  float* ws = scr + (t & 32);
  const auto ws_at = [&](int i) { return ws + 64 * (i >> 2) + 8 * (i & 3); };
  // lane = 4 (e - 1) + slot, 28 lanes: the block maximum at the first (slot < 2) / last source bin of every pair, two halves
  float val[NP];
  {
    const int e = min((lane >> 2) + 1, 7), slot = lane & 3;
    const int az = ti % sp.nz - hg.cz, aw = ti / sp.nz - hg.cw;
    const int ize = rnd_eighths(az, e) + hg.cz, iwe = rnd_eighths(aw, e) + hg.cw;
    const int cs = sp.geom[iwe * sp.nz + ize].c;
    const float* bm = hg.bmax[e - 1] + (size_t)((iwe - hg.iw_lo[e - 1]) * hg.iz_cnt[e - 1] + (ize - hg.iz_lo[e - 1])) * hg.seg_count[e - 1] * (kBmaxBlocks * 2) +
                      (slot & 1);
    const int segf = hg.seg_first[e - 1], seg_last = hg.seg_count[e - 1] - 1;
    const int uoff = cs - (int)sp.seg_base - sp.hw_max;
    const int step = sp.step, hwm = sp.hw_max;
    const float inv_step = 1.0f / (float)step;
    const bool last = (slot & 2) != 0;
    const int ph = last ? 1 : 0;
    const int boff = s0 - c;
    // Branch-free, 32-bit: point j = 2 b + ph (b = s0 - c + n < 2^30) reads source half-bin (j e + 4) >> 3, i.e. source
    // bin x = (j e + 4) >> 4 = (b >> 3) e + (((2 (b & 7) + ph) e + 4) >> 4).  Invalid pairs load a clamped (legal) entry
    // and are zeroed afterwards.
#pragma unroll
    for (int i = 0; i < NP; i++) {
      const int kp = KLO + 2 * i;
      const int n_first = max(256 * kp, n_lo), n_last = min(256 * kp + 511, n_hi - 1);
      const int bb = boff + (last ? n_last : n_first);
      const int x = (bb >> 3) * e + (((2 * (bb & 7) + ph) * e + 4) >> 4);
      const int u = x + uoff;                                  // the unit that owns bin x of this template: segment u / step, output r + hw_max
      int seg = (int)((float)u * inv_step);                    // u / step: float estimate, corrected by at most one
      int r = u - seg * step;
      seg += (r >= step) - (r < 0);
      r += (r < 0 ? step : 0) - (r >= step ? step : 0);
      const int sidx = min(max(seg - segf, 0), seg_last);
      const float v = __ldg(bm + (sidx * kBmaxBlocks + bmax_block(r + hwm)) * 2);
      val[i] = (n_last >= n_first && lane < 28) ? v : 0.f;
    }
  }
  // the bound of fraction e for pair i = the largest of its four values (lanes 4 (e - 1) .. 4 (e - 1) + 3), left at ws_at(i)[e - 1]
#pragma unroll
  for (int i = 0; i < NP; i++) val[i] = fmaxf(val[i], __shfl_xor_sync(0xffffffffu, val[i], 1));
#pragma unroll
  for (int i = 0; i < NP; i++) val[i] = fmaxf(val[i], __shfl_xor_sync(0xffffffffu, val[i], 2));
  if ((lane & 3) == 0 && lane < 28) {
#pragma unroll
    for (int i = 0; i < NP; i++) ws_at(i)[lane >> 2] = val[i];
  }
  // the warp's own largest power of every pair (powers are >= 0: their bit patterns order like unsigned integers); lane i keeps pair i's
  float own = 0.f;
  {
    const float4 pa = reinterpret_cast<const float4*>(pms)[t], pb = reinterpret_cast<const float4*>(pms)[64 + t];   // phase 0, per pair
    const float p0m[8] = {pa.x, pa.y, pa.z, pa.w, pb.x, pb.y, pb.z, pb.w};
#pragma unroll
    for (int i = 0; i < NP; i++) {
      const int k0 = KLO + 2 * i, k1 = k0 + 1;
      const float p1m = fmaxf(fmaxf(fmaxf(pw[k0], pw[16 + k0]), fmaxf(pw[32 + k0], pw[48 + k0])),
                              fmaxf(fmaxf(pw[k1], pw[16 + k1]), fmaxf(pw[32 + k1], pw[48 + k1])));
      const float m = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(fmaxf(p0m[i], p1m))));
      own = lane == i ? m : own;
    }
  }
  __syncwarp();
  bool need = false;
  if (lane < NP) {
    const float4 b03 = *reinterpret_cast<const float4*>(ws_at(lane)), b46 = *reinterpret_cast<const float4*>(ws_at(lane) + 4);
    const float be[7] = {b03.x, b03.y, b03.z, b03.w, b46.x, b46.y, b46.z};
    float ub[4];
    harm_stage_sums(own, be, ub);
#pragma unroll
    for (int q = 0; q < 4; q++) need |= ub[q] >= rec[q].s;
    const int kp = KLO + 2 * lane;
    need = need && (min(256 * kp + 511, n_hi - 1) >= max(256 * kp, n_lo));
  }
  const uint32_t mask = __ballot_sync(0xffffffffu, need);
  __syncwarp();                                // ws is reused for the phase-1 powers of the units that gather
  return mask;
}

// One (segment, template) unit of the top-harmonic pass, called when phase 1 is done.  Phase-0 powers are in tensor
// memory at tmP, phase-1 powers in shared memory p1s (register r of thread t at r*64 + t), the per-thread phase-0
// maxima of every pair of batches in pms ([2][64] float4, written and read by the same thread); register
// r = 16 a + k holds n = t + 64 n1, n1 = 4 k + a... see harm_batch.  Point j = 2 (s0 - c + n) + ph reads sub-plane e at
// (j e + 4) >> 3 = ((jt e + 4) >> 3) + 16 n1 e with jt = 2 (s0 - c + t) + ph: one pointer per (fraction, phase), moved
// on by 64 e per k.  The loop over k is rolled (an unrolled gather body of 5000 instructions on top of the transforms
// thrashed the instruction cache: no_instruction stalls 1.2 per issue).
template <bool STORE, bool PRUNE>
__device__ __forceinline__ void harm_unit(const SearchParams& sp, const SearchJob& jb, const float (&pw)[64], float* p1s, const float* pms,
                                          uint32_t tmP, int t, int lane, int s0, int c, int ti, int n_lo, int n_hi,
                                          HarmRecord* rec, float* stash) {
  const HarmGather& hg = sp.hg;
  constexpr int KLO = PRUNE ? 1 : 0, KHI = PRUNE ? 15 : 16;   // PRUNE: k = 0 and 15 (n1 < 4, n1 >= 60) are never valid
  const long long jt = 2LL * (s0 - c + t);
  const float* q0[7];
  const float* q1[7];
  bool have = false;
  int kq = 0;
  // registers with n1 = n / 64 in [8, 56) are valid for every thread of a segment inside the box (hw_max <= 512)
  const bool inner_valid = __all_sync(0xffffffffu, n_lo <= t + 64 * 8 && n_hi >= t + 64 * 56);
  float2* dst = nullptr;
  if (STORE) {
    const int row = (ti / sp.nz - hg.out_iw_lo) * hg.out_iz_cnt + (ti % sp.nz - hg.out_iz_lo);
    dst = reinterpret_cast<float2*>(hg.out + (size_t)row * (size_t)(2 * jb.r_cnt) + 2 * (ptrdiff_t)(s0 - c - (int)jb.r_lo + t));
  }
  float mx[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
  // The gathers cost far more than the transforms (896 four-byte loads per thread and template through one L1 pipe per SM:
  // ~15 us per template and SM against 6.4 us of arithmetic), so in arg-max mode they are done only for the pairs of
  // batches whose bound (harm_bounds_need) can reach the record.  In batches of 56 independent loads per thread (about
  // what one warp can have outstanding), all issued before the first sum.
  const uint32_t need = STORE ? 0xffffffffu : harm_bounds_mask<KLO, KHI>(sp, s0, c, ti, n_lo, n_hi, lane, t, pms, pw, p1s, rec);
  if (need == 0) return;
#pragma unroll
  for (int r = 0; r < 64; r++) p1s[r * 64 + t] = pw[r];   // phase-1 powers: only for the units that gather
#pragma unroll 1
  for (int kp = KLO; kp < KHI; kp += 2) {
    if (!((need >> ((kp - KLO) >> 1)) & 1u)) continue;
    if (!have) {
      harm_pointers(sp, ti, jt, 4 * kp, q0, q1);
      have = true;
    } else {
#pragma unroll
      for (int e = 1; e <= 7; e++) {
        q0[e - 1] += 64 * e * (kp - kq);
        q1[e - 1] += 64 * e * (kp - kq);
      }
    }
    harm_batch<STORE>(hg, q0, q1, tmP, p1s, kp, t, n_lo, n_hi, inner_valid, dst, mx);
#pragma unroll
    for (int e = 1; e <= 7; e++) {
      q0[e - 1] += 64 * e;
      q1[e - 1] += 64 * e;
    }
    harm_batch<STORE>(hg, q0, q1, tmP, p1s, kp + 1, t, n_lo, n_hi, inner_valid, dst, mx);
    kq = kp + 1;     // where the pointers stand
  }
  if (STORE) return;
  // Arg-max.  Hot path: four running maxima per thread and one vote per unit.  Only when some sum of this warp reaches
  // the warp's record (initially the stage threshold) is the unit rescanned for the position.
  bool trig = false;
#pragma unroll
  for (int q = 0; q < 4; q++) trig |= mx[q] >= rec[q].s;
  if (!__any_sync(0xffffffffu, trig)) return;
  harm_pointers(sp, ti, jt, 0, q0, q1);
  float* st0 = stash;          // [64][64] phase-0 powers, register r of thread t at r*64 + t (written and read by the same thread)
#pragma unroll 1
  for (int a = 0; a < 4; a++) {
    float p0c[16];
    tmem_ld16(tmP + 16 * a, p0c);
#pragma unroll
    for (int k = 0; k < 16; k++) st0[(16 * a + k) * 64 + t] = p0c[k];
  }
  __syncwarp();
  float bs[4];
  int bj[4] = {-1, -1, -1, -1};
#pragma unroll
  for (int q = 0; q < 4; q++) bs[q] = hg.thr[q];
#pragma unroll 1
  for (int r = 0; r < 64; r++) {
    const int n1 = dft64_out_index(r);
    const int n = t + 64 * n1;
    if (n < n_lo || n >= n_hi) continue;
#pragma unroll 1
    for (int ph = 0; ph < 2; ph++) {
      const float p8 = ph ? p1s[r * 64 + t] : st0[r * 64 + t];
      float g[7];
#pragma unroll
      for (int e = 1; e <= 7; e++) g[e - 1] = __ldg((ph ? q1[e - 1] : q0[e - 1]) + 16 * n1 * e);
      float sv[4];
      harm_stage_sums(p8, g, sv);
      const int j = (int)jt + 128 * n1 + ph;
#pragma unroll
      for (int q = 0; q < 4; q++)
        if (sv[q] > bs[q] || (sv[q] == bs[q] && bj[q] >= 0 && j < bj[q])) {   // only sums above the threshold; ties -> smallest j
          bs[q] = sv[q];
          bj[q] = j;
        }
    }
  }
#pragma unroll
  for (int q = 0; q < 4; q++) {
    float b = bs[q];
    int jj = bj[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ob = __shfl_xor_sync(0xffffffffu, b, o);
      const int oj = __shfl_xor_sync(0xffffffffu, jj, o);
      if (oj >= 0 && (jj < 0 || ob > b || (ob == b && oj < jj))) {
        b = ob;
        jj = oj;
      }
    }
    if (lane == 0 && jj >= 0) {
      const HarmRecord cur = rec[q];
      if (cur.j < 0 || harm_better_ti(b, jj, ti, cur.s, cur.j, cur.ti)) {
        rec[q].s = b;
        rec[q].j = jj;
        rec[q].ti = ti;
      }
    }
  }
  __syncwarp();
}

// PRUNE (hw_max >= 256): outputs n < 256 and n >= 3840 lie outside the valid window [hw_max, 4096 - hw_max) of every
// template; they are outputs 0 and 15 of each last-stage DFT_16 (registers 16a and 16a + 15), whose final butterfly
// operations and power are then never computed (their power is reported as 0).
template <int MODE, int NG, bool PRUNE>
__global__ void __launch_bounds__(64 * NG, NG == 2 ? 2 : 1) k_search64(const __grid_constant__ SearchParams sp) {
  constexpr int L = 4096, NT = 64, P = 64;
  constexpr int NLAYER = (NG + 1) / 2;                          // groups of four warps: one TMEM lane quarter each
  constexpr int TCOLS = 128 * (NLAYER + 1) <= 256 ? 256 : 512;  // F: 128 columns per layer; twiddles: 128 columns shared by all layers
  // plane and harmonic modes park the phase-0 powers of the current template in tensor memory (64 columns of the
  // thread's own lane) until phase 1 is done: both phases then leave together (interleaved float2 pairs / harmonic sums)
  constexpr bool kStashP0 = MODE == MODE_PLANE || MODE == MODE_HARM || MODE == MODE_HARM_STORE;
  constexpr bool kBox = kStashP0;                               // the job is an (r, iz, iw) box, not the whole grid
  static_assert(!kStashP0 || NG == 4, "the phase-0 stash needs the 512-column layout");
  extern __shared__ __align__(16) unsigned char smem_raw[];
  float2* ex_all = reinterpret_cast<float2*>(smem_raw);
  unsigned long long* mbar_all = reinterpret_cast<unsigned long long*>(ex_all + NG * kEx64);  // [group][4]
  __shared__ long long s_item[NG];
  __shared__ uint32_t s_tmem;
  __shared__ HarmRecord s_rec[2 * NG][4];   // MODE_HARM: running arg-max of every warp, h = 1,2,4,8
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, grp = warp >> 1, t = threadIdx.x & 63;
  float2* ex = ex_all + grp * kEx64;
  float* p1s = reinterpret_cast<float*>(mbar_all + 4 * NG) + grp * (P * NT);   // harmonic modes: [P][NT] phase-1 powers of the group
  float* pms = reinterpret_cast<float*>(mbar_all + 4 * NG) + NG * (P * NT) + grp * (16 * NT);   // and [16][NT] per-thread maxima of every k
  const uint32_t mbS = smem_u32(mbar_all + 4 * grp);   // segment copy landed (tx)
  const uint32_t mbG = mbS + 8;                        // G copy landed (tx)
  const uint32_t mbR = mbS + 16;                       // all 64 threads have read G out of ex
  const uint32_t mbW = mbS + 24;                       // all 64 threads have finished their pass-2 loads from ex
  const int barid = 1 + grp;

  if (warp == 0) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(&s_tmem)), "n"(TCOLS));
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;");
  }
  if (t == 0) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbS));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(mbG));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbR), "r"(NT));
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(mbW), "r"(NT));
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  const uint32_t tbase = s_tmem + ((uint32_t)((warp & 3) * 32) << 16);
  TmemArray<L> tmF, tmT;
  tmF.addr = tbase + 128 * (warp >> 2);
  tmT.addr = tbase + 128 * NLAYER;
  const uint32_t tmP = tbase + 128 * (NLAYER + 1) + 64 * (warp >> 2);   // phase-0 power stash (kStashP0)
  if (MODE == MODE_HARM && lane < 4) {
    s_rec[warp][lane].s = sp.hg.thr[lane];
    s_rec[warp][lane].j = -1;
    s_rec[warp][lane].ti = 0;
  }
  if (warp < 4) {   // the twiddles depend on t = thread index mod 64 only: one copy per TMEM lane serves every layer
#pragma unroll
    for (int h = 0; h < 4; h++) {
      float2 w[16];
#pragma unroll
      for (int i = 0; i < 16; i++) w[i] = tw64_mixed(16 * h + i, t);
      tmT.store16(h, w);
    }
  }
  asm volatile("tcgen05.fence::before_thread_sync;");
  __syncthreads();
  asm volatile("tcgen05.fence::after_thread_sync;");
  uint32_t sphase = 0;   // parity of the segment-copy mbarrier
  uint32_t tphase = 0;   // parity of mbG, mbR and mbW: each completes exactly one phase per template-phase
  const auto nohook = [] {};
  const long long nitems = sp.nitems;

  for (;;) {
    if (t == 0) s_item[grp] = (long long)atomicAdd(sp.work, 1ULL);
    bar_sync_named(barid, NT);
    const long long item = s_item[grp];
    if (item >= nitems) break;
    const WorkItem wi = decode_item(sp, item);
    const SearchJob& jb = sp.jobs[wi.q];
    const float2* spec = sp.spec[wi.b];
    const int iz_cnt = jb.iz_cnt;
    const int hw_j = jb.hw, step_j = jb.step;                          // this job's overlap (SearchJob)
    const int s0 = (int)(jb.seg_base + wi.seg * (int64_t)step_j);      // first bin of the segment (even); |s0| < 2^31 (nbins <= 2^30)

    // ---- a-2: stage the segment in the exchange buffer: TMA bulk copy when fully inside the spectrum, guarded loads at the edges
    const bool interior = (s0 >= 0) && ((int64_t)s0 + L <= sp.nbins);
    if (interior) {
      if (t == 0) bulk_copy_g2s(smem_u32(ex), spec + s0, (uint32_t)(L * 8), mbS);
      mbar_wait(mbS, sphase);
      sphase ^= 1u;
    } else {
      for (int k = t; k < L; k += NT) {
        const int64_t b = (int64_t)s0 + k;
        ex[k] = (b >= 0 && b < sp.nbins) ? spec[b] : make_float2(0.f, 0.f);
      }
      bar_sync_named(barid, NT);
    }
    // ---- forward FFT; F goes to TMEM in the pass-1 layout: array index k1 holds F[64*k1 + t]
    {
      float2 v[P];
#pragma unroll
      for (int k1 = 0; k1 < 64; k1++) v[k1] = ex[64 * k1 + t];
      bar_sync_named(barid, NT);                         // ex is about to be reused as the exchange buffer
      fft64_passes<-1>(v, tmT, ex, t, barid, nohook, nohook, nohook);
      bar_sync_named(barid, NT);                         // all pass-2 loads of ex done
#pragma unroll
      for (int r = 0; r < 64; r++) ex[t + 64 * dft64_out_index(r)] = v[r];
      bar_sync_named(barid, NT);
      // chunk h of the tensor-memory copy serves the radix-4 butterflies b = 4h .. 4h+3 of pass 1: entry 4 m + a = F[64 (16 a + 4 h + m) + t]
#pragma unroll
      for (int h = 0; h < 4; h++) {
        float2 fq[16];
#pragma unroll
        for (int i = 0; i < 16; i++) fq[i] = ex[64 * (16 * (i & 3) + 4 * h + (i >> 2)) + t];
        tmF.store16(h, fq);
      }
      bar_sync_named(barid, NT);
    }

    // ---- loop over the template-phases of this chunk (numbetween = 1: one phase per template, tp = template)
    const bool two = sp.nb == 2;
    const int tp_lo = wi.chunk * jb.chunk_tp;
    const int tp_hi = min(jb.ntp, tp_lo + jb.chunk_tp);
    int any0 = 0;  // candidate mode: phase-0 powers of this warp exceeded the threshold and were stashed
    // template walk of the box, row-major: ti_n = index of the template of the NEXT template-phase, iz_left = templates
    // left in its w-row
    // (an overlap class walks its list jb.order instead: tl_n = position of the next template in it)
    int ti_n, iz_left;
    const int* order = jb.order;
    int tl_n = two ? tp_lo >> 1 : tp_lo;
    {
      const int izr = tl_n % iz_cnt, iwr = tl_n / iz_cnt;
      ti_n = order ? __ldg(order + tl_n) : (jb.iw_lo + iwr) * sp.nz + jb.iz_lo + izr;
      iz_left = iz_cnt - izr;
    }
    if (t == 0)   // G of the first template-phase of the item (ex is free: the barrier above; chunks start at phase 0)
      bulk_copy_g2s(smem_u32(ex), sp.G + (size_t)ti_n * sp.nb * L, (uint32_t)(L * 8), mbG);
    uint32_t g_ready = 0;   // answer of the probe of mbG started before the epilogue of the previous template-phase
    for (int tp = tp_lo; tp < tp_hi; tp++) {
      const int ph = two ? (tp & 1) : 0;
      const int ti = ti_n;
      const int c = sp.geom[ti].c;
      // next template-phase: the same template's phase 1, or phase 0 of the next template of the box
      if (ph == 1 || !two) {
        if (order) {
          ++tl_n;
          if (tp + 1 < tp_hi) ti_n = __ldg(order + tl_n);
        } else {
          ++ti_n;
          if (--iz_left == 0) {
            iz_left = iz_cnt;
            ti_n += sp.nz - iz_cnt;
          }
        }
      }
      // ---- a-3: Y = F .* G (G from the exchange buffer, F from TMEM), inverse FFT
      float2 v[P];
      if (!g_ready) mbar_wait(mbG, tphase);
      __syncwarp();   // tcgen05.ld is .sync.aligned: the warp must be converged
      {
        const float4* g4 = reinterpret_cast<const float4*>(ex) + t;
        float fa[32], fb[32];   // F chunks, double-buffered: chunk h+1 is in flight while chunk h is multiplied
        tmF.issue16(0, fa);
#pragma unroll
        for (int h = 0; h < 4; h++) {
          float(&cur)[32] = (h & 1) ? fb : fa;
          float(&nxt)[32] = (h & 1) ? fa : fb;
          tmem_ld32_wait(cur);
          if (h < 3) tmF.issue16(h + 1, nxt);
          // Y = F .* G fused with the first radix-4 layer of the inverse transform: the bank holds G in the mixed form
          // of dft16_layerA_tw, (g0.re, g0.im), (c1, t1), (c2, t2), (c3 / c1, t3) with g = c (1 + i t), so a butterfly of
          // four products costs 13 packed instructions instead of 8 + 8
#pragma unroll
          for (int m = 0; m < 4; m++) {
            const int b = 4 * h + m;
            const float4 ga = g4[(8 * h + 2 * m) * NT], gb = g4[(8 * h + 2 * m + 1) * NT];
            const float2 w[4] = {make_float2(ga.x, ga.y), make_float2(ga.z, ga.w), make_float2(gb.x, gb.y), make_float2(gb.z, gb.w)};
            float2 x0 = make_float2(cur[8 * m], cur[8 * m + 1]), x1 = make_float2(cur[8 * m + 2], cur[8 * m + 3]);
            float2 x2 = make_float2(cur[8 * m + 4], cur[8 * m + 5]), x3 = make_float2(cur[8 * m + 6], cur[8 * m + 7]);
            dft16_layerA_tw<1, false>(x0, x1, x2, x3, w);
            v[b] = x0;
            v[16 + b] = x1;
            v[32 + b] = x2;
            v[48 + b] = x3;
          }
        }
      }
      mbar_arrive(mbR);
      uint32_t r_ready = 0;
      const auto mid = [&] { r_ready = mbar_probe(mbR, tphase); };
      const auto pre = [&] {
        if (!r_ready) mbar_wait(mbR, tphase);
      };
      const auto post = [&] {
        mbar_arrive(mbW);
        if (t == 0 && tp + 1 < tp_hi) {
          mbar_wait(mbW, tphase);
          bulk_copy_g2s(smem_u32(ex), sp.G + ((size_t)ti_n * sp.nb + (two ? ph ^ 1 : 0)) * L, (uint32_t)(L * 8), mbG);
        }
        __syncwarp();
      };
      fft64_passes<1, true>(v, tmT, ex, t, barid, mid, pre, post);
      tphase ^= 1u;
      g_ready = tp + 1 < tp_hi ? mbar_probe(mbG, tphase) : 0u;   // has the next G landed?  (asked now, needed after the epilogue)
      // ---- a-4: overlap discard + power.  n = t + 64*n1 ; b = s0 + n - c ; j = 2b + ph.
      // valid outputs: n in [n_lo, n_hi) = window [hw_max, hw_max + step) clipped to the bins this call covers (32-bit: all
      // bin indices are below 2^30)
      int n_lo, n_hi;
      {
        const int blo = kBox ? (int)jb.r_lo : 0, bhi = kBox ? (int)(jb.r_lo + jb.r_cnt) : (int)sp.nbins;
        n_lo = max(hw_j, min(blo - s0 + c, L));
        n_hi = min(hw_j + step_j, max(bhi - s0 + c, 0));
      }
      float pw[P];
#pragma unroll
      for (int i = 0; i < P; i++)
        pw[i] = (PRUNE && ((i & 15) == 0 || (i & 15) == 15)) ? 0.f : fmaf(v[i].x, v[i].x, v[i].y * v[i].y);
      if (kStashP0 && two && ph == 0) {
#pragma unroll
        for (int h = 0; h < 2; h++) {
          float q32[32];
#pragma unroll
          for (int i = 0; i < 32; i++) q32[i] = pw[32 * h + i];
          tmem_st32(tmP + 32 * h, q32);
        }
        if (MODE == MODE_HARM) {   // the largest phase-0 power of the four registers 16 a + k of every k (bounds of harm_unit)
#pragma unroll
          for (int q4 = 0; q4 < 2; q4++) {   // per pair of batches (k = KLO + 2 i, KLO + 2 i + 1): [2][NT] float4, pairs 4 q4 .. 4 q4 + 3
            float pm[4];
#pragma unroll
            for (int u = 0; u < 4; u++) {
              const int k0 = (PRUNE ? 1 : 0) + 2 * (4 * q4 + u), k1 = k0 + 1;
              pm[u] = k1 < 16 ? fmaxf(fmaxf(fmaxf(pw[k0], pw[16 + k0]), fmaxf(pw[32 + k0], pw[48 + k0])),
                                      fmaxf(fmaxf(pw[k1], pw[16 + k1]), fmaxf(pw[32 + k1], pw[48 + k1])))
                              : 0.f;
            }
            reinterpret_cast<float4*>(pms)[q4 * NT + t] = make_float4(pm[0], pm[1], pm[2], pm[3]);
          }
        }
      } else if (MODE == MODE_PLANE && !two) {
        // numbetween = 1: one float per bin, row index = template
        float* dst = jb.plane + (size_t)tp * (size_t)jb.r_cnt + (ptrdiff_t)(s0 - c - (int)jb.r_lo + t);
#pragma unroll
        for (int r = 0; r < P; r++) {
          if (PRUNE && ((r & 15) == 0 || (r & 15) == 15)) continue;
          const int n1 = dft64_out_index(r);
          const int n = t + 64 * n1;
          if (n >= n_lo && n < n_hi) dst[64 * n1] = pw[r];
        }
      } else if (MODE == MODE_PLANE) {
        // both phases leave as interleaved float2 pairs: every warp store covers 256 contiguous bytes (full 32-byte
        // sectors, no L2 fill reads)
        float* row = jb.plane + (size_t)(tp >> 1) * (size_t)(2 * jb.r_cnt);   // row-major box: row index = template-phase / 2
        const int boff = s0 - c - (int)jb.r_lo;
        float2* dst = reinterpret_cast<float2*>(row + 2 * (ptrdiff_t)(boff + t));   // + 64 n1 float2 per register
        // registers with n1 = n / 64 in [8, 56) are valid for every thread of a segment inside the box (hw_max <= 512):
        // no predicate; registers known to be outside every window (PRUNE) are skipped
        const bool inner_valid = __all_sync(0xffffffffu, n_lo <= t + 64 * 8 && n_hi >= t + 64 * 56);
        float bm[kBmaxBlocks];   // block maxima of this thread's valid outputs (both phases); powers are >= 0
#pragma unroll
        for (int g = 0; g < kBmaxBlocks; g++) bm[g] = 0.f;
        // two copies of the store loop, chosen by a warp-uniform branch: with inner_valid the 48 inner registers need no predicate at all
        const auto emit = [&](auto inner_c) {
          constexpr bool INNER = decltype(inner_c)::value;
#pragma unroll
          for (int h = 0; h < 2; h++) {
            float p0c[32];
            tmem_ld32(tmP + 32 * h, p0c);
#pragma unroll
            for (int i = 0; i < 32; i++) {
              const int r = 32 * h + i;
              if (PRUNE && ((r & 15) == 0 || (r & 15) == 15)) continue;
              const int n1 = dft64_out_index(r);
              const int n = t + 64 * n1;
              const bool ok = (INNER && n1 >= 8 && n1 < 56) ? true : (n >= n_lo && n < n_hi);
              if (ok) {
                dst[64 * n1] = make_float2(p0c[i], pw[r]);
                bm[bmax_block(64 * n1)] = fmaxf(bm[bmax_block(64 * n1)], fmaxf(p0c[i], pw[r]));
              }
            }
          }
        };
        if (inner_valid) emit(std::true_type{});
        else emit(std::false_type{});
        if (jb.bmax) {   // one value per (row, segment, block, warp of the group): plain stores, every entry has one owner
          // (powers are >= 0, so their bit patterns order like unsigned integers: one warp reduction per block)
#pragma unroll
          for (int g = 0; g < kBmaxBlocks; g++) bm[g] = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(bm[g])));
          if (lane < kBmaxBlocks) {
            float mine = bm[0];
#pragma unroll
            for (int g = 1; g < kBmaxBlocks; g++) mine = lane == g ? bm[g] : mine;
            jb.bmax[((((size_t)(tp >> 1) * jb.seg_count + (wi.seg - jb.seg_first)) * kBmaxBlocks + lane) << 1) + (warp & 1)] = mine;
          }
        }
      } else if (MODE == MODE_HARM || MODE == MODE_HARM_STORE) {
        harm_unit<MODE == MODE_HARM_STORE, PRUNE>(sp, jb, pw, p1s, pms, tmP, t, lane, s0, c, ti, n_lo, n_hi, s_rec[warp],
                                                   sp.stash + ((size_t)blockIdx.x * NG + grp) * (2 * L));
      } else {
        if (MODE == MODE_CAND_STATS) {
          // SURVEY.md 8(f) N2 / PAPER.md:43,45: mean and standard deviation of every (z,w) row, fused: sum of P and P^2
          // over the valid points of this unit, one fp64 atomic pair per warp
          // four independent accumulator pairs (no 64-long dependent chains); registers whose n1 = n / 64 lies in [8, 56)
          // are valid for every thread of an interior segment (hw_max <= 512) and are summed without a predicate
          // (packed: two powers per FADD2 / FFMA2, two accumulator pairs per sum)
          float2 b1[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)}, b2[2] = {make_float2(0.f, 0.f), make_float2(0.f, 0.f)};
          const bool inner_valid = __all_sync(0xffffffffu, n_lo <= t + 64 * 8 && n_hi >= t + 64 * 56);
          if (inner_valid) {
#pragma unroll
            for (int r = 0; r < P; r += 2) {
              float pa = pw[r], pb = pw[r + 1];
              const int n1a = dft64_out_index(r), n1b = dft64_out_index(r + 1);
              if (n1a < 8 || n1a >= 56) {
                const int n = t + 64 * n1a;
                pa = (n >= n_lo && n < n_hi) ? pa : 0.f;
              }
              if (n1b < 8 || n1b >= 56) {
                const int n = t + 64 * n1b;
                pb = (n >= n_lo && n < n_hi) ? pb : 0.f;
              }
              const float2 pp = make_float2(pa, pb);
              b1[(r >> 1) & 1] = __fadd2_rn(b1[(r >> 1) & 1], pp);
              b2[(r >> 1) & 1] = __ffma2_rn(pp, pp, b2[(r >> 1) & 1]);
            }
          } else {
#pragma unroll
            for (int r = 0; r < P; r += 2) {
              const int na = t + 64 * dft64_out_index(r), nb2 = t + 64 * dft64_out_index(r + 1);
              const float2 pp = make_float2((na >= n_lo && na < n_hi) ? pw[r] : 0.f, (nb2 >= n_lo && nb2 < n_hi) ? pw[r + 1] : 0.f);
              b1[(r >> 1) & 1] = __fadd2_rn(b1[(r >> 1) & 1], pp);
              b2[(r >> 1) & 1] = __ffma2_rn(pp, pp, b2[(r >> 1) & 1]);
            }
          }
          const float a1[4] = {b1[0].x, b1[0].y, b1[1].x, b1[1].y}, a2[4] = {b2[0].x, b2[0].y, b2[1].x, b2[1].y};
          float s1 = (a1[0] + a1[1]) + (a1[2] + a1[3]), s2 = (a2[0] + a2[1]) + (a2[2] + a2[3]);
#pragma unroll
          for (int o = 16; o > 0; o >>= 1) {
            s1 += __shfl_xor_sync(0xffffffffu, s1, o);
            s2 += __shfl_xor_sync(0xffffffffu, s2, o);
          }
          if (lane == 0) {
            atomicAdd(sp.rowstats + 2 * (size_t)ti, (double)s1);
            atomicAdd(sp.rowstats + 2 * (size_t)ti + 1, (double)s2);
          }
        }
        // ---- a-5: threshold + local max.  Hot path: one max-reduction and a vote.
        float mx = pw[0];
#pragma unroll
        for (int i = 1; i < P; i++) mx = fmaxf(mx, pw[i]);
        const int anyhit = __any_sync(0xffffffffu, mx > sp.threshold);
        // rare-path stash of the group: [2][P][NT] powers of the current template; register i of thread t at i*NT + t
        // (written and read by the same thread)
        float* st0 = sp.stash + ((size_t)blockIdx.x * NG + grp) * (2 * L);
        float* st1 = st0 + L;
        const float NEG = -INFINITY;
        if (!two) {
          if (anyhit) {       // numbetween = 1: the neighbours of bin b are bins b - 1 and b + 1 of the same phase
#pragma unroll
            for (int i = 0; i < P; i++) st0[i * NT + t] = pw[i];
            __syncwarp();
            const int iz = ti % sp.nz, iw = ti / sp.nz;
#pragma unroll 1
            for (int i = 0; i < P; i++) {
              const int n = t + 64 * dft64_out_index(i);
              const bool valid = (n >= n_lo) && (n < n_hi);
              const float p = valid ? st0[i * NT + t] : NEG;
              const float l = __shfl_up_sync(0xffffffffu, p, 1);      // P[b-1]
              const float r = __shfl_down_sync(0xffffffffu, p, 1);    // P[b+1]
              if (!valid) continue;
              const int b = s0 + n - c;
              test_point(sp, wi.b, b, iz, iw, p, b > 0 ? l : NEG, b < (int)sp.nbins - 1 ? r : NEG,
                         (lane == 0 || n == hw_j) && (b > 0), (lane == 31 || n == hw_j + step_j - 1) && (b < (int)sp.nbins - 1));
            }
            __syncwarp();
          }
        } else if (ph == 0) {
          any0 = anyhit;
          if (anyhit) {
#pragma unroll
            for (int i = 0; i < P; i++) st0[i * NT + t] = pw[i];
          }
        } else if (anyhit | any0) {
#pragma unroll
          for (int i = 0; i < P; i++) st1[i * NT + t] = pw[i];
          __syncwarp();
          const int iz = ti % sp.nz, iw = ti / sp.nz;
#pragma unroll 1
          for (int i = 0; i < P; i++) {
            const int n = t + 64 * dft64_out_index(i);
            const bool valid = (n >= n_lo) && (n < n_hi);
            const float p1 = valid ? st1[i * NT + t] : NEG;
            const float p0 = (valid && any0) ? st0[i * NT + t] : NEG;
            const float l1 = __shfl_up_sync(0xffffffffu, p1, 1);    // P1[n-1]
            const float r0 = __shfl_down_sync(0xffffffffu, p0, 1);  // P0[n+1]
            if (!valid) continue;
            const int b = s0 + n - c;
            // phase-0 point j = 2b: left neighbour (b-1, phase 1), right neighbour (b, phase 1)
            test_point(sp, wi.b, 2 * b, iz, iw, p0, b > 0 ? l1 : NEG, p1, (lane == 0 || n == hw_j) && (b > 0), false);
            // phase-1 point j = 2b+1: left neighbour (b, phase 0), right neighbour (b+1, phase 0)
            test_point(sp, wi.b, 2 * b + 1, iz, iw, p1, p0, b < (int)sp.nbins - 1 ? r0 : NEG, false,
                       (lane == 31 || n == hw_j + step_j - 1) && (b < (int)sp.nbins - 1));
          }
          __syncwarp();
        }
      }
    }
    bar_sync_named(barid, NT);
  }
  if (MODE == MODE_HARM) {
    __syncwarp();
    if (lane < 4) {
      const HarmRecord rc = s_rec[warp][lane];
      jerk_cand c;
      c.j = rc.j;
      c.iz = (int16_t)(rc.ti % sp.nz);
      c.iw = (int16_t)(rc.ti / sp.nz);
      c.power = rc.s;
      c.flags = 0;
      sp.hg.warpbest[(size_t)lane * (gridDim.x * 2 * NG) + blockIdx.x * 2 * NG + warp] = c;
    }
  }
  __syncthreads();
  if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(s_tmem), "n"(TCOLS));
}

// Seam records: every above-threshold point whose left (phase 0) or right (phase 1) neighbour belongs to another
// warp or segment.  A seam point is a candidate iff it passed its own-side test and no seam record at the missing
// neighbour position beats it (a neighbour that emitted nothing is <= threshold < this power).  A point is owned by
// exactly one (segment, warp), so a position appears at most once in the list.  Short lists are settled by direct
// comparison; longer ones through an open-addressing hash table on (template, j) built in the stash region, which is
// idle once the search kernel has finished.  A list that did not fit in d_work cannot be settled: the call then reports
// *d_count = UINT64_MAX (include/jerk.h), never a silently shortened result.
constexpr unsigned long long kSeamDirect = 512;        // lists up to this length: O(n^2) scan in k_seam_resolve alone
constexpr unsigned long long kSeamHashMaxSlots = 1ull << 23;   // 32 MB of the 37 MB stash; seam_cap <= slots / 2

__device__ __forceinline__ unsigned long long seam_count(const SearchParams& sp) {
  const unsigned long long ns = sp.work[1];
  return ns > sp.seam_cap ? sp.seam_cap : ns;
}
__device__ __forceinline__ uint32_t seam_slots(unsigned long long ns) {      // power of two >= 4 ns, at most kSeamHashMaxSlots (>= 2 ns: seam_cap)
  uint32_t m = 2048;
  while ((unsigned long long)m < 4 * ns && m < kSeamHashMaxSlots) m <<= 1;
  return m;
}
__device__ __forceinline__ uint32_t seam_hash(int ti, int j, uint32_t mask) {
  unsigned long long k = ((unsigned long long)(uint32_t)ti << 32) | (uint32_t)j;
  k *= 0x9E3779B97F4A7C15ull;
  return (uint32_t)(k >> 32) & mask;
}
__global__ void k_seam_clear(SearchParams sp) {
  const unsigned long long ns = seam_count(sp);
  if (ns <= kSeamDirect || sp.work[2]) return;
  uint32_t* table = reinterpret_cast<uint32_t*>(sp.stash);
  const uint32_t m = seam_slots(ns);
  for (uint32_t i = blockIdx.x * blockDim.x + threadIdx.x; i < m; i += gridDim.x * blockDim.x) table[i] = 0u;
}
__device__ __forceinline__ int seam_row(const SearchParams& sp, const jerk_cand& a) {   // (spectrum, template) of a record
  return (int)(a.flags >> 8) * (sp.nz * sp.nw_grid) + a.iw * sp.nz + a.iz;
}
__global__ void k_seam_insert(SearchParams sp) {
  const unsigned long long ns = seam_count(sp);
  if (ns <= kSeamDirect || sp.work[2]) return;
  uint32_t* table = reinterpret_cast<uint32_t*>(sp.stash);
  const uint32_t mask = seam_slots(ns) - 1;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < ns;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    const jerk_cand a = sp.seams[i];
    uint32_t h = seam_hash(seam_row(sp, a), a.j, mask);
    while (atomicCAS(table + h, 0u, (uint32_t)i + 1u) != 0u) h = (h + 1) & mask;
  }
}
// power of the seam record at (row, j), -inf when there is none (that point was not above the threshold)
__device__ __forceinline__ float seam_lookup(const SearchParams& sp, unsigned long long ns, bool direct, const uint32_t* table,
                                             uint32_t mask, int row, int j) {
  if (direct) {
    for (unsigned long long k = 0; k < ns; k++) {
      const jerk_cand b = sp.seams[k];
      if (b.j == j && seam_row(sp, b) == row) return b.power;
    }
    return -INFINITY;
  }
  uint32_t h = seam_hash(row, j, mask);
  for (uint32_t e; (e = table[h]) != 0u; h = (h + 1) & mask) {
    const jerk_cand b = sp.seams[e - 1];
    if (b.j == j && seam_row(sp, b) == row) return b.power;
  }
  return -INFINITY;
}
__global__ void k_seam_resolve(SearchParams sp) {
  if (sp.work[2]) {      // the seam list overflowed d_work: the result would be incomplete
    if (blockIdx.x == 0 && threadIdx.x < sp.nspec) sp.count[threadIdx.x] = ~0ULL;
    return;
  }
  const unsigned long long ns = seam_count(sp);
  const bool direct = ns <= kSeamDirect;
  const uint32_t* table = reinterpret_cast<const uint32_t*>(sp.stash);
  const uint32_t mask = seam_slots(ns) - 1;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < ns;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    const jerk_cand a = sp.seams[i];
    if (a.flags & SEAM_WITNESS) continue;
    const int row = seam_row(sp, a);
    bool ok = true;
    if (a.flags & SEAM_LEFT) ok = a.power > seam_lookup(sp, ns, direct, table, mask, row, a.j - 1);            // P > P[j-1]
    if (ok && (a.flags & SEAM_RIGHT)) ok = a.power >= seam_lookup(sp, ns, direct, table, mask, row, a.j + 1);   // P >= P[j+1]
    if (ok) {
      atomicAdd(sp.work + 3, 1ULL);
      emit_cand(sp, (int)(a.flags >> 8), a.j, a.iz, a.iw, a.power);
    }
  }
}

// S/N filter of a candidate list ("above a certain threshold" in units of the output's
// standard deviation): snr = (P - mean_row) / std_row with the row statistics of k_search64<MODE_CAND_STATS>.
__global__ void k_snr_filter(const double* __restrict__ rowstats, int nz, double npts_row, const jerk_cand* __restrict__ in,
                             const unsigned long long* __restrict__ count_in, long long max_in, float snr_thr, jerk_cand* out,
                             long long max_out, unsigned long long* count_out) {
  unsigned long long n = *count_in;
  if (n > (unsigned long long)max_in) n = (unsigned long long)max_in;
  for (unsigned long long i = blockIdx.x * (unsigned long long)blockDim.x + threadIdx.x; i < n;
       i += (unsigned long long)gridDim.x * blockDim.x) {
    jerk_cand c = in[i];
    const size_t ti = (size_t)c.iw * nz + c.iz;
    const double mean = rowstats[2 * ti] / npts_row;
    const double var = rowstats[2 * ti + 1] / npts_row - mean * mean;
    if (!(var > 0.0)) continue;
    const float snr = (float)(((double)c.power - mean) / sqrt(var));
    if (snr > snr_thr) {
      const unsigned long long slot = atomicAdd(count_out, 1ULL);
      if ((long long)slot < max_out) {
        c.flags = __float_as_uint(snr);
        out[slot] = c;
      }
    }
  }
}

// Cross-row sifting (second half; PAPER.md:47 names it as future work): a strong signal yields one
// local-max candidate in every nearby (z,w) row.  Non-maximum suppression over the candidate list: a candidate is dropped
// iff another one within |dj| <= wj, |diz| <= wz, |diw| <= ww beats it (larger power; ties -> smaller (iw, iz, j)).
// The rule does not depend on the order of the list.  O(n^2) pair tests, tiled through shared memory.
__device__ __forceinline__ bool sift_beats(const jerk_cand& b, const jerk_cand& a) {
  if (b.power != a.power) return b.power > a.power;
  if (b.iw != a.iw) return b.iw < a.iw;
  if (b.iz != a.iz) return b.iz < a.iz;
  return b.j < a.j;
}
__global__ void __launch_bounds__(256) k_sift(const jerk_cand* __restrict__ in, const unsigned long long* __restrict__ count_in,
                                              long long max_in, int wj, int wz, int ww, jerk_cand* out, long long max_out,
                                              unsigned long long* count_out) {
  __shared__ jerk_cand tile[256];
  unsigned long long n64 = *count_in;
  if (n64 > (unsigned long long)max_in) n64 = (unsigned long long)max_in;
  const int n = (int)n64;
  for (int base = blockIdx.x * 256; base < n; base += gridDim.x * 256) {
    const int i = base + threadIdx.x;
    jerk_cand a;
    a.j = 0; a.iz = a.iw = 0; a.power = 0.f; a.flags = 0;
    if (i < n) a = in[i];
    bool alive = i < n;
    for (int t0 = 0; t0 < n; t0 += 256) {
      __syncthreads();
      if (t0 + (int)threadIdx.x < n) tile[threadIdx.x] = in[t0 + threadIdx.x];
      __syncthreads();
      const int m = min(256, n - t0);
      for (int k = 0; k < m; k++) {
        const jerk_cand b = tile[k];
        const bool near = abs(b.j - a.j) <= wj && abs((int)b.iz - (int)a.iz) <= wz && abs((int)b.iw - (int)a.iw) <= ww;
        if (near && (t0 + k != i) && sift_beats(b, a)) alive = false;
      }
    }
    if (alive) {
      const unsigned long long slot = atomicAdd(count_out, 1ULL);
      if ((long long)slot < max_out) out[slot] = a;
    }
  }
}

// Overlap classes of a candidate search (SearchJob::order): the templates of up to three boxes of the grid, in row-major
// order, are distributed over classes of similar half-width, class = (hw - hw_lo) / width, each class keeping the
// row-major order (stable, so the list is the same on every call).  One block; out[cls_off[class] + rank] = ti.
struct OrderParams {
  int nboxes;
  int iz_lo[3], iz_cnt[3], iw_lo[3], iw_cnt[3];
  int total;                  // templates of all boxes
  int hw_lo, width;
  int cls_off[kMaxJobs];      // first position of every class in `out`
  const TemplateGeom* geom;
  int nz;
  int* out;
};
__global__ void __launch_bounds__(1024) k_order(const OrderParams op) {
  __shared__ int cursor[kMaxJobs];
  __shared__ int wc[32][kMaxJobs];    // templates of every class held by every warp in the current tile
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  if (tid < kMaxJobs) cursor[tid] = op.cls_off[tid];
  for (int base = 0; base < op.total; base += 1024) {
    if (tid < 32 * kMaxJobs) (&wc[0][0])[tid] = 0;
    __syncthreads();
    int i = base + tid, cls = -1, ti = 0;
    if (i < op.total) {
      int b = 0;
      while (b + 1 < op.nboxes && i >= op.iz_cnt[b] * op.iw_cnt[b]) {
        i -= op.iz_cnt[b] * op.iw_cnt[b];
        b++;
      }
      ti = (op.iw_lo[b] + i / op.iz_cnt[b]) * op.nz + op.iz_lo[b] + i % op.iz_cnt[b];
      cls = (op.geom[ti].hw - op.hw_lo) / op.width;
    }
    const unsigned same = __match_any_sync(0xffffffffu, cls);
    const int rank = __popc(same & ((1u << lane) - 1u));
    if (cls >= 0 && rank == 0) wc[warp][cls] = __popc(same);
    __syncthreads();
    if (cls >= 0) {
      int off = cursor[cls] + rank;
      for (int w = 0; w < warp; w++) off += wc[w][cls];
      op.out[off] = ti;
    }
    __syncthreads();
    if (tid < kMaxJobs) {
      int n = 0;
      for (int w = 0; w < 32; w++) n += wc[w][tid];
      cursor[tid] += n;
    }
    __syncthreads();
  }
}

__global__ void k_reset(unsigned long long* work, unsigned long long* count, int ncount) {
  if (threadIdx.x < 8) work[threadIdx.x] = 0ULL;
  if (count && (int)threadIdx.x < ncount) count[threadIdx.x] = 0ULL;
}

// ------------------------------------------------------------------------------------------------- harmonic stage
// Row a-6 (BASELINE.json configs[4]; reading S13):  S_h(j,iz',iw') = sum_{k=1..h} P[rnd(j k/h); rnd(iz' k/h), rnd(iw' k/h)]
// with signed grid indices and rnd = round half away from zero.  Every fraction k/h of h in {1,2,4,8} is e/8, e = 1..8, and
// the stage sums nest:  S1 = P8;  S2 = S1 + P4;  S4 = S2 + P2 + P6;  S8 = S4 + P1 + P3 + P5 + P7   (Pe = sub-plane of e/8).
struct HarmSub {           // sub-plane of fraction e/8 for the current box, as written by the plane-mode search kernel
  const float* base;       // P[iw_rel][iz_rel][j - j0]
  long long j0, nj;        // first half-bin index stored (even) and row length
  int iz_lo, iz_cnt, iw_lo;
};
struct HarmParams {
  HarmSub sub[8];          // index e-1
  long long j_lo, nj;      // top-harmonic box along r, half-bin indices [j_lo, j_lo+nj)
  int iz_lo, iz_cnt, iw_lo, iw_cnt;
  int cz, cw;              // centre indices (nz-1)/2, (nw-1)/2
  int jtile, ntiles;       // half-bin indices per block, blocks per (iz,iw) row
  jerk_cand* blockbest;    // arg-max mode: [4][nblocks] best of each block for h = 1,2,4,8
  float* out;              // store mode: S_h of the box, out[iw_rel][iz_rel][j - j_lo]
  int out_stage;           // store mode: log2(h)
};

// better(a, b): a beats b as the arg-max: larger sum, ties -> smallest (iw, iz, j) in row-major order
__device__ __forceinline__ bool harm_better(float sa, int ja, int iza, int iwa, float sb, int jb, int izb, int iwb) {
  if (sa != sb) return sa > sb;
  if (iwa != iwb) return iwa < iwb;
  if (iza != izb) return iza < izb;
  return ja < jb;
}

template <bool STORE>
__global__ void __launch_bounds__(256) k_harm(const __grid_constant__ HarmParams hp) {
  const int tile = blockIdx.x % hp.ntiles;
  const int row = blockIdx.x / hp.ntiles;
  const int izr = row % hp.iz_cnt, iwr = row / hp.iz_cnt;
  const int iz = hp.iz_lo + izr, iw = hp.iw_lo + iwr;
  const int az = iz - hp.cz, aw = iw - hp.cw;
  // tile [jb, je) of half-bin indices; all index arithmetic inside the tile is 32-bit relative to j8 = jb rounded down
  // to a multiple of 8:  (j e + 4) >> 3 = (j8 / 8) e + ((jl e + 4) >> 3),  jl = j - j8
  const long long jb = hp.j_lo + (long long)tile * hp.jtile;
  const long long je = min(hp.j_lo + hp.nj, jb + hp.jtile);
  const long long j8 = jb & ~7LL;
  const int l_lo = (int)(jb - j8), l_hi = (int)(je - j8);
  const float* rp[8];
#pragma unroll
  for (int e = 1; e <= 8; e++) {
    const HarmSub& sb = hp.sub[e - 1];
    const int ize = rnd_eighths(az, e) + hp.cz, iwe = rnd_eighths(aw, e) + hp.cw;
    rp[e - 1] = sb.base + ((long long)(iwe - sb.iw_lo) * sb.iz_cnt + (ize - sb.iz_lo)) * sb.nj - sb.j0 + (j8 >> 3) * e;
  }
  float best[4] = {-INFINITY, -INFINITY, -INFINITY, -INFINITY};
  int bj[4] = {-1, -1, -1, -1};
  float* orow = STORE ? hp.out + ((long long)iwr * hp.iz_cnt + izr) * hp.nj - hp.j_lo + j8 : nullptr;
  // Strength-reduced gathers: for l = l0 + 256 k the source index ((l e + 4) >> 3) = ((l0 e + 4) >> 3) + 32 k e exactly, and
  // l0 advances by 1024 per iteration, so every thread keeps one pointer per fraction, reads at compile-time offsets
  // and bumps the pointer by 128 e floats per iteration (the kernel was issue-bound on index arithmetic: 107
  // instructions per point, ALU pipe 71 % busy).
  constexpr int U = 4;   // points per thread in flight: 32 independent loads before the first use
  const int l_first = l_lo + (int)threadIdx.x;
  const float* pe_ptr[8];
#pragma unroll
  for (int e = 1; e <= 8; e++) pe_ptr[e - 1] = rp[e - 1] + ((l_first * e + 4) >> 3);
  for (int l0 = l_first; l0 < l_hi; l0 += 256 * U) {
    float pe[U][8];
#pragma unroll
    for (int k = 0; k < U; k++) {
      const bool ok = l0 + 256 * k < l_hi;
#pragma unroll
      for (int e = 1; e <= 8; e++) pe[k][e - 1] = ok ? __ldg(pe_ptr[e - 1] + 32 * k * e) : 0.f;
    }
#pragma unroll
    for (int e = 1; e <= 8; e++) pe_ptr[e - 1] += 32 * U * e;
#pragma unroll
    for (int k = 0; k < U; k++) {
      const int l = l0 + 256 * k;
      if (l >= l_hi) break;
      float sv[4];
      sv[0] = pe[k][7];
      sv[1] = sv[0] + pe[k][3];
      sv[2] = sv[1] + pe[k][1] + pe[k][5];
      sv[3] = sv[2] + pe[k][0] + pe[k][2] + pe[k][4] + pe[k][6];
      if (STORE) {
        orow[l] = sv[hp.out_stage];
      } else {
#pragma unroll
        for (int q = 0; q < 4; q++)
          if (sv[q] > best[q]) {        // l increases per thread: strict > keeps the smallest j among equals
            best[q] = sv[q];
            bj[q] = l;
          }
      }
    }
  }
  if (STORE) return;
  __shared__ float s_best[4][8];
  __shared__ int s_bj[4][8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int q = 0; q < 4; q++) {
    float b = best[q];
    int jj = bj[q];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
      const float ob = __shfl_xor_sync(0xffffffffu, b, o);
      const int oj = __shfl_xor_sync(0xffffffffu, jj, o);
      if (oj >= 0 && (jj < 0 || ob > b || (ob == b && oj < jj))) {
        b = ob;
        jj = oj;
      }
    }
    if (lane == 0) {
      s_best[q][warp] = b;
      s_bj[q][warp] = jj;
    }
  }
  __syncthreads();
  if (threadIdx.x < 4) {
    const int q = threadIdx.x;
    float b = s_best[q][0];
    int jj = s_bj[q][0];
    for (int w = 1; w < 8; w++) {
      const float ob = s_best[q][w];
      const int oj = s_bj[q][w];
      if (oj >= 0 && (jj < 0 || ob > b || (ob == b && oj < jj))) {
        b = ob;
        jj = oj;
      }
    }
    jerk_cand c;
    c.j = jj < 0 ? -1 : (int)(j8 + jj);
    c.iz = (int16_t)iz;
    c.iw = (int16_t)iw;
    c.power = b;
    c.flags = 0;
    hp.blockbest[(size_t)q * gridDim.x + blockIdx.x] = c;
  }
}

// Arg-max fold of per-stage candidate lists: block b of the grid reduces in[q][b, b + gridDim.x, ...] (q = 0..3, n_in
// records per stage).  A multi-block launch writes its partial results to out[q][blockIdx.x]; the final single-block
// launch (running != nullptr) merges its result into running[q] (`first`: overwrite).
__global__ void __launch_bounds__(256) k_harm_fold(const jerk_cand* in, int n_in, jerk_cand* out, jerk_cand* running, int first) {
  __shared__ jerk_cand s_c[256];
  for (int q = 0; q < 4; q++) {
    jerk_cand b;
    b.j = -1;
    b.iz = b.iw = 0;
    b.power = -INFINITY;
    b.flags = 0;
    for (int i = blockIdx.x * 256 + threadIdx.x; i < n_in; i += 256 * gridDim.x) {
      const jerk_cand c = in[(size_t)q * n_in + i];
      if (c.j >= 0 && (b.j < 0 || harm_better(c.power, c.j, c.iz, c.iw, b.power, b.j, b.iz, b.iw))) b = c;
    }
    s_c[threadIdx.x] = b;
    __syncthreads();
    for (int o = 128; o > 0; o >>= 1) {
      if (threadIdx.x < o) {
        const jerk_cand c = s_c[threadIdx.x + o], m = s_c[threadIdx.x];
        if (c.j >= 0 && (m.j < 0 || harm_better(c.power, c.j, c.iz, c.iw, m.power, m.j, m.iz, m.iw))) s_c[threadIdx.x] = c;
      }
      __syncthreads();
    }
    if (threadIdx.x == 0) {
      const jerk_cand c = s_c[0];
      if (running) {
        const jerk_cand m = running[q];
        if (first || (c.j >= 0 && (m.j < 0 || harm_better(c.power, c.j, c.iz, c.iw, m.power, m.j, m.iz, m.iw)))) running[q] = c;
      } else {
        out[(size_t)q * gridDim.x + blockIdx.x] = c;
      }
    }
    __syncthreads();
  }
}

// d_top[s] = running[log2 h_s] if its sum exceeds the stage threshold, else {j = -1, power = 0}
struct HarmEmit {
  int nstages;
  int stage[4];
  float thr[4];
};
__global__ void k_harm_emit(const jerk_cand* running, jerk_cand* top, HarmEmit he) {
  const int s = threadIdx.x;
  if (s >= he.nstages) return;
  jerk_cand c = running[he.stage[s]];
  if (!(c.j >= 0 && c.power > he.thr[s])) {
    c.j = -1;
    c.iz = c.iw = 0;
    c.power = 0.f;
  }
  c.flags = 0;
  top[s] = c;
}

// ------------------------------------------------------------------------------------------------- host helpers
template <int L, int MODE>
static size_t search_smem_bytes() {
  return (size_t)(FftGeom<L>::EX1 + FftGeom<L>::EX2 + Tw2Table<L>::FLOATS2) * sizeof(float2) + 2 * sizeof(unsigned long long);
}

template <int L, int MODE>
static cudaError_t launch_search(const jerk_plan* plan, const SearchParams& sp, cudaStream_t st) {
  using Gm = FftGeom<L>;
  size_t smem = search_smem_bytes<L, MODE>();
  cudaError_t e = cudaFuncSetAttribute(k_search<L, MODE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  // Resident CTAs per SM.  cudaOccupancyMaxActiveBlocksPerMultiprocessor answers 1 for every kernel that allocates
  // tensor memory, although CTAs do co-reside as long as their TMEM columns fit (512 per SM): compute it from the
  // kernel's own resource use.
  cudaFuncAttributes fa;
  e = cudaFuncGetAttributes(&fa, k_search<L, MODE>);
  if (e != cudaSuccess) return e;
  int regs_per_cta = ((fa.numRegs + 7) / 8 * 8) * Gm::NT;
  int occ = 65536 / regs_per_cta;
  occ = std::min(occ, (int)(233472 / (smem + fa.sharedSizeBytes + 1024)));
  occ = std::min(occ, 2048 / Gm::NT);
  occ = std::min(occ, 512 / TmemCols<L>::value);
  if (occ < 1) occ = 1;
  long long nitems = sp.nitems;
  long long grid = (long long)plan->sm_count * occ;
  const long long slots = (long long)(plan->stash_bytes / (2ull * L * sizeof(float)));   // one stash slot per CTA
  if (grid > slots) grid = slots;
  if (grid > nitems) grid = nitems;
  if (grid < 1) grid = 1;
  k_search<L, MODE><<<(unsigned)grid, Gm::NT, smem, st>>>(sp);
  return cudaGetLastError();
}

// FFT groups per CTA of k_search64: two (two CTAs per SM, 256 TMEM columns each) in the candidate modes, four (one CTA
// per SM, all 512 columns: the phase-0 stash) in the plane and harmonic modes: 8 warps per SM either way, up to 255
// registers.  Six groups (12 warps, 168 registers: the register file is 16 K per scheduler, i.e. 170 registers at three
// warps each) measured 172 ms/search against 158 ms: the spills and the tighter schedule cost more than the third warp
// per scheduler hides.
template <int MODE>
struct K64 {
  static constexpr int NG = (MODE == MODE_CAND || MODE == MODE_CAND_STATS) ? 2 : 4;
  static constexpr int CTAS_PER_SM = NG == 2 ? 2 : 1;
  static constexpr size_t SMEM = (size_t)NG * kEx64 * sizeof(float2) + 4 * NG * sizeof(unsigned long long) +
                                 ((MODE == MODE_HARM || MODE == MODE_HARM_STORE) ? (size_t)NG * (64 + 16) * 64 * sizeof(float) : 0);   // + phase-1 powers, per-k maxima
};

// CTAs of a k_search64 launch: every SM full, never more FFT groups than stash slots or work items
template <int MODE>
static unsigned search64_grid(const jerk_plan* plan, long long nitems) {
  constexpr int NG = K64<MODE>::NG;
  long long grid = (long long)plan->sm_count * K64<MODE>::CTAS_PER_SM;
  const long long slots = (long long)(plan->stash_bytes / (2ull * 4096 * sizeof(float)));   // stash slots of one FFT group
  if (grid * NG > slots) grid = slots / NG;
  if (grid > (nitems + NG - 1) / NG) grid = (nitems + NG - 1) / NG;
  if (grid < 1) grid = 1;
  return (unsigned)grid;
}

template <int MODE, bool PRUNE>
static cudaError_t launch_search64p(const jerk_plan* plan, const SearchParams& sp, cudaStream_t st) {
  constexpr int NG = K64<MODE>::NG;
  cudaError_t e = cudaFuncSetAttribute(k_search64<MODE, NG, PRUNE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)K64<MODE>::SMEM);
  if (e != cudaSuccess) return e;
  k_search64<MODE, NG, PRUNE><<<search64_grid<MODE>(plan, sp.nitems), 64 * NG, K64<MODE>::SMEM, st>>>(sp);
  return cudaGetLastError();
}

template <int MODE>
static cudaError_t launch_search64(const jerk_plan* plan, const SearchParams& sp, cudaStream_t st) {
  bool prune = true;   // outputs n < 256 and n >= 3840 are outside the valid window of every job of the launch
  for (int q = 0; q < sp.njobs; q++) prune = prune && sp.jobs[q].hw >= 256;
  return prune ? launch_search64p<MODE, true>(plan, sp, st) : launch_search64p<MODE, false>(plan, sp, st);
}

template <int MODE>
static cudaError_t dispatch_search(const jerk_plan* plan, const SearchParams& sp, cudaStream_t st) {
  switch (plan->L) {
    case 1024: return launch_search<1024, MODE>(plan, sp, st);
    case 2048: return launch_search<2048, MODE>(plan, sp, st);
    case 4096: return launch_search64<MODE>(plan, sp, st);
    case 8192: return launch_search<8192, MODE>(plan, sp, st);
  }
  return cudaErrorInvalidValue;
}

template <int L>
static cudaError_t launch_bank(const jerk_plan* plan, const BankParams& bp, int ti_cnt, cudaStream_t st) {
  using Gm = FftGeom<L>;
  size_t smem = (size_t)(Gm::EX1 + Gm::EX2 + Tw2Table<L>::FLOATS2 + 4 * plan->hw_max + 1) * sizeof(float2);
  cudaError_t e = cudaFuncSetAttribute(k_bank<L>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
  if (e != cudaSuccess) return e;
  k_bank<L><<<ti_cnt, Gm::NT, smem, st>>>(bp);
  return cudaGetLastError();
}

static bool is_integer(double v) { return fabs(v - round(v)) < 1e-9; }

static uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

static void fill_params(const jerk_plan* plan, SearchParams& sp, const void* d_spec, void* d_work, uint64_t work_bytes) {
  memset(&sp, 0, sizeof(sp));
  sp.spec[0] = (const float2*)d_spec;
  sp.nbins = plan->nbins;
  sp.geom = (const TemplateGeom*)plan->d_bank;
  // template ti's filters are at G + ti * nb * L: for a partial bank (jerk_templates_range) the base is moved back by the
  // templates that are not there (never dereferenced outside the range: bank_covers is checked by every entry point)
  sp.G = (const float2*)((const unsigned char*)plan->d_bank + plan->geom_bytes) - (ptrdiff_t)plan->bank_ti_lo * plan->numbetween * plan->L;
  sp.nz = plan->nz;
  sp.nw_grid = plan->nw;
  sp.nspec = 1;
  sp.nb = plan->numbetween;
  sp.hw_max = plan->hw_max;
  sp.step = plan->step;
  sp.seg_base = plan->seg_base;
  sp.work = (unsigned long long*)d_work;
  sp.stash = (float*)((unsigned char*)d_work + kWorkHeader + plan->order_bytes);
  sp.seams = (jerk_cand*)((unsigned char*)d_work + kWorkHeader + plan->order_bytes + plan->stash_bytes);
  sp.seam_cap = std::min<uint64_t>((work_bytes - kWorkHeader - plan->order_bytes - plan->stash_bytes) / sizeof(jerk_cand), kSeamHashMaxSlots / 2);
}

// k_reset, the candidate-mode search launch `search`, then the seam kernels
template <class F>
static int run_candidate_search(jerk_plan* p, const SearchParams& sp, const OrderParams& op, cudaStream_t st, const char* what, F search) {
  k_reset<<<1, 32, 0, st>>>(sp.work, sp.count, sp.nspec);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_reset launch: ") + cudaGetErrorString(e));
  if (sp.nitems == 0) return JERK_OK;   // empty box
  if (op.total) {
    k_order<<<1, 1024, 0, st>>>(op);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_order launch: ") + cudaGetErrorString(e));
  }
  e = search();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string(what) + " launch: " + cudaGetErrorString(e));
  const int blocks = p->sm_count * 2;
  k_seam_clear<<<blocks, 256, 0, st>>>(sp);
  k_seam_insert<<<blocks, 256, 0, st>>>(sp);
  k_seam_resolve<<<blocks, 256, 0, st>>>(sp);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("seam kernels launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

// true iff every template of the box is in the bank the plan holds
static bool bank_covers(const jerk_plan* p, int iz_lo, int iz_cnt, int iw_lo, int iw_cnt) {
  if (iz_cnt <= 0 || iw_cnt <= 0) return true;
  const int first = iw_lo * p->nz + iz_lo, last = (iw_lo + iw_cnt - 1) * p->nz + iz_lo + iz_cnt - 1;
  return first >= p->bank_ti_lo && last < p->bank_ti_lo + p->bank_ti_cnt;
}

// segments whose outputs b = s0 + n - c (n in [hw_max, hw_max+step), |c| <= c_max) can touch bins [r_lo, r_lo+r_cnt)
static void job_segments(const jerk_plan* p, int64_t r_lo, int64_t r_cnt, int64_t* first, int64_t* count) {
  int64_t lo = r_lo - p->c_max - p->seg_base - p->hw_max - p->step + 1;  // s*step >= lo
  int64_t hi = r_lo + r_cnt - 1 + p->c_max - p->seg_base - p->hw_max;    // s*step <= hi
  int64_t s_first = lo <= 0 ? 0 : (lo + p->step - 1) / p->step;
  int64_t s_last = hi < 0 ? -1 : hi / p->step;
  if (s_last > p->nseg - 1) s_last = p->nseg - 1;
  *first = s_first;
  *count = s_last < s_first ? 0 : s_last - s_first + 1;
}

// Appends the box (r, iz, iw) as a job of `sp` (sp.nb and sp.nspec must be set).  Returns false when the box is empty (nothing appended).
// Segments whose outputs b = s0 + n - c (n in [hw_max, hw_max+step), |c| <= c_max) can touch [r_lo, r_lo+r_cnt) are selected.
static bool add_job(const jerk_plan* p, SearchParams& sp, int64_t r_lo, int64_t r_cnt, int iz_lo, int iz_cnt, int iw_lo,
                    int iw_cnt, float* plane, int chunk_tp) {
  if (r_cnt <= 0 || iz_cnt <= 0 || iw_cnt <= 0 || sp.njobs >= kMaxJobs) return false;
  int64_t s_first, s_count;
  job_segments(p, r_lo, r_cnt, &s_first, &s_count);
  if (s_count == 0) return false;
  SearchJob& jb = sp.jobs[sp.njobs];
  jb.seg_first = s_first;
  jb.seg_count = s_count;
  jb.r_lo = r_lo;
  jb.r_cnt = r_cnt;
  jb.iz_lo = iz_lo;
  jb.iz_cnt = iz_cnt;
  jb.iw_lo = iw_lo;
  jb.iw_cnt = iw_cnt;
  jb.ntp = sp.nb * iz_cnt * iw_cnt;
  jb.chunk_tp = chunk_tp;
  jb.plane = plane;
  jb.bmax = nullptr;
  jb.hw = p->hw_max;
  jb.step = p->step;
  jb.seg_base = p->seg_base;
  jb.order = nullptr;
  long long nchunks = (jb.ntp + chunk_tp - 1) / chunk_tp;
  sp.nitems += nchunks * jb.seg_count * sp.nspec;
  jb.item_end = sp.nitems;
  sp.njobs++;
  return true;
}

// template-phases per work item: kChunkTP when the box is large; smaller (even, >= 16) when the box alone could not
// give every resident CTA a few items
static int pick_chunk_tp(const jerk_plan* p, int64_t r_cnt, int iz_cnt, int iw_cnt) {
  long long ntp = (long long)p->numbetween * iz_cnt * iw_cnt;   // template-phases
  long long segs = r_cnt / p->step + 2;
  long long want_items = 32LL * 4 * (p->sm_count > 0 ? p->sm_count : 148);   // >= 32 rounds of work items per resident FFT group: tail < 3 %
  int c = kChunkTP;
  while (c > 32 && ((ntp + c - 1) / c) * segs < want_items) c >>= 1;
  return c;
}

struct TemplateBox {
  int iz_lo, iz_cnt, iw_lo, iw_cnt;
};

// Jobs of a candidate search over the templates of `boxes` (at most three, disjoint).  The overlap of an overlap-save
// segment only has to cover the half-width of the templates it is correlated with (y[n] is exact for
// n in [hw, L - hw)), so the plan splits the grid's templates into up to kMaxJobs classes of similar half-width
// (plan_classes) and every class is searched on its own segmentation: step = L - 2 hw_class instead of L - 2 hw_max.  On
// the zmax 200 / wmax 600 grid (hw from 8 to 258, 134 on average) that is 6 % fewer (segment, template) units for the
// same points.  The candidate rule is one-dimensional along r inside a (z,w) row, and a row belongs to exactly one
// class -- the same one in every call, whatever the box -- so results do not depend on how the grid is cut into boxes.
// Small grids (fewer than 1024 templates) form one class and keep the plain box job.  Returns the k_order parameters in
// `op` (op.total = 0: no list needed).
static void add_class_jobs(const jerk_plan* p, SearchParams& sp, const TemplateBox* boxes, int nboxes, void* d_work, OrderParams& op,
                           int64_t r_lo = 0, int64_t r_cnt = -1) {      // bins [r_lo, r_lo + r_cnt) (default: the whole spectrum)
  memset(&op, 0, sizeof(op));
  if (r_cnt < 0) r_cnt = p->nbins;
  if (p->ncls < 2) {
    for (int b = 0; b < nboxes; b++)
      add_job(p, sp, r_lo, r_cnt, boxes[b].iz_lo, boxes[b].iz_cnt, boxes[b].iw_lo, boxes[b].iw_cnt, nullptr,
              r_cnt == p->nbins ? kChunkTP : pick_chunk_tp(p, r_cnt, boxes[b].iz_cnt, boxes[b].iw_cnt));
    return;
  }
  long long total = 0;
  int cnt[kMaxJobs] = {0};
  for (int b = 0; b < nboxes; b++) {
    total += (long long)boxes[b].iz_cnt * boxes[b].iw_cnt;
    for (int iw = boxes[b].iw_lo; iw < boxes[b].iw_lo + boxes[b].iw_cnt; iw++)
      for (int iz = boxes[b].iz_lo; iz < boxes[b].iz_lo + boxes[b].iz_cnt; iz++)
        cnt[(p->geom[(size_t)iw * p->nz + iz].hw - p->cls_lo) / p->cls_width]++;
  }
  if (total == 0) return;
  op.nboxes = nboxes;
  for (int b = 0; b < nboxes; b++) {
    op.iz_lo[b] = boxes[b].iz_lo;
    op.iz_cnt[b] = boxes[b].iz_cnt;
    op.iw_lo[b] = boxes[b].iw_lo;
    op.iw_cnt[b] = boxes[b].iw_cnt;
  }
  op.total = (int)total;
  op.hw_lo = p->cls_lo;
  op.width = p->cls_width;
  op.geom = (const TemplateGeom*)p->d_bank;
  op.nz = p->nz;
  op.out = (int*)((unsigned char*)d_work + kWorkHeader);
  int off = 0;
  for (int k = 0; k < p->ncls; k++) {
    op.cls_off[k] = off;
    const int n = cnt[k];
    if (n == 0) continue;
    const int hw = p->cls_hw[k];
    SearchJob& jb = sp.jobs[sp.njobs];
    memset(&jb, 0, sizeof(jb));
    jb.hw = hw;
    jb.step = p->L - 2 * hw;
    int64_t base = -((int64_t)p->c_max + hw);      // as in jerk_plan_create, with the class's half-width
    if (base & 1) base -= 1;
    jb.seg_base = base;
    {   // segments whose outputs b = s0 + n - c (n in [hw, hw + step), |c| <= c_max) can touch the bins of the call
      const int64_t nseg = (p->nbins + p->c_max - hw - base + jb.step - 1) / jb.step;
      const int64_t lo = r_lo - p->c_max - base - hw - jb.step + 1, hi = r_lo + r_cnt - 1 + p->c_max - base - hw;
      const int64_t s_first = lo <= 0 ? 0 : (lo + jb.step - 1) / jb.step;
      const int64_t s_last = std::min<int64_t>(hi < 0 ? -1 : hi / jb.step, nseg - 1);
      if (s_last < s_first) continue;
      jb.seg_first = s_first;
      jb.seg_count = s_last - s_first + 1;
    }
    jb.r_lo = r_lo;
    jb.r_cnt = r_cnt;
    jb.iz_cnt = n;                                 // (a one-row box of n templates: the kernels' box arithmetic stays defined)
    jb.iw_cnt = 1;
    jb.ntp = sp.nb * n;
    jb.chunk_tp = kChunkTP;
    jb.order = op.out + off;
    sp.nitems += (long long)((jb.ntp + jb.chunk_tp - 1) / jb.chunk_tp) * jb.seg_count * sp.nspec;
    jb.item_end = sp.nitems;
    sp.njobs++;
    off += n;
  }
  // a short r-range: shrink the work items until every resident FFT group gets a few
  const long long want_items = 32LL * 4 * (p->sm_count > 0 ? p->sm_count : 148);
  while (sp.nitems < want_items && sp.njobs && sp.jobs[0].chunk_tp > 32) {
    sp.nitems = 0;
    for (int q = 0; q < sp.njobs; q++) {
      SearchJob& jb = sp.jobs[q];
      jb.chunk_tp >>= 1;
      sp.nitems += (long long)((jb.ntp + jb.chunk_tp - 1) / jb.chunk_tp) * jb.seg_count * sp.nspec;
      jb.item_end = sp.nitems;
    }
  }
}

// the plan's overlap classes: equal-width bins of the half-width, at least 512 templates per class on average
static void plan_classes(jerk_plan* p) {
  static_assert(kMaxJobs == 16, "jerk_plan::cls_hw holds one entry per job of a launch");
  int hw_lo = p->hw_max, hw_hi = 0;
  for (const TemplateGeom& g : p->geom) {
    hw_lo = std::min(hw_lo, g.hw);
    hw_hi = std::max(hw_hi, g.hw);
  }
  int ncls = std::min(std::min(kMaxJobs, p->T / 512), hw_hi - hw_lo + 1);
  if (ncls < 2) ncls = 1;
  p->ncls = ncls;
  p->cls_lo = hw_lo;
  p->cls_width = (hw_hi - hw_lo + ncls) / ncls;   // ceil((hw_hi - hw_lo + 1) / ncls)
  for (int k = 0; k < 16; k++) p->cls_hw[k] = 0;
  for (const TemplateGeom& g : p->geom) {
    int& h = p->cls_hw[(g.hw - hw_lo) / p->cls_width];
    h = std::max(h, g.hw);
  }
}

}  // namespace jerk

using namespace jerk;

// ------------------------------------------------------------------------------------------------- C ABI
extern "C" {

const char* jerk_strerror(int status) {
  switch (status) {
    case JERK_OK: return "JERK_OK";
    case JERK_EINVAL: return "JERK_EINVAL: invalid argument";
    case JERK_ENOMEM: return "JERK_ENOMEM: caller buffer too small";
    case JERK_ECUDA: return "JERK_ECUDA: CUDA error";
    case JERK_ESTATE: return "JERK_ESTATE: template bank not built";
    case JERK_ENODEV: return "JERK_ENODEV: no sm_100 device";
    case JERK_EOVERFLOW: return "JERK_EOVERFLOW: more candidates or seam records than the caller's buffers hold";
    case JERK_ELIMIT: return "JERK_ELIMIT: request exceeds a fixed built-in capacity (jerk_prepare_spectrum_static: at most 2^21 samples; use jerk_prepare_spectrum with caller scratch)";
  }
  return "unknown jerk status";
}

const char* jerk_last_error(const jerk_plan* plan) { return plan ? plan->err.c_str() : "null plan"; }

int jerk_plan_create(jerk_plan** out, int64_t nbins, double zmax, double dz, double wmax, double dw, int numbetween,
                     int seg_len) {
  if (!out) return JERK_EINVAL;
  *out = nullptr;
  if (nbins < 1 || zmax < 0 || wmax < 0 || !(dz > 0) || !(dw > 0)) return JERK_EINVAL;
  if (!is_integer(zmax / dz) || !is_integer(wmax / dw)) return JERK_EINVAL;
  if (numbetween != 1 && numbetween != 2) return JERK_EINVAL;
  if (seg_len != 0 && seg_len != 1024 && seg_len != 2048 && seg_len != 4096 && seg_len != 8192) return JERK_EINVAL;
  if (nbins > (int64_t)1 << 30) return JERK_EINVAL;  // j = 2b+p is reported as int32
  jerk_plan* p = new jerk_plan();
  p->nbins = nbins;
  p->zmax = zmax;
  p->dz = dz;
  p->wmax = wmax;
  p->dw = dw;
  p->numbetween = numbetween;
  p->L = seg_len;
  p->nz = (int)llround(2.0 * zmax / dz) + 1;
  p->nw = (int)llround(2.0 * wmax / dw) + 1;
  if (p->nz >= 32768 || p->nw >= 32768 || (int64_t)p->nz * p->nw > (1 << 24)) {
    delete p;
    return JERK_EINVAL;
  }
  p->T = p->nz * p->nw;
  p->geom.resize(p->T);
  p->hw_max = 0;
  p->c_max = 0;
  for (int iw = 0; iw < p->nw; iw++)
    for (int iz = 0; iz < p->nz; iz++) {
      TemplateGeom g = template_geom(-zmax + iz * dz, -wmax + iw * dw);
      p->geom[(size_t)iw * p->nz + iz] = g;
      if (g.hw > p->hw_max) p->hw_max = g.hw;
      if (abs(g.c) > p->c_max) p->c_max = abs(g.c);
    }
  // seg_len 0: the library's choice.  The result does not depend on the segment length (SURVEY.md 8(c) pin P9); 4096 is
  // the length of the two-pass kernel (k_search64) and is taken whenever the templates leave a positive step.
  if (seg_len == 0) {
    seg_len = 4096 - 2 * p->hw_max >= 2 ? 4096 : 8192;
    // a tiny search (config 1: 147 templates x 10 segments) cannot fill the 592 resident FFT groups of the two-pass
    // kernel even with the smallest work items (32 template-phases); the 1024-point kernel has four times the segments
    const int64_t items4096 = ((int64_t)numbetween * p->T + 31) / 32 * (nbins / (4096 - 2 * p->hw_max) + 2);
    if (seg_len == 4096 && items4096 < 2 * 592 && 1024 - 2 * p->hw_max >= 512) seg_len = 1024;
  }
  p->L = seg_len;
  p->step = seg_len - 2 * p->hw_max;
  if (p->step < 2) {
    delete p;
    return JERK_EINVAL;
  }
  // first segment: s0 <= -(c_max + hw_max), even (16-byte aligned bulk copies); output b = s0 + n - c, n in [hw_max, hw_max+step)
  int64_t base = -((int64_t)p->c_max + p->hw_max);
  if (base & 1) base -= 1;
  p->seg_base = base;
  // last segment must reach b = nbins-1 for c = +c_max:  base + (nseg-1)*step + hw_max + step - 1 - c_max >= nbins - 1
  int64_t need = nbins + p->c_max - p->hw_max - base;
  p->nseg = (need + p->step - 1) / p->step;
  p->geom_bytes = align_up((uint64_t)p->T * sizeof(TemplateGeom), kBankAlign);
  p->bank_bytes = p->geom_bytes + (uint64_t)p->T * numbetween * seg_len * sizeof(float2);
  plan_classes(p);
  p->stash_bytes = kStashBytes;
  p->order_bytes = align_up((uint64_t)p->T * sizeof(int), 256);
  p->work_bytes = kWorkHeader + p->order_bytes + p->stash_bytes + kSeamCapDefault * sizeof(jerk_cand);
  p->d_bank = nullptr;
  p->bank_ti_lo = p->bank_ti_cnt = 0;
  p->sm_count = 0;
  *out = p;
  return JERK_OK;
}

int jerk_plan_destroy(jerk_plan* plan) {
  delete plan;
  return JERK_OK;
}

int jerk_plan_info(const jerk_plan* p, jerk_plan_info_t* info) {
  if (!p || !info) return JERK_EINVAL;
  memset(info, 0, sizeof(*info));
  info->nbins = p->nbins;
  info->zmax = p->zmax;
  info->dz = p->dz;
  info->wmax = p->wmax;
  info->dw = p->dw;
  info->numbetween = p->numbetween;
  info->seg_len = p->L;
  info->nz = p->nz;
  info->nw = p->nw;
  info->ntemplates = p->T;
  info->hw_max = p->hw_max;
  info->c_max = p->c_max;
  info->step = p->step;
  info->seg_base = p->seg_base;
  info->nseg = p->nseg;
  info->points = (int64_t)p->numbetween * p->nbins * p->T;
  info->bank_bytes = p->bank_bytes;
  info->work_bytes = p->work_bytes;
  // nominal segments ceil(nbins/step), 2T template-phases, 5 L log2 L + 6 L + 3 step flops each
  double nseg_nom = ceil((double)p->nbins / (double)p->step);
  double l2 = log2((double)p->L);
  info->flops_per_search = nseg_nom * (double)p->numbetween * p->T * (5.0 * p->L * l2 + 6.0 * p->L + 3.0 * p->step);
  // what a whole-grid candidate search executes: every overlap class on its own segmentation
  info->nclasses = p->ncls;
  if (p->ncls < 2) {
    info->units_per_search = p->nseg * (int64_t)p->numbetween * p->T;
    info->flops_per_search_executed = (double)info->units_per_search * (5.0 * p->L * l2 + 6.0 * p->L + 3.0 * p->step);
  } else {
    std::vector<int64_t> cnt(p->ncls, 0);
    for (const TemplateGeom& g : p->geom) cnt[(g.hw - p->cls_lo) / p->cls_width]++;
    for (int k = 0; k < p->ncls; k++) {
      if (!cnt[k]) continue;
      const int hw = p->cls_hw[k], step = p->L - 2 * hw;
      int64_t base = -((int64_t)p->c_max + hw);
      if (base & 1) base -= 1;
      const int64_t nseg = (p->nbins + p->c_max - hw - base + step - 1) / step;
      const int64_t units = nseg * p->numbetween * cnt[k];
      info->units_per_search += units;
      info->flops_per_search_executed += (double)units * (5.0 * p->L * l2 + 6.0 * p->L + 3.0 * step);
    }
  }
  return JERK_OK;
}

int jerk_template_units(const jerk_plan* p, int64_t* h_units, int n) {
  if (!p || !h_units || n != p->T) return JERK_EINVAL;
  if (p->ncls < 2) {
    for (int ti = 0; ti < p->T; ti++) h_units[ti] = p->nseg * (int64_t)p->numbetween;
    return JERK_OK;
  }
  std::vector<int64_t> nseg_cls(p->ncls, 0);
  for (int k = 0; k < p->ncls; k++) {      // the segmentation of class k, as in jerk_plan_info / add_class_jobs
    const int hw = p->cls_hw[k], step = p->L - 2 * hw;
    int64_t base = -((int64_t)p->c_max + hw);
    if (base & 1) base -= 1;
    nseg_cls[k] = (p->nbins + p->c_max - hw - base + step - 1) / step;
  }
  for (int ti = 0; ti < p->T; ti++) h_units[ti] = nseg_cls[(p->geom[ti].hw - p->cls_lo) / p->cls_width] * (int64_t)p->numbetween;
  return JERK_OK;
}

int jerk_template_geometry(const jerk_plan* p, int iz, int iw, int* c, int* hw) {
  if (!p || iz < 0 || iz >= p->nz || iw < 0 || iw >= p->nw) return JERK_EINVAL;
  const TemplateGeom& g = p->geom[(size_t)iw * p->nz + iz];
  if (c) *c = g.c;
  if (hw) *hw = g.hw;
  return JERK_OK;
}

uint64_t jerk_plane_bytes(int64_t r_cnt, int iz_cnt, int iw_cnt) {
  if (r_cnt < 0 || iz_cnt < 0 || iw_cnt < 0) return 0;
  return (uint64_t)iw_cnt * (uint64_t)iz_cnt * (uint64_t)(2 * r_cnt) * sizeof(float);
}

static int ensure_device(jerk_plan* p) {
  if (p->sm_count > 0) return JERK_OK;
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return fail(p, JERK_ENODEV, "cudaGetDevice failed: no CUDA device");
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return fail(p, JERK_ENODEV, "cudaGetDeviceProperties failed");
  if (prop.major != 10) return fail(p, JERK_ENODEV, "device is not sm_100 (B200): this library has no other code path");
  p->sm_count = prop.multiProcessorCount;
  return JERK_OK;
}

uint64_t jerk_bank_bytes_range(const jerk_plan* p, int ti_cnt) {
  if (!p || ti_cnt < 0 || ti_cnt > p->T) return 0;
  return p->geom_bytes + (uint64_t)ti_cnt * p->numbetween * p->L * sizeof(float2);
}

int jerk_templates_range(jerk_plan* p, int ti_lo, int ti_cnt, void* d_bank, uint64_t bank_bytes, void* stream) {
  if (!p || !d_bank) return JERK_EINVAL;
  // ti_cnt == 0 (a rank of a sharded search that is left without templates: more ranks than templates) is legal: the
  // geometry tables are copied, no filter is built, and only empty ranges can be searched afterwards
  if (ti_lo < 0 || ti_cnt < 0 || ti_lo > p->T - ti_cnt) return fail(p, JERK_EINVAL, "template range outside [0, ntemplates)");
  if (bank_bytes < jerk_bank_bytes_range(p, ti_cnt)) return fail(p, JERK_ENOMEM, "bank buffer smaller than jerk_bank_bytes_range");
  if ((uintptr_t)d_bank % kBankAlign) return fail(p, JERK_EINVAL, "d_bank must be 256-byte aligned");
  int rc = ensure_device(p);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpyAsync(d_bank, p->geom.data(), (size_t)p->T * sizeof(TemplateGeom), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("geom copy: ") + cudaGetErrorString(e));
  BankParams bp;
  bp.zmax = p->zmax;
  bp.dz = p->dz;
  bp.wmax = p->wmax;
  bp.dw = p->dw;
  bp.nz = p->nz;
  bp.nw = p->nw;
  bp.nb = p->numbetween;
  bp.ti_lo = ti_lo;
  bp.geom = (const TemplateGeom*)d_bank;
  bp.G = (float2*)((unsigned char*)d_bank + p->geom_bytes);
  switch (ti_cnt ? p->L : 0) {
    case 0: break;
    case 1024: e = launch_bank<1024>(p, bp, ti_cnt, st); break;
    case 2048: e = launch_bank<2048>(p, bp, ti_cnt, st); break;
    case 4096: e = launch_bank<4096>(p, bp, ti_cnt, st); break;
    default: e = launch_bank<8192>(p, bp, ti_cnt, st); break;
  }
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_bank launch: ") + cudaGetErrorString(e));
  p->d_bank = d_bank;
  p->bank_ti_lo = ti_lo;
  p->bank_ti_cnt = ti_cnt;
  return JERK_OK;
}

int jerk_templates(jerk_plan* p, void* d_bank, uint64_t bank_bytes, void* stream) {
  if (!p) return JERK_EINVAL;
  return jerk_templates_range(p, 0, p->T, d_bank, bank_bytes, stream);
}

int jerk_templates_taps(jerk_plan* p, int iz, int iw, void* d_taps, uint64_t taps_bytes, void* stream) {
  if (!p || !d_taps || iz < 0 || iz >= p->nz || iw < 0 || iw >= p->nw) return JERK_EINVAL;
  int rc = ensure_device(p);
  if (rc) return rc;
  const TemplateGeom& g = p->geom[(size_t)iw * p->nz + iz];
  if (taps_bytes < (uint64_t)(4 * g.hw + 1) * sizeof(float2)) return fail(p, JERK_ENOMEM, "taps buffer too small");
  k_taps<<<8, 128, 0, (cudaStream_t)stream>>>(-p->zmax + iz * p->dz, -p->wmax + iw * p->dw, g.c, g.hw, (float2*)d_taps);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_taps launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

static int check_common(jerk_plan* p, const void* d_spec, void* d_work, uint64_t work_bytes) {
  if (!p || !d_spec || !d_work) return JERK_EINVAL;
  if (!p->d_bank) return fail(p, JERK_ESTATE, "jerk_templates has not been called");
  if (work_bytes < p->work_bytes) return fail(p, JERK_ENOMEM, "work buffer smaller than plan work_bytes");
  if ((uintptr_t)d_spec % 16) return fail(p, JERK_EINVAL, "d_spec must be 16-byte aligned");
  if ((uintptr_t)d_work % 256) return fail(p, JERK_EINVAL, "d_work must be 256-byte aligned");
  return ensure_device(p);
}

int jerk_search_plane(jerk_plan* p, const void* d_spec, int64_t r_lo, int64_t r_cnt, int iz_lo, int iz_cnt, int iw_lo,
                      int iw_cnt, float* d_plane, uint64_t plane_bytes, void* d_work, uint64_t work_bytes, void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (r_lo < 0 || r_cnt < 0 || r_lo + r_cnt > p->nbins || iz_lo < 0 || iz_cnt < 0 || iz_lo + iz_cnt > p->nz || iw_lo < 0 ||
      iw_cnt < 0 || iw_lo + iw_cnt > p->nw)
    return fail(p, JERK_EINVAL, "plane sub-range outside the plan's grid");
  if (plane_bytes < jerk_plane_bytes(r_cnt, iz_cnt, iw_cnt) / 2 * p->numbetween) return fail(p, JERK_ENOMEM, "plane buffer too small");
  if (r_cnt == 0 || iz_cnt == 0 || iw_cnt == 0) return JERK_OK;  // empty range: nothing to write, d_plane may be NULL
  if (!d_plane) return JERK_EINVAL;
  if ((uintptr_t)d_plane % 8) return fail(p, JERK_EINVAL, "d_plane must be 8-byte aligned");
  if (!bank_covers(p, iz_lo, iz_cnt, iw_lo, iw_cnt)) return fail(p, JERK_ESTATE, "the template box is not inside the range jerk_templates_range built");
  cudaStream_t st = (cudaStream_t)stream;
  SearchParams sp;
  fill_params(p, sp, d_spec, d_work, work_bytes);
  if (!add_job(p, sp, r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt, d_plane, pick_chunk_tp(p, r_cnt, iz_cnt, iw_cnt))) return JERK_OK;
  k_reset<<<1, 32, 0, st>>>(sp.work, nullptr, 0);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_reset launch: ") + cudaGetErrorString(e));
  e = dispatch_search<MODE_PLANE>(p, sp, st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_search(plane) launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

int jerk_search_candidates_range(jerk_plan* p, const void* d_spec, float threshold, int iz_lo, int iz_cnt, int iw_lo, int iw_cnt,
                                 jerk_cand* d_cands, int64_t max_cands, unsigned long long* d_count, void* d_work,
                                 uint64_t work_bytes, void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (!d_cands || !d_count || max_cands < 0) return JERK_EINVAL;
  if (iz_lo < 0 || iz_cnt < 0 || iz_lo + iz_cnt > p->nz || iw_lo < 0 || iw_cnt < 0 || iw_lo + iw_cnt > p->nw)
    return fail(p, JERK_EINVAL, "template box outside the plan's grid");
  if (!bank_covers(p, iz_lo, iz_cnt, iw_lo, iw_cnt)) return fail(p, JERK_ESTATE, "the template box is not inside the range jerk_templates_range built");
  cudaStream_t st = (cudaStream_t)stream;
  SearchParams sp;
  fill_params(p, sp, d_spec, d_work, work_bytes);
  const TemplateBox box{iz_lo, iz_cnt, iw_lo, iw_cnt};
  OrderParams op;
  add_class_jobs(p, sp, &box, 1, d_work, op);   // an empty box adds nothing: *d_count = 0
  sp.threshold = threshold;
  sp.cands = d_cands;
  sp.max_cands = max_cands;
  sp.count = d_count;
  return run_candidate_search(p, sp, op, st, "k_search(cand)", [&] { return dispatch_search<MODE_CAND>(p, sp, st); });
}

int jerk_search_candidates(jerk_plan* p, const void* d_spec, float threshold, jerk_cand* d_cands, int64_t max_cands,
                           unsigned long long* d_count, void* d_work, uint64_t work_bytes, void* stream) {
  if (!p) return JERK_EINVAL;
  return jerk_search_candidates_range(p, d_spec, threshold, 0, p->nz, 0, p->nw, d_cands, max_cands, d_count, d_work, work_bytes,
                                      stream);
}

int jerk_search_candidates_templates(jerk_plan* p, const void* d_spec, float threshold, int ti_lo, int ti_cnt, jerk_cand* d_cands,
                                     int64_t max_cands, unsigned long long* d_count, void* d_work, uint64_t work_bytes, void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (!d_cands || !d_count || max_cands < 0) return JERK_EINVAL;
  if (ti_lo < 0 || ti_cnt < 0 || ti_lo + ti_cnt > p->T) return fail(p, JERK_EINVAL, "template range outside [0, ntemplates)");
  if (ti_cnt && (ti_lo < p->bank_ti_lo || ti_lo + ti_cnt > p->bank_ti_lo + p->bank_ti_cnt))
    return fail(p, JERK_ESTATE, "the template range is not inside the range jerk_templates_range built");
  cudaStream_t st = (cudaStream_t)stream;
  SearchParams sp;
  fill_params(p, sp, d_spec, d_work, work_bytes);
  // a flat range of templates is at most three boxes: the rest of the first w-row, whole w-rows, the start of the last one
  TemplateBox boxes[3];
  int nboxes = 0;
  int ti = ti_lo, left = ti_cnt;
  if (left && ti % p->nz) {
    const int n = std::min(left, p->nz - ti % p->nz);
    boxes[nboxes++] = TemplateBox{ti % p->nz, n, ti / p->nz, 1};
    ti += n;
    left -= n;
  }
  if (left >= p->nz) {
    const int rows = left / p->nz;
    boxes[nboxes++] = TemplateBox{0, p->nz, ti / p->nz, rows};
    ti += rows * p->nz;
    left -= rows * p->nz;
  }
  if (left) boxes[nboxes++] = TemplateBox{0, left, ti / p->nz, 1};
  OrderParams op;
  add_class_jobs(p, sp, boxes, nboxes, d_work, op);
  sp.threshold = threshold;
  sp.cands = d_cands;
  sp.max_cands = max_cands;
  sp.count = d_count;
  return run_candidate_search(p, sp, op, st, "k_search(cand)", [&] { return dispatch_search<MODE_CAND>(p, sp, st); });
}

int jerk_search_candidates_batch(jerk_plan* p, const void* const* h_d_specs, int nspec, float threshold, jerk_cand* d_cands,
                                 int64_t max_cands, unsigned long long* d_counts, void* d_work, uint64_t work_bytes, void* stream) {
  if (!p || !h_d_specs || nspec < 0 || !d_cands || !d_counts || max_cands < 0) return JERK_EINVAL;
  if (!bank_covers(p, 0, p->nz, 0, p->nw)) return fail(p, JERK_ESTATE, "the batched search needs the whole bank (jerk_templates)");
  cudaStream_t st = (cudaStream_t)stream;
  for (int b0 = 0; b0 < nspec; b0 += kMaxBatch) {      // one launch per kMaxBatch spectra: the bank is streamed once for all of them
    const int nb = std::min(kMaxBatch, nspec - b0);
    for (int b = 0; b < nb; b++) {
      int rc = check_common(p, h_d_specs[b0 + b], d_work, work_bytes);
      if (rc) return rc;
    }
    SearchParams sp;
    fill_params(p, sp, h_d_specs[b0], d_work, work_bytes);
    for (int b = 0; b < nb; b++) sp.spec[b] = (const float2*)h_d_specs[b0 + b];
    sp.nspec = nb;
    const TemplateBox grid{0, p->nz, 0, p->nw};
    OrderParams op;
    add_class_jobs(p, sp, &grid, 1, d_work, op);
    sp.threshold = threshold;
    sp.cands = d_cands + (size_t)b0 * max_cands;
    sp.max_cands = max_cands;
    sp.count = d_counts + b0;
    int rc = run_candidate_search(p, sp, op, st, "k_search(cand, batch)", [&] { return dispatch_search<MODE_CAND>(p, sp, st); });
    if (rc) return rc;
  }
  return JERK_OK;
}

int jerk_search_candidates_stats(jerk_plan* p, const void* d_spec, float threshold, jerk_cand* d_cands, int64_t max_cands,
                                 unsigned long long* d_count, double* d_rowstats, uint64_t rowstats_bytes, void* d_work,
                                 uint64_t work_bytes, void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (!d_cands || !d_count || !d_rowstats || max_cands < 0) return JERK_EINVAL;
  if (rowstats_bytes < (uint64_t)p->T * 2 * sizeof(double)) return fail(p, JERK_ENOMEM, "row statistics buffer smaller than 16 bytes per template");
  if ((uintptr_t)d_rowstats % 8) return fail(p, JERK_EINVAL, "d_rowstats must be 8-byte aligned");
  if (!bank_covers(p, 0, p->nz, 0, p->nw)) return fail(p, JERK_ESTATE, "row statistics need the whole bank (jerk_templates)");
  cudaStream_t st = (cudaStream_t)stream;
  SearchParams sp;
  fill_params(p, sp, d_spec, d_work, work_bytes);
  const TemplateBox grid{0, p->nz, 0, p->nw};
  OrderParams op;
  add_class_jobs(p, sp, &grid, 1, d_work, op);
  sp.threshold = threshold;
  sp.cands = d_cands;
  sp.max_cands = max_cands;
  sp.count = d_count;
  sp.rowstats = d_rowstats;
  cudaError_t e = cudaMemsetAsync(d_rowstats, 0, (size_t)p->T * 2 * sizeof(double), st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("row statistics memset: ") + cudaGetErrorString(e));
  return run_candidate_search(p, sp, op, st, "k_search(cand+stats)", [&] { return dispatch_search<MODE_CAND_STATS>(p, sp, st); });
}

int jerk_snr_filter(jerk_plan* p, const double* d_rowstats, const jerk_cand* d_cands_in, const unsigned long long* d_count_in,
                    int64_t max_in, float snr_threshold, jerk_cand* d_cands_out, int64_t max_out, unsigned long long* d_count_out,
                    void* stream) {
  if (!p || !d_rowstats || !d_cands_in || !d_count_in || !d_cands_out || !d_count_out || max_in < 0 || max_out < 0) return JERK_EINVAL;
  if (d_cands_in == d_cands_out) return fail(p, JERK_EINVAL, "jerk_snr_filter is out of place");
  int rc = ensure_device(p);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(d_count_out, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("count memset: ") + cudaGetErrorString(e));
  k_snr_filter<<<p->sm_count, 256, 0, st>>>(d_rowstats, p->nz, (double)p->numbetween * (double)p->nbins, d_cands_in, d_count_in, max_in, snr_threshold,
                                            d_cands_out, max_out, d_count_out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_snr_filter launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

int jerk_sift_candidates(jerk_plan* p, const jerk_cand* d_cands_in, const unsigned long long* d_count_in, int64_t max_in, int wj, int wz,
                         int ww, jerk_cand* d_cands_out, int64_t max_out, unsigned long long* d_count_out, void* stream) {
  if (!p || !d_cands_in || !d_count_in || !d_cands_out || !d_count_out || max_in < 0 || max_out < 0 || wj < 0 || wz < 0 || ww < 0)
    return JERK_EINVAL;
  if (max_in > (1 << 20)) return fail(p, JERK_EINVAL, "jerk_sift_candidates handles lists of at most 2^20 records (pair tests are O(n^2))");
  if (d_cands_in == d_cands_out) return fail(p, JERK_EINVAL, "jerk_sift_candidates is out of place");
  int rc = ensure_device(p);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemsetAsync(d_count_out, 0, sizeof(unsigned long long), st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("count memset: ") + cudaGetErrorString(e));
  k_sift<<<p->sm_count * 4, 256, 0, st>>>(d_cands_in, d_count_in, max_in, wj, wz, ww, d_cands_out, max_out, d_count_out);
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_sift launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

// D2H of the count and of min(count, max_cands) records; the overflow conditions become statuses here, where the call
// is synchronous anyway
static int fetch_candidates(jerk_plan* p, jerk_cand* h_cands, int64_t max_cands, unsigned long long* h_count, const jerk_cand* d_cands,
                            const unsigned long long* d_count, cudaStream_t st) {
  cudaError_t e = cudaMemcpyAsync(h_count, d_count, sizeof(unsigned long long), cudaMemcpyDeviceToHost, st);
  if (e == cudaSuccess) e = cudaStreamSynchronize(st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("D2H count: ") + cudaGetErrorString(e));
  unsigned long long n = *h_count;
  if (n == ~0ULL) return fail(p, JERK_EOVERFLOW, "seam records overflowed d_work: pass a larger work buffer (16 bytes per extra record) or raise the threshold");
  const bool over = (int64_t)n > max_cands;
  if (over) n = (unsigned long long)max_cands;
  if (n) {
    e = cudaMemcpyAsync(h_cands, d_cands, (size_t)n * sizeof(jerk_cand), cudaMemcpyDeviceToHost, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("D2H candidates: ") + cudaGetErrorString(e));
  }
  if (over) return fail(p, JERK_EOVERFLOW, "more candidates than max_cands: the first max_cands records were copied, *h_count holds the total");
  return JERK_OK;
}

int jerk_search_candidates_host(jerk_plan* p, const void* h_spec, float threshold, jerk_cand* h_cands, int64_t max_cands,
                                unsigned long long* h_count, void* d_spec, jerk_cand* d_cands, unsigned long long* d_count,
                                void* d_work, uint64_t work_bytes, void* stream) {
  if (!p || !h_spec || !h_cands || !h_count || !d_spec) return JERK_EINVAL;
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpyAsync(d_spec, h_spec, (size_t)p->nbins * sizeof(float2), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("H2D spectrum: ") + cudaGetErrorString(e));
  int rc = jerk_search_candidates(p, d_spec, threshold, d_cands, max_cands, d_count, d_work, work_bytes, stream);
  if (rc) return rc;
  return fetch_candidates(p, h_cands, max_cands, h_count, d_cands, d_count, st);
}

int jerk_search_series_host(jerk_plan* p, const float* h_series, int64_t nsamples, int block, float threshold, jerk_cand* h_cands,
                            int64_t max_cands, unsigned long long* h_count, float* d_series, void* d_spec, void* d_scratch,
                            uint64_t scratch_bytes, jerk_cand* d_cands, unsigned long long* d_count, void* d_work, uint64_t work_bytes,
                            void* stream) {
  if (!p || !h_series || !h_cands || !h_count || !d_series || !d_spec || !d_scratch) return JERK_EINVAL;
  if (nsamples != 2 * p->nbins) return fail(p, JERK_EINVAL, "the series must have 2 * nbins samples");
  cudaStream_t st = (cudaStream_t)stream;
  cudaError_t e = cudaMemcpyAsync(d_series, h_series, (size_t)nsamples * sizeof(float), cudaMemcpyHostToDevice, st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("H2D series: ") + cudaGetErrorString(e));
  int rc = jerk_prepare_spectrum(d_series, nsamples, block, d_spec, d_scratch, scratch_bytes, stream);
  if (rc) return fail(p, rc, "jerk_prepare_spectrum failed (size, alignment or scratch)");
  rc = jerk_search_candidates(p, d_spec, threshold, d_cands, max_cands, d_count, d_work, work_bytes, stream);
  if (rc) return rc;
  return fetch_candidates(p, h_cands, max_cands, h_count, d_cands, d_count, st);
}

// ---- harmonic stage (row a-6)
}  // extern "C" (reopened below)

namespace jerk {

constexpr int64_t kHarmChunkBins = 1 << 16;      // r-chunk of the top-harmonic axis that jerk_harmonic_scratch_bytes sizes for
constexpr int64_t kHarmChunkBinsMax = 1 << 19;   // larger caller buffers are used up to this chunk (fewer segment-edge recomputations)
constexpr int kHarmJTile = 8192;              // half-bin indices per k_harm block
constexpr uint64_t kHarmHeader = 256;         // running[4] arg-max records
constexpr uint64_t kHarmGuard = 65536;        // guard band before the first and after the last stored sub-plane (see ld_gather7): > (4096 + c_max) * 2 * 7/8 floats
constexpr int kHarmFoldBlocks = 128;          // first level of the arg-max fold

struct HarmBox {
  int64_t r_lo, r_cnt;
  int iz_lo, iz_cnt, iw_lo, iw_cnt;
};
struct HarmSubBox {       // source box of fraction e/8
  int64_t r_lo, r_cnt;
  int iz_lo, iz_cnt, iw_lo, iw_cnt;
  uint64_t offset, bytes;  // inside the scratch buffer
  int64_t seg_first, seg_count;     // segments of the launch that stores it
  uint64_t bmax_offset;             // block maxima [row][seg][kBmaxBlocks][2] (fused path)
};

static int host_rnd_eighths(int a, int e) {
  int m = (abs(a) * e + 4) >> 3;
  return a < 0 ? -m : m;
}

// Source boxes of the fractions for a top-harmonic box (all index maps are monotone, so boxes map to boxes), their
// placement in scratch after the header, the arg-max records, and the total bytes needed.  seg_len 4096 (`fused`): the
// top-harmonic pass itself is the consumer, fraction 8/8 is never stored and the records are one per warp of that launch;
// other lengths: all eight sub-planes are stored and k_harm sums them (records per k_harm block).
// The fused path's pruning bounds a pair of batches (512 outputs, at most 449 source bins of a fraction) by the block maxima
// at its first and last source bin only (harm_bounds_mask), which is exact as long as no block of a unit is shorter
// than 449 outputs.  The edge blocks are cut to 1024 - hw_max outputs by the valid window: hw_max <= 575 would do, 512 is
// the documented gate.  Wider templates take the stored-sub-plane path (k_harm), which has no bounds.
static bool harm_fused(const jerk_plan* p) { return p->L == 4096 && p->hw_max <= 512; }

static uint64_t harm_layout(const jerk_plan* p, const HarmBox& bx, HarmSubBox (&sub)[8], uint64_t* best_off, int* nblocks, int* ntiles) {
  const bool fused = harm_fused(p);
  const int cz = (p->nz - 1) / 2, cw = (p->nw - 1) / 2;
  const int64_t j_lo = 2 * bx.r_lo, j_hi = 2 * (bx.r_lo + bx.r_cnt) - 1;   // inclusive
  uint64_t off = kHarmHeader + (fused ? kHarmGuard : 0);
  for (int e = 1; e <= 8; e++) {
    HarmSubBox& sb = sub[e - 1];
    const int64_t js_lo = (j_lo * e + 4) >> 3, js_hi = (j_hi * e + 4) >> 3;
    sb.r_lo = js_lo >> 1;
    sb.r_cnt = (js_hi >> 1) - sb.r_lo + 1;
    sb.iz_lo = host_rnd_eighths(bx.iz_lo - cz, e) + cz;
    sb.iz_cnt = host_rnd_eighths(bx.iz_lo + bx.iz_cnt - 1 - cz, e) + cz - sb.iz_lo + 1;
    sb.iw_lo = host_rnd_eighths(bx.iw_lo - cw, e) + cw;
    sb.iw_cnt = host_rnd_eighths(bx.iw_lo + bx.iw_cnt - 1 - cw, e) + cw - sb.iw_lo + 1;
    sb.offset = off;
    sb.bytes = (fused && e == 8) ? 0 : align_up((uint64_t)sb.iw_cnt * sb.iz_cnt * (uint64_t)(2 * sb.r_cnt) * sizeof(float), 256);
    off += sb.bytes;
  }
  if (fused) {
    off += kHarmGuard;
    for (int e = 1; e <= 7; e++) {      // block maxima of the stored sub-planes: the bounds of the top-harmonic pass
      HarmSubBox& sb = sub[e - 1];
      job_segments(p, sb.r_lo, sb.r_cnt, &sb.seg_first, &sb.seg_count);
      sb.bmax_offset = off;
      off += align_up((uint64_t)sb.iw_cnt * sb.iz_cnt * (uint64_t)sb.seg_count * kBmaxBlocks * 2 * sizeof(float), 256);
    }
  }
  *ntiles = (int)((2 * bx.r_cnt + kHarmJTile - 1) / kHarmJTile);
  *nblocks = fused ? kStashSlots * 2 : bx.iw_cnt * bx.iz_cnt * *ntiles;      // fused: an upper bound on the warps of the launch
  *best_off = off;
  off += align_up((uint64_t)4 * *nblocks * sizeof(jerk_cand), 256);
  off += align_up((uint64_t)4 * kHarmFoldBlocks * sizeof(jerk_cand), 256);   // partial arg-max records of the two-level fold
  return off;
}

// Sub-planes of one box (one plane-mode launch with one job per fraction), then the sums in arg-max or store mode:
// inside the top-harmonic search pass itself for seg_len 4096 (k_search64<MODE_HARM>), by k_harm otherwise.
static int harm_box(jerk_plan* p, const void* d_spec, const HarmBox& bx, unsigned char* scratch, uint64_t scratch_bytes,
                    void* d_work, uint64_t work_bytes, float* d_out, int out_stage, const float* thr4, bool first, cudaStream_t st) {
  const bool fused = harm_fused(p);
  HarmSubBox sub[8];
  uint64_t bb_off;
  int nblocks, ntiles;
  if (harm_layout(p, bx, sub, &bb_off, &nblocks, &ntiles) > scratch_bytes)
    return fail(p, JERK_ENOMEM, "harmonic scratch buffer too small for this box");
  SearchParams sp;
  fill_params(p, sp, d_spec, d_work, work_bytes);
  HarmParams hp;
  memset(&hp, 0, sizeof(hp));
  for (int e = 1; e <= (fused ? 7 : 8); e++) {
    const HarmSubBox& sb = sub[e - 1];
    float* plane = (float*)(scratch + sb.offset);
    if (!add_job(p, sp, sb.r_lo, sb.r_cnt, sb.iz_lo, sb.iz_cnt, sb.iw_lo, sb.iw_cnt, plane, kChunkTP))
      return fail(p, JERK_EINVAL, "harmonic stage: empty sub-box");
    if (fused && !d_out) sp.jobs[sp.njobs - 1].bmax = (float*)(scratch + sb.bmax_offset);
    hp.sub[e - 1].base = plane;
    hp.sub[e - 1].j0 = 2 * sb.r_lo;
    hp.sub[e - 1].nj = 2 * sb.r_cnt;
    hp.sub[e - 1].iz_lo = sb.iz_lo;
    hp.sub[e - 1].iz_cnt = sb.iz_cnt;
    hp.sub[e - 1].iw_lo = sb.iw_lo;
  }
  // small boxes: shrink the work items until every resident FFT group gets a few
  const long long want_items = 32LL * 4 * p->sm_count;
  while (sp.nitems < want_items && sp.jobs[0].chunk_tp > 32) {
    sp.nitems = 0;
    for (int q = 0; q < sp.njobs; q++) {
      SearchJob& jb = sp.jobs[q];
      jb.chunk_tp >>= 1;
      sp.nitems += (long long)((jb.ntp + jb.chunk_tp - 1) / jb.chunk_tp) * jb.seg_count;
      jb.item_end = sp.nitems;
    }
  }
  k_reset<<<1, 32, 0, st>>>(sp.work, nullptr, 0);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_reset launch: ") + cudaGetErrorString(e));
  e = dispatch_search<MODE_PLANE>(p, sp, st);
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_search(harmonic sub-planes) launch: ") + cudaGetErrorString(e));
  jerk_cand* best = (jerk_cand*)(scratch + bb_off);
  jerk_cand* partial = (jerk_cand*)(scratch + bb_off + align_up((uint64_t)4 * nblocks * sizeof(jerk_cand), 256));
  if (fused) {
    // the top-harmonic pass: the search of the box itself, summing the seven stored sub-planes into its own powers
    SearchParams tp;
    fill_params(p, tp, d_spec, d_work, work_bytes);
    OrderParams op;
    memset(&op, 0, sizeof(op));
    {   // on the overlap classes of the candidate searches (add_class_jobs): a template has one segmentation in every call
      const TemplateBox tb{bx.iz_lo, bx.iz_cnt, bx.iw_lo, bx.iw_cnt};
      add_class_jobs(p, tp, &tb, 1, d_work, op, bx.r_lo, bx.r_cnt);
      if (tp.njobs == 0) return fail(p, JERK_EINVAL, "harmonic stage: empty box");
    }
    HarmGather& hg = tp.hg;
    for (int f = 0; f < 7; f++) {
      hg.base[f] = hp.sub[f].base;
      hg.j0[f] = hp.sub[f].j0;
      hg.nj[f] = hp.sub[f].nj;
      hg.iz_lo[f] = hp.sub[f].iz_lo;
      hg.iz_cnt[f] = hp.sub[f].iz_cnt;
      hg.iw_lo[f] = hp.sub[f].iw_lo;
    }
    for (int f = 0; f < 7; f++) {
      hg.bmax[f] = (const float*)(scratch + sub[f].bmax_offset);
      hg.seg_first[f] = (int)sub[f].seg_first;
      hg.seg_count[f] = (int)sub[f].seg_count;
    }
    hg.cz = (p->nz - 1) / 2;
    hg.cw = (p->nw - 1) / 2;
    for (int q = 0; q < 4; q++) hg.thr[q] = thr4 ? thr4[q] : 0.f;
    hg.warpbest = best;
    hg.out = d_out;
    hg.out_stage = out_stage;
    hg.out_iz_lo = bx.iz_lo;
    hg.out_iz_cnt = bx.iz_cnt;
    hg.out_iw_lo = bx.iw_lo;
    k_reset<<<1, 32, 0, st>>>(tp.work, nullptr, 0);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_reset launch: ") + cudaGetErrorString(e));
    if (op.total) {
      k_order<<<1, 1024, 0, st>>>(op);
      e = cudaGetLastError();
      if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_order launch: ") + cudaGetErrorString(e));
    }
    if (d_out) {
      e = launch_search64<MODE_HARM_STORE>(p, tp, st);
    } else {
      e = launch_search64<MODE_HARM>(p, tp, st);
      const int nwarps = (int)search64_grid<MODE_HARM>(p, tp.nitems) * 2 * K64<MODE_HARM>::NG;
      if (e == cudaSuccess) {
        k_harm_fold<<<1, 256, 0, st>>>(best, nwarps, nullptr, (jerk_cand*)scratch, first ? 1 : 0);
        e = cudaGetLastError();
      }
    }
    if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_search64(top-harmonic pass) launch: ") + cudaGetErrorString(e));
    return JERK_OK;
  }
  hp.j_lo = 2 * bx.r_lo;
  hp.nj = 2 * bx.r_cnt;
  hp.iz_lo = bx.iz_lo;
  hp.iz_cnt = bx.iz_cnt;
  hp.iw_lo = bx.iw_lo;
  hp.iw_cnt = bx.iw_cnt;
  hp.cz = (p->nz - 1) / 2;
  hp.cw = (p->nw - 1) / 2;
  hp.jtile = kHarmJTile;
  hp.ntiles = ntiles;
  hp.blockbest = best;
  hp.out = d_out;
  hp.out_stage = out_stage;
  if (d_out) {
    k_harm<true><<<nblocks, 256, 0, st>>>(hp);
  } else {
    k_harm<false><<<nblocks, 256, 0, st>>>(hp);
    k_harm_fold<<<kHarmFoldBlocks, 256, 0, st>>>(hp.blockbest, nblocks, partial, nullptr, 0);
    k_harm_fold<<<1, 256, 0, st>>>(partial, kHarmFoldBlocks, nullptr, (jerk_cand*)scratch, first ? 1 : 0);
  }
  e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_harm launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

static int stage_of(int h) { return h == 1 ? 0 : h == 2 ? 1 : h == 4 ? 2 : h == 8 ? 3 : -1; }

// largest r-chunk (bins) of the full (iz, iw) grid whose scratch fits in `bytes` (0 if not even one 256-bin chunk fits)
static int64_t harm_chunk_for(const jerk_plan* p, uint64_t bytes) {
  int64_t c = std::min<int64_t>(p->nbins, kHarmChunkBinsMax);
  for (;;) {
    // rounding can add a source bin per fraction depending on r_lo: size for a box 16 bins longer
    HarmBox bx{0, c + 16, 0, p->nz, 0, p->nw};
    HarmSubBox sub[8];
    uint64_t bb;
    int nb, nt;
    if (harm_layout(p, bx, sub, &bb, &nb, &nt) <= bytes) return c;
    if (c <= 256) return 0;
    c = (c + 1) / 2;
  }
}

}  // namespace jerk

extern "C" {

uint64_t jerk_harmonic_scratch_bytes(const jerk_plan* p) {
  if (!p) return 0;
  HarmBox bx{0, std::min<int64_t>(p->nbins, kHarmChunkBins) + 16, 0, p->nz, 0, p->nw};   // +16: see harm_chunk_for
  HarmSubBox sub[8];
  uint64_t bb;
  int nb, nt;
  return harm_layout(p, bx, sub, &bb, &nb, &nt);
}

int jerk_harmonic_sum(jerk_plan* p, const void* d_spec, int nstages, const int* h_harm, const float* h_thr, jerk_cand* d_top,
                      void* d_scratch, uint64_t scratch_bytes, void* d_work, uint64_t work_bytes, void* stream) {
  if (!p) return JERK_EINVAL;
  return jerk_harmonic_sum_range(p, d_spec, nstages, h_harm, h_thr, 0, p->nbins, d_top, d_scratch, scratch_bytes, d_work, work_bytes, stream);
}

int jerk_harmonic_sum_range(jerk_plan* p, const void* d_spec, int nstages, const int* h_harm, const float* h_thr, int64_t r_lo,
                            int64_t r_cnt, jerk_cand* d_top, void* d_scratch, uint64_t scratch_bytes, void* d_work, uint64_t work_bytes,
                            void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (nstages < 1 || nstages > 4 || !h_harm || !h_thr || !d_top || !d_scratch) return JERK_EINVAL;
  if ((uintptr_t)d_scratch % 256) return fail(p, JERK_EINVAL, "d_scratch must be 256-byte aligned");
  HarmEmit he;
  he.nstages = nstages;
  for (int s = 0; s < nstages; s++) {
    he.stage[s] = stage_of(h_harm[s]);
    he.thr[s] = h_thr[s];
    if (he.stage[s] < 0) return fail(p, JERK_EINVAL, "harmonic stages must be 1, 2, 4 or 8");
  }
  if (p->numbetween != 2) return fail(p, JERK_EINVAL, "the harmonic stage needs numbetween = 2");
  if (!bank_covers(p, 0, p->nz, 0, p->nw)) return fail(p, JERK_ESTATE, "the harmonic stage needs the whole bank (jerk_templates)");
  float thr4[4] = {INFINITY, INFINITY, INFINITY, INFINITY};   // per stage index log2 h: the lowest threshold asked for (unrequested stages are not tracked)
  for (int s = 0; s < nstages; s++) thr4[he.stage[s]] = fminf(thr4[he.stage[s]], h_thr[s]);
  if (r_lo < 0 || r_cnt < 0 || r_lo > p->nbins - r_cnt) return fail(p, JERK_EINVAL, "harmonic r-range outside [0, nbins)");
  const int64_t chunk = harm_chunk_for(p, scratch_bytes);
  if (chunk == 0) return fail(p, JERK_ENOMEM, "harmonic scratch buffer too small (see jerk_harmonic_scratch_bytes)");
  cudaStream_t st = (cudaStream_t)stream;
  bool first = true;
  if (r_cnt == 0) {   // an empty range (a surplus rank of a sharded stage): no running record, every stage reports j = -1
    cudaError_t e0 = cudaMemsetAsync(d_scratch, 0xFF, kHarmHeader, st);
    if (e0 != cudaSuccess) return fail(p, JERK_ECUDA, std::string("harmonic header memset: ") + cudaGetErrorString(e0));
  }
  for (int64_t r0 = r_lo; r0 < r_lo + r_cnt; r0 += chunk) {
    HarmBox bx{r0, std::min<int64_t>(chunk, r_lo + r_cnt - r0), 0, p->nz, 0, p->nw};
    rc = harm_box(p, d_spec, bx, (unsigned char*)d_scratch, scratch_bytes, d_work, work_bytes, nullptr, 0, thr4, first, st);
    if (rc) return rc;
    first = false;
  }
  k_harm_emit<<<1, 32, 0, st>>>((const jerk_cand*)d_scratch, d_top, he);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return fail(p, JERK_ECUDA, std::string("k_harm_emit launch: ") + cudaGetErrorString(e));
  return JERK_OK;
}

int jerk_harmonic_plane(jerk_plan* p, const void* d_spec, int h, int64_t r_lo, int64_t r_cnt, int iz_lo, int iz_cnt, int iw_lo,
                        int iw_cnt, float* d_out, uint64_t out_bytes, void* d_scratch, uint64_t scratch_bytes, void* d_work,
                        uint64_t work_bytes, void* stream) {
  int rc = check_common(p, d_spec, d_work, work_bytes);
  if (rc) return rc;
  if (stage_of(h) < 0) return fail(p, JERK_EINVAL, "h must be 1, 2, 4 or 8");
  if (p->numbetween != 2) return fail(p, JERK_EINVAL, "the harmonic stage needs numbetween = 2");
  if (!bank_covers(p, 0, p->nz, 0, p->nw)) return fail(p, JERK_ESTATE, "the harmonic stage needs the whole bank (jerk_templates)");
  if (r_lo < 0 || r_cnt < 0 || r_lo + r_cnt > p->nbins || iz_lo < 0 || iz_cnt < 0 || iz_lo + iz_cnt > p->nz || iw_lo < 0 ||
      iw_cnt < 0 || iw_lo + iw_cnt > p->nw)
    return fail(p, JERK_EINVAL, "harmonic plane sub-range outside the plan's grid");
  if (out_bytes < jerk_plane_bytes(r_cnt, iz_cnt, iw_cnt)) return fail(p, JERK_ENOMEM, "harmonic plane buffer too small");
  if (r_cnt == 0 || iz_cnt == 0 || iw_cnt == 0) return JERK_OK;
  if (!d_out || !d_scratch) return JERK_EINVAL;
  if ((uintptr_t)d_scratch % 256) return fail(p, JERK_EINVAL, "d_scratch must be 256-byte aligned");
  HarmBox bx{r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt};
  return harm_box(p, d_spec, bx, (unsigned char*)d_scratch, scratch_bytes, d_work, work_bytes, d_out, stage_of(h), nullptr, true, (cudaStream_t)stream);
}

}  // extern "C"
