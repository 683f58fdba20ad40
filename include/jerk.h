/*
 * jerk.h — C-ABI of the B200-native Fourier-domain jerk-search hot path (arXiv 1911.01353).
 *
 * What the library computes (BASELINE.json north_star):
 * the overlap-and-save correlation of a normalised complex spectrum X[0..nbins) with a bank of
 * (z = fdot*T^2, w = fddot*T^3) Fourier-response templates at numbetween = 2 half-bin phases,
 *
 *     A[j; z,w] = sum_m X[b+m] * conj(R_{z,w}(m - p/2)),   j = 2b + p,  p in {0,1},   P = |A|^2,
 *     R_{z,w}(q) = int_0^1 exp(2 pi i (z u^2/2 + w u^3/6 - q u)) du,
 *
 * with the template of (z,w) truncated to |m - c(z,w)| <= hw(z,w), hw = ceil(|z|/2 + |w|/4) + 8 and
 * c = the rounded midpoint of the frequency excursion z u + w u^2/2 (readings S3-S6).
 * Powers are either written out (plane mode) or thresholded into 1-D local-max candidates
 * (P > thr, P > P[j-1], P >= P[j+1] along r within one (z,w) row) inside the same kernel.
 *
 * Conventions
 *  - Every function returns an int status: JERK_OK (0) or a negative jerk_status.  Nothing throws,
 *    aborts or prints.  jerk_strerror() names a status; jerk_last_error() gives call detail.
 *  - Pointers named d_* are DEVICE pointers, h_* are HOST pointers.  The library never allocates,
 *    frees or retains ownership of device memory and never creates streams: every device buffer is
 *    caller-owned (e.g. torch.Tensor.data_ptr()), every call takes the caller's cudaStream_t
 *    (passed as void*) and is asynchronous on it unless stated otherwise.
 *  - The plan is the only library-owned object (host memory).  A plan and the d_work buffer passed with it serve ONE
 *    call at a time: two searches of the same plan (or with the same d_work) must not overlap, on any stream or thread
 *    (the work-item counter, the seam records and the error text live there).  Use one plan + d_work per stream.
 *  - One GPU, sm_100a only; there is no CPU fallback of any kind.
 *  - Grid: z_iz = -zmax + iz*dz (iz = 0..nz-1), w_iw = -wmax + iw*dw (iw = 0..nw-1); template index
 *    ti = iw*nz + iz; r = j/2 bins.
 */
#ifndef JERK_H_
#define JERK_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum jerk_status {
  JERK_OK = 0,
  JERK_EINVAL = -1,   /* bad argument (message in jerk_last_error)                        */
  JERK_ENOMEM = -2,   /* a caller-provided buffer is smaller than the *_bytes the plan asks */
  JERK_ECUDA = -3,    /* a CUDA runtime call or launch failed                              */
  JERK_ESTATE = -4,   /* jerk_templates has not been called for this plan                  */
  JERK_ENODEV = -5,   /* no sm_100 device is current                                       */
  JERK_EOVERFLOW = -6, /* (host entry points) more candidates than max_cands, or more seam records than d_work holds */
  JERK_ELIMIT = -7    /* the request is larger than a fixed, built-in capacity (jerk_prepare_spectrum_static)          */
} jerk_status;

typedef struct jerk_plan jerk_plan;

/* One candidate: r = j/2, z = -zmax + iz*dz, w = -wmax + iw*dw.  16 bytes. */
typedef struct jerk_cand {
  int32_t j;        /* half-bin index, 0 <= j < 2*nbins                                   */
  int16_t iz;
  int16_t iw;
  float power;      /* |A|^2 as computed in fp32 on the device                            */
  uint32_t flags;   /* 0 in the output list (used internally for segment/warp seams)      */
} jerk_cand;

typedef struct jerk_plan_info_t {
  int64_t nbins;
  double zmax, dz, wmax, dw;
  int32_t numbetween;
  int32_t seg_len;       /* L: overlap-save segment (FFT) length                          */
  int32_t nz, nw;
  int32_t ntemplates;    /* nz*nw                                                         */
  int32_t hw_max;        /* max half-width over the bank (overlap is 2*hw_max)            */
  int32_t c_max;         /* max |c(z,w)|                                                  */
  int32_t step;          /* valid outputs per segment = L - 2*hw_max                      */
  int64_t seg_base;      /* first segment starts at this (negative, even) bin            */
  int64_t nseg;          /* segments covering [0, nbins) for every template               */
  int64_t points;        /* numbetween*nbins*nz*nw (r,z,w) points of one full search       */
  uint64_t bank_bytes;   /* size of the template bank buffer jerk_templates fills          */
  uint64_t work_bytes;   /* size of the scratch buffer the search calls need (counters, the   */
                         /* template list of the overlap classes, power stash, 2^20 seam records) */
  double flops_per_search; /* algorithmic FP32 flops: nseg_nominal*2T*(5L log2 L + 6L + 3 step) */
  /* Overlap classes of the candidate searches: templates of similar half-width share a segmentation with
   * step = L - 2*hw_class instead of L - 2*hw_max (fewer segments for narrow templates; same results).             */
  int32_t nclasses;      /* 1: one segmentation (small grids)                                                      */
  int32_t reserved;
  int64_t units_per_search;          /* (segment, template-phase) units a whole-grid candidate search executes     */
  double flops_per_search_executed;  /* the same per-unit formula summed over those units (step of each class)     */
} jerk_plan_info_t;

/*
 * jerk_plan_create — host only (BASELINE.json north_star: jerk_plan_create(nbins, zmax, dz, wmax, dw,
 * numbetween, seg_len)).  Validates the grid and derives nz, nw, c(z,w), hw(z,w), hw_max, step, nseg.
 * Requirements: nbins >= 1; zmax, wmax >= 0; dz, dw > 0 with zmax/dz and wmax/dw integers;
 * numbetween 2 (the half-bin phases p = 0, 1) or 1 (integer bins only, p = 0: half the work; the FDAS-style option of
 * SURVEY.md 8(f) N4; planes then hold one float per bin and the harmonic stage is not offered); seg_len in {1024, 2048, 4096, 8192} and seg_len - 2*hw_max >= 2, or seg_len == 0 for the library's
 * choice (4096, the fastest kernel, whenever it leaves a positive step; 1024 for searches too small to fill that kernel's
 * resident FFT groups; the result does not depend on seg_len); nz, nw < 32768.
 * *out receives a plan that jerk_plan_destroy frees.  Errors: JERK_EINVAL.
 */
int jerk_plan_create(jerk_plan** out, int64_t nbins, double zmax, double dz, double wmax, double dw,
                     int numbetween, int seg_len);
int jerk_plan_destroy(jerk_plan* plan);

/* Copies the derived sizes into *info (host).  Errors: JERK_EINVAL on NULL. */
int jerk_plan_info(const jerk_plan* plan, jerk_plan_info_t* info);

/* Centre c and half-width hw (bins) of template (iz, iw) as the plan computed them (host only). */
int jerk_template_geometry(const jerk_plan* plan, int iz, int iw, int* c, int* hw);

/*
 * jerk_template_units — work per template, for balancing a template-sharded search: h_units[ti]
 * (HOST, n = ntemplates entries, flat index ti = iw*nz + iz) receives the number of (segment, template-phase) units a
 * whole-spectrum candidate search executes for template ti.  Templates are searched on the segmentation of their overlap
 * class (step = seg_len - 2 hw_class), so wide templates cost more units than narrow ones; the sum over ti is
 * jerk_plan_info's units_per_search.  Host-only.  Errors: JERK_EINVAL (null, n != ntemplates).
 */
int jerk_template_units(const jerk_plan* plan, int64_t* h_units, int n);

/* Bytes of a plane-mode output for a sub-range: iw_cnt*iz_cnt*(2*r_cnt)*sizeof(float). */
uint64_t jerk_plane_bytes(int64_t r_cnt, int iz_cnt, int iw_cnt);

/*
 * jerk_templates — build the template bank (BASELINE.json north_star item (1)).
 * For every (z,w) and phase p the response R_{z,w}(c + m' - p/2), |m'| <= hw, is evaluated by fp64
 * Gauss-Legendre quadrature on the device, placed at index (m' mod L) of a zero array, forward-FFTed,
 * conjugated and scaled by 1/L; the result G[ti][p][L] (complex64, in the kernel's own element order)
 * is written to d_bank together with the c/hw tables.  d_bank: DEVICE, >= bank_bytes, 256-byte aligned,
 * caller-owned; the plan remembers the pointer and the caller must keep it alive and unmodified while
 * searching.  Asynchronous on `stream` except for one small host->device table copy.
 * Errors: JERK_EINVAL, JERK_ENOMEM (bank_bytes too small), JERK_ECUDA.
 */
int jerk_templates(jerk_plan* plan, void* d_bank, uint64_t bank_bytes, void* stream);

/*
 * jerk_templates_range — build only templates ti in [ti_lo, ti_lo + ti_cnt) (flat index ti = iw*nz + iz) into d_bank
 * (>= jerk_bank_bytes_range(plan, ti_cnt) bytes: the c/hw tables of the whole grid + ti_cnt filters).  This is what one
 * rank of a template-sharded multi-GPU search holds ("each GPU holds 1/G of the bank"); afterwards the
 * plan searches only boxes / ranges inside it (JERK_ESTATE otherwise).  jerk_templates is the range [0, ntemplates).
 * ti_cnt == 0 is allowed (a rank left without templates when there are more ranks than templates): only the tables are
 * written, and the plan then accepts empty search ranges only.
 */
uint64_t jerk_bank_bytes_range(const jerk_plan* plan, int ti_cnt);
int jerk_templates_range(jerk_plan* plan, int ti_lo, int ti_cnt, void* d_bank, uint64_t bank_bytes, void* stream);

/*
 * jerk_templates_taps — export the raw half-bin lattice R_{z,w}(c - hw + i/2), i = 0..4hw, of one
 * template as complex64 pairs into d_taps (DEVICE, >= (4hw+1)*8 bytes).  Test hook for row a-1.
 */
int jerk_templates_taps(jerk_plan* plan, int iz, int iw, void* d_taps, uint64_t taps_bytes, void* stream);

/*
 * jerk_search_plane — plane-output mode (rows a-2..a-4).  Writes P[iw_rel][iz_rel][j - 2*r_lo] (float32,
 * r fastest) for r_lo <= b < r_lo + r_cnt, iz_lo <= iz < iz_lo + iz_cnt, iw_lo <= iw < iw_lo + iw_cnt.
 * d_spec: DEVICE complex64 X[nbins], 16-byte aligned.  d_plane: DEVICE, >= jerk_plane_bytes(...), 8-byte
 * aligned.  d_work: DEVICE scratch >= work_bytes, 256-byte aligned (contents are overwritten).
 * Errors: JERK_EINVAL (range), JERK_ENOMEM, JERK_ESTATE, JERK_ECUDA.
 */
int jerk_search_plane(jerk_plan* plan, const void* d_spec, int64_t r_lo, int64_t r_cnt, int iz_lo, int iz_cnt,
                      int iw_lo, int iw_cnt, float* d_plane, uint64_t plane_bytes, void* d_work,
                      uint64_t work_bytes, void* stream);

/*
 * jerk_search_candidates — candidate mode (rows a-2..a-5): the whole (r,z,w) volume is searched and only
 * local-max candidates above `threshold` leave the chip.  d_cands: DEVICE array of max_cands records
 * (unordered on return); d_count: DEVICE uint64, set by the call to the total number of candidates found
 * (may exceed max_cands: the excess is dropped, the caller detects overflow by count > max_cands).
 * d_work as above; after the call d_work's first 64 bytes hold diagnostic counters
 * (uint64: [0] work-item counter, [1] seam records, [2] seam overflow flag, [3] candidates settled at seams).
 * Seams: an above-threshold point whose r-neighbour is computed by another warp or segment is parked as a 16-byte seam
 * record in d_work (about 1 in 32 above-threshold points) and settled after the kernel.  plan work_bytes leaves room for
 * 2^20 records; a larger d_work (work_bytes argument) holds 16 bytes per extra record, up to 2^22.  If the records do
 * not fit the result would be incomplete: the call then sets *d_count = UINT64_MAX (never a silently shortened list),
 * which the "count > max_cands" test every caller must make catches; the *_host entry points return JERK_EOVERFLOW.
 * Errors: JERK_EINVAL, JERK_ENOMEM, JERK_ESTATE, JERK_ECUDA.
 */
int jerk_search_candidates(jerk_plan* plan, const void* d_spec, float threshold, jerk_cand* d_cands,
                           int64_t max_cands, unsigned long long* d_count, void* d_work,
                           uint64_t work_bytes, void* stream);

/*
 * jerk_search_candidates_range — candidate mode restricted to the template box iz in [iz_lo, iz_lo+iz_cnt),
 * iw in [iw_lo, iw_lo+iw_cnt) (all r).  This is the unit of multi-GPU sharding (partition by template,
 * w-rows first): the candidate rule is one-dimensional along r inside a (z,w) row (reading S10), so the union of
 * the candidates of disjoint boxes that cover the grid equals the result of jerk_search_candidates.
 * An empty box (iz_cnt == 0 or iw_cnt == 0) sets *d_count = 0.  Other arguments and errors as jerk_search_candidates.
 */
int jerk_search_candidates_range(jerk_plan* plan, const void* d_spec, float threshold, int iz_lo, int iz_cnt,
                                 int iw_lo, int iw_cnt, jerk_cand* d_cands, int64_t max_cands,
                                 unsigned long long* d_count, void* d_work, uint64_t work_bytes, void* stream);

/*
 * jerk_search_candidates_templates — the same for a FLAT range of templates ti in [ti_lo, ti_lo + ti_cnt), ti = iw*nz + iz
 * (one launch over at most three boxes).  Splitting [0, ntemplates) evenly over G ranks leaves at most one template of
 * imbalance; with jerk_templates_range every rank builds and holds only its own part of the bank.
 */
int jerk_search_candidates_templates(jerk_plan* plan, const void* d_spec, float threshold, int ti_lo, int ti_cnt,
                                     jerk_cand* d_cands, int64_t max_cands, unsigned long long* d_count, void* d_work,
                                     uint64_t work_bytes, void* stream);

/*
 * jerk_search_candidates_batch — many spectra against one bank (PAPER.md:27 the search runs once per
 * de-dispersion trial of the pipeline, PAPER.md:39 one bank of filters serves all of them).  h_d_specs: HOST array of
 * nspec DEVICE pointers (each a d_spec as above, all of the plan's nbins).  The spectrum index is one more dimension of
 * the work-item space: one launch per 32 spectra walks every 8 MB chunk of the bank once for all of their segments.
 * Spectrum b gets its own list d_cands[b*max_cands ..) and count d_counts[b] (DEVICE, nspec entries), each exactly what
 * jerk_search_candidates would return for that spectrum alone (same records, unordered; same overflow rules, the seam
 * room of d_work being shared by the spectra of one launch).
 */
int jerk_search_candidates_batch(jerk_plan* plan, const void* const* h_d_specs, int nspec, float threshold,
                                 jerk_cand* d_cands, int64_t max_cands, unsigned long long* d_counts, void* d_work,
                                 uint64_t work_bytes, void* stream);

/*
 * jerk_search_candidates_stats + jerk_snr_filter — the paper's own candidate front end (PAPER.md:43
 * peaks "above a certain threshold" of the output plane, "mean and standard deviation along with candidate
 * selection dominate the execution time"), fused: ONE pass of the search kernel collects local-max candidates above the
 * absolute power `threshold` AND the per-row sums of P and P^2 over all 2*nbins points of every (z,w) row:
 * d_rowstats (DEVICE, double[ntemplates][2], 8-byte aligned, rowstats_bytes >= 16*ntemplates) receives
 * {sum P, sum P^2} of row ti = iw*nz + iz (zeroed by the call; fp64 atomics: the last bits depend on scheduling).
 * jerk_snr_filter then keeps the candidates with snr = (P - mean_row)/std_row > snr_threshold (population standard
 * deviation; rows with zero variance keep nothing), out of place into d_cands_out / d_count_out (DEVICE, zeroed by
 * the call; unordered; overflow as in jerk_search_candidates) with the snr stored as float bits in `flags`.
 * Other arguments and errors as jerk_search_candidates.
 */
int jerk_search_candidates_stats(jerk_plan* plan, const void* d_spec, float threshold, jerk_cand* d_cands,
                                 int64_t max_cands, unsigned long long* d_count, double* d_rowstats,
                                 uint64_t rowstats_bytes, void* d_work, uint64_t work_bytes, void* stream);
int jerk_snr_filter(jerk_plan* plan, const double* d_rowstats, const jerk_cand* d_cands_in,
                    const unsigned long long* d_count_in, int64_t max_in, float snr_threshold,
                    jerk_cand* d_cands_out, int64_t max_out, unsigned long long* d_count_out, void* stream);

/*
 * jerk_sift_candidates — cross-row sifting of a candidate list (PAPER.md:47 future work): a strong
 * signal gives one local-max candidate in every nearby (z,w) row (reading S10); this keeps a candidate iff no
 * other candidate of the list with |dj| <= wj, |diz| <= wz and |diw| <= ww beats it (larger power; equal powers:
 * smaller (iw, iz, j)).  The result does not depend on the order of the list and is a fixed point of the operation.
 * Out of place into d_cands_out / d_count_out (DEVICE; zeroed by the call; unordered; records unchanged); at most
 * 2^20 input records (O(n^2) pair tests).  Errors: JERK_EINVAL, JERK_ENODEV, JERK_ECUDA.
 */
int jerk_sift_candidates(jerk_plan* plan, const jerk_cand* d_cands_in, const unsigned long long* d_count_in,
                         int64_t max_in, int wj, int wz, int ww, jerk_cand* d_cands_out, int64_t max_out,
                         unsigned long long* d_count_out, void* stream);

/*
 * jerk_search_candidates_host — the same search with HOST input/output (end-to-end entry point):
 * copies h_spec (host, ideally pinned, nbins complex64) to d_spec, searches, copies the count and
 * min(count, max_cands) records back to h_count / h_cands and synchronises the stream before returning.
 * All device buffers are still caller-owned staging.  Being synchronous it reports both overflow conditions as
 * JERK_EOVERFLOW: count > max_cands (the first max_cands records are copied, *h_count is the total) and a seam-record
 * overflow (*h_count = UINT64_MAX, nothing copied).
 */
int jerk_search_candidates_host(jerk_plan* plan, const void* h_spec, float threshold, jerk_cand* h_cands,
                                int64_t max_cands, unsigned long long* h_count, void* d_spec,
                                jerk_cand* d_cands, unsigned long long* d_count, void* d_work,
                                uint64_t work_bytes, void* stream);

/*
 * jerk_search_series_host — the whole pipeline from a HOST time series: copies h_series (host, ideally pinned, float32,
 * nsamples = 2*nbins) to d_series, jerk_prepare_spectrum (block-normalised spectrum into d_spec), jerk_search_candidates,
 * copies the count and min(count, max_cands) records back and synchronises the stream.  All device buffers are
 * caller-owned staging (d_series: nsamples floats, 16-byte aligned; d_spec: nbins complex64; d_scratch:
 * jerk_spectrum_scratch_bytes(nsamples)); errors as the calls it is made of.
 */
int jerk_search_series_host(jerk_plan* plan, const float* h_series, int64_t nsamples, int block, float threshold,
                            jerk_cand* h_cands, int64_t max_cands, unsigned long long* h_count, float* d_series,
                            void* d_spec, void* d_scratch, uint64_t scratch_bytes, jerk_cand* d_cands,
                            unsigned long long* d_count, void* d_work, uint64_t work_bytes, void* stream);

/*
 * jerk_harmonic_sum — fused harmonic-sum stage (row a-6; BASELINE.json configs[4]; section 3):
 * S_h(j,iz',iw') = sum_{k=1..h} P[rnd(j k/h); rnd(iz' k/h), rnd(iw' k/h)] with signed grid indices
 * iz' = iz-(nz-1)/2, iw' = iw-(nw-1)/2 and rnd = round half away from zero (reading S13).
 * For each of nstages (1..4) stages (h_harm[s] in {1,2,4,8}, thresholds h_thr[s]; HOST arrays) d_top[s]
 * (DEVICE, nstages records) receives the arg-max of S_h over the whole (j,iz,iw) grid — the position of the
 * top harmonic, power = S_h; ties go to the smallest (iw,iz,j) — if it exceeds the threshold, else
 * {j=-1, iz=0, iw=0, power=0}.  The volume is processed in r-chunks sized to d_scratch.  seg_len 4096: per chunk one
 * plane-mode launch stores the seven sub-planes of fractions 1/8..7/8 (and the block maxima of every unit) in
 * d_scratch, and the search of the chunk itself (fraction 8/8, never stored) adds the gathered sub-harmonic powers to
 * its own powers on chip and keeps the arg-max; the gathers are skipped wherever an exact upper bound built from the
 * block maxima cannot reach the running record.  Other seg_len, and seg_len 4096 with templates wider than
 * hw_max = 512 (the bound needs blocks of at least 449 valid outputs): all eight sub-planes are stored and summed by a
 * separate kernel.
 * d_scratch: DEVICE, 256-byte aligned, >= 1/256 of jerk_harmonic_scratch_bytes(plan) (that size gives the
 * default 65536-bin chunk; smaller buffers give smaller chunks, larger ones longer chunks up to 524288 bins with
 * fewer segment-edge recomputations); d_work as for the search calls.
 * Asynchronous on `stream`.  Errors: JERK_EINVAL, JERK_ENOMEM, JERK_ESTATE, JERK_ECUDA.
 */
uint64_t jerk_harmonic_scratch_bytes(const jerk_plan* plan);
int jerk_harmonic_sum(jerk_plan* plan, const void* d_spec, int nstages, const int* h_harm, const float* h_thr,
                      jerk_cand* d_top, void* d_scratch, uint64_t scratch_bytes, void* d_work,
                      uint64_t work_bytes, void* stream);

/*
 * jerk_harmonic_sum_range — the same restricted to top-harmonic positions r_lo <= b < r_lo + r_cnt (half-bin indices
 * 2 r_lo <= j < 2 (r_lo + r_cnt)): d_top[s] is the arg-max of S_h over that part of the volume.  This is one rank's share of
 * a harmonic stage sharded by r-range ("the r-range partition ... needed for the harmonic stage"): the
 * sub-harmonic powers a range needs lie at r e/8 <= r, so every rank reads the whole spectrum and holds the whole bank, and
 * the ranks' records are folded by (largest power, then smallest (iw, iz, j)).  The values do not depend on how the r axis
 * is cut: the union over disjoint ranges equals jerk_harmonic_sum bit for bit.  r_cnt == 0: every stage reports j = -1.
 * jerk_harmonic_sum is the range [0, nbins).  Errors: as jerk_harmonic_sum, JERK_EINVAL for a range outside [0, nbins).
 */
int jerk_harmonic_sum_range(jerk_plan* plan, const void* d_spec, int nstages, const int* h_harm, const float* h_thr,
                            int64_t r_lo, int64_t r_cnt, jerk_cand* d_top, void* d_scratch, uint64_t scratch_bytes,
                            void* d_work, uint64_t work_bytes, void* stream);

/*
 * jerk_harmonic_plane — plane-output mode of the same stage: writes S_h (h in {1,2,4,8}) for the box
 * r_lo <= b < r_lo+r_cnt, iz_lo <= iz < iz_lo+iz_cnt, iw_lo <= iw < iw_lo+iw_cnt as
 * d_out[iw_rel][iz_rel][j - 2*r_lo] (float32, >= jerk_plane_bytes(r_cnt, iz_cnt, iw_cnt)).  The box is handled
 * as one chunk: JERK_ENOMEM if d_scratch cannot hold its eight sub-planes (a box no larger than the default
 * chunk always fits in jerk_harmonic_scratch_bytes(plan)).
 */
int jerk_harmonic_plane(jerk_plan* plan, const void* d_spec, int h, int64_t r_lo, int64_t r_cnt, int iz_lo,
                        int iz_cnt, int iw_lo, int iw_cnt, float* d_out, uint64_t out_bytes, void* d_scratch,
                        uint64_t scratch_bytes, void* d_work, uint64_t work_bytes, void* stream);

/*
 * Spectrum preparation, the step upstream of the search (BASELINE.json configs[0] "The real FFT
 * gives 32768 complex bins, normalised to unit mean power per 1000-bin block"; reading S15):
 *   X[k] = sum_n x[n] exp(-2 pi i k n / N), k = 0 .. N/2-1 (DC kept, Nyquist dropped), then every consecutive block of
 *   `block` bins (the last one may be shorter) divided by sqrt(mean |X|^2) of that block (an all-zero block is left).
 * d_series: DEVICE float32[nsamples], 16-byte aligned (as d_spec and d_scratch), nsamples a power of two in [2^11, 2^25]; d_spec: DEVICE
 * complex64[nsamples/2] (the d_spec of the search calls); d_scratch: DEVICE, jerk_spectrum_scratch_bytes(nsamples)
 * bytes; all caller-owned.  Asynchronous on `stream`; no plan is needed.  d_series is not modified.
 * Errors: JERK_EINVAL (size, alignment, null), JERK_ENOMEM (scratch too small), JERK_ENODEV, JERK_ECUDA.
 */
uint64_t jerk_spectrum_scratch_bytes(int64_t nsamples);
int jerk_prepare_spectrum(const float* d_series, int64_t nsamples, int block, void* d_spec, void* d_scratch,
                          uint64_t scratch_bytes, void* stream);

/*
 * jerk_prepare_spectrum_mode — the same with a choice of normalisation (SURVEY.md 8(f) N1 "mean as in config 1;
 * median-based and red-noise variants"; the spectrum of a real de-dispersed series, whose noise floor is
 * neither white nor free of strong narrow signals; the paper gives no recipe: readings):
 *   JERK_NORM_MEAN      every `block`-bin block divided by sqrt(mean |X|^2)             (= jerk_prepare_spectrum)
 *   JERK_NORM_MEDIAN    every `block`-bin block divided by sqrt(median |X|^2 / ln 2): for exponentially distributed noise
 *                       powers the median is ln 2 times the mean, and a few strong bins do not move it (even count: mean of
 *                       the two middle values; zero median: block left as it is)
 *   JERK_NORM_REDNOISE  the median rule on blocks whose length grows with frequency, to follow a steep low-frequency noise
 *                       slope: lengths 6, 7, 8, ... each min(block, len + max(1, len / 8)) (integer division), from bin 0
 * block <= 4096 for the median modes (the block is sorted in shared memory), >= 8 for JERK_NORM_REDNOISE.
 * jerk_spectrum_scratch_bytes(nsamples) covers every mode (nsamples/2 complex64 + the red-noise block table);
 * JERK_NORM_MEAN and JERK_NORM_MEDIAN need only the first nsamples/2 * 8 bytes of it.
 */
enum { JERK_NORM_MEAN = 0, JERK_NORM_MEDIAN = 1, JERK_NORM_REDNOISE = 2 };
int jerk_prepare_spectrum_mode(const float* d_series, int64_t nsamples, int block, int mode, void* d_spec, void* d_scratch,
                               uint64_t scratch_bytes, void* stream);

/*
 * jerk_prepare_spectrum_static — jerk_prepare_spectrum (mean normalisation) without a scratch argument, for callers
 * that have no device memory to give and no way to get any: code that runs where cudaMalloc is off limits (inside a
 * host framework whose memory pool owns the whole GPU and forbids side allocations, a real-time acquisition loop that
 * must not take the allocator's lock or its implicit device synchronisation, a plug-in that is handed exactly two
 * buffers — input and output — by its host application).  The transform's intermediate array, which the other entry
 * points take as d_scratch, is here an 8 MiB array built into the library image; the call itself allocates nothing
 * (no cudaMalloc, cudaFree or allocating library routine) and computes exactly what jerk_prepare_spectrum computes.
 *
 * Limit: nsamples <= JERK_STATIC_SPECTRUM_MAX_SAMPLES (2^21, i.e. 2^20 bins); longer series get JERK_ELIMIT and must
 * use jerk_prepare_spectrum with their own scratch.  The price of the built-in array: every GPU on which this library
 * is loaded keeps those 8 MiB until the process exits, whether or not this call is ever made.
 *
 * Sharing: there is ONE array per GPU, used by every call on that GPU from any thread or stream.  Two calls whose GPU
 * work can overlap (different streams, or the same series prepared twice at once) race on it and both results are
 * then undefined: issue them on one stream, or order the streams with events.  The array still holds the previous
 * call's intermediate data when the next call starts; that is harmless, because every call overwrites the part it
 * later reads, so nothing is (or needs to be) cleared.
 *
 * First call on a device: the library looks up, once per device and with that device current, the device address of
 * its array (a symbol-address query that allocates nothing but is a set-up step rather than stream work).  Make the
 * first call on each device during initialisation, before any stream capture is begun.
 *
 * d_series, d_spec, stream, alignment and the lower size limit (2^11) as jerk_prepare_spectrum; both buffers remain
 * caller-owned, d_series is not modified.  Asynchronous on `stream`.
 * Errors: JERK_ELIMIT (nsamples above the limit), JERK_EINVAL (null, size not a power of two or < 2^11, alignment,
 * block < 1), JERK_ENODEV (no sm_100 device current), JERK_ECUDA (address query or launch failed).
 */
#define JERK_STATIC_SPECTRUM_MAX_SAMPLES (1 << 21)
int jerk_prepare_spectrum_static(const float* d_series, int64_t nsamples, int block, void* d_spec, void* stream);

const char* jerk_strerror(int status);
const char* jerk_last_error(const jerk_plan* plan);

#ifdef __cplusplus
}
#endif
#endif /* JERK_H_ */
