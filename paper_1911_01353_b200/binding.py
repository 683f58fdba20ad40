"""Thin ctypes binding of include/jerk.h — argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C-ABI; PyTorch is used here only
for device memory and streams (torch.Tensor.data_ptr(), torch.cuda.current_stream()).  There is no
CPU fallback: if libjerk_b200.so is missing or a call fails, a JerkError is raised.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libjerk_b200.so")

JERK_OK, JERK_EINVAL, JERK_ENOMEM, JERK_ECUDA, JERK_ESTATE, JERK_ENODEV, JERK_EOVERFLOW, JERK_ELIMIT = 0, -1, -2, -3, -4, -5, -6, -7
STATIC_SPECTRUM_MAX_SAMPLES = 1 << 21   # JERK_STATIC_SPECTRUM_MAX_SAMPLES (include/jerk.h)
SEAM_OVERFLOW = (1 << 64) - 1      # *d_count after a search whose seam records did not fit in d_work (include/jerk.h)

CAND_DTYPE = np.dtype([("j", "<i4"), ("iz", "<i2"), ("iw", "<i2"), ("power", "<f4"), ("flags", "<u4")])
assert CAND_DTYPE.itemsize == 16


class JerkError(RuntimeError):
    def __init__(self, status, detail=""):
        self.status = status
        super().__init__(f"jerk status {status}: {detail}")


class PlanInfo(C.Structure):
    _fields_ = [
        ("nbins", C.c_int64), ("zmax", C.c_double), ("dz", C.c_double), ("wmax", C.c_double), ("dw", C.c_double),
        ("numbetween", C.c_int32), ("seg_len", C.c_int32), ("nz", C.c_int32), ("nw", C.c_int32),
        ("ntemplates", C.c_int32), ("hw_max", C.c_int32), ("c_max", C.c_int32), ("step", C.c_int32),
        ("seg_base", C.c_int64), ("nseg", C.c_int64), ("points", C.c_int64),
        ("bank_bytes", C.c_uint64), ("work_bytes", C.c_uint64), ("flops_per_search", C.c_double),
        ("nclasses", C.c_int32), ("reserved", C.c_int32), ("units_per_search", C.c_int64),
        ("flops_per_search_executed", C.c_double),
    ]


EXPORTS = [
    "jerk_plan_create", "jerk_plan_destroy", "jerk_plan_info", "jerk_template_geometry", "jerk_template_units", "jerk_plane_bytes",
    "jerk_templates", "jerk_templates_range", "jerk_bank_bytes_range", "jerk_templates_taps", "jerk_search_plane",
    "jerk_search_candidates", "jerk_search_candidates_range", "jerk_search_candidates_templates",
    "jerk_search_candidates_batch", "jerk_search_candidates_stats", "jerk_snr_filter",
    "jerk_sift_candidates",
    "jerk_search_candidates_host", "jerk_search_series_host", "jerk_harmonic_scratch_bytes", "jerk_harmonic_sum", "jerk_harmonic_sum_range", "jerk_harmonic_plane", "jerk_spectrum_scratch_bytes",
    "jerk_prepare_spectrum", "jerk_prepare_spectrum_mode", "jerk_prepare_spectrum_static", "jerk_strerror",
    "jerk_last_error",
]

_lib = None


def load_library() -> C.CDLL:
    """dlopen the in-tree shared library; fails loudly if it has not been built."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH):
        raise JerkError(JERK_ENODEV, f"{LIB_PATH} not built: run `python -m paper_1911_01353_b200.build` "
                                     "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, i64, u64, dbl, i32 = C.c_void_p, C.c_int64, C.c_uint64, C.c_double, C.c_int
    lib.jerk_plan_create.argtypes = [C.POINTER(vp), i64, dbl, dbl, dbl, dbl, i32, i32]
    lib.jerk_plan_destroy.argtypes = [vp]
    lib.jerk_plan_info.argtypes = [vp, C.POINTER(PlanInfo)]
    lib.jerk_template_geometry.argtypes = [vp, i32, i32, C.POINTER(i32), C.POINTER(i32)]
    lib.jerk_template_units.argtypes = [vp, C.POINTER(i64), i32]
    lib.jerk_plane_bytes.argtypes = [i64, i32, i32]
    lib.jerk_plane_bytes.restype = u64
    lib.jerk_templates.argtypes = [vp, vp, u64, vp]
    lib.jerk_templates_range.argtypes = [vp, i32, i32, vp, u64, vp]
    lib.jerk_bank_bytes_range.argtypes = [vp, i32]
    lib.jerk_bank_bytes_range.restype = u64
    lib.jerk_templates_taps.argtypes = [vp, i32, i32, vp, u64, vp]
    lib.jerk_search_plane.argtypes = [vp, vp, i64, i64, i32, i32, i32, i32, vp, u64, vp, u64, vp]
    lib.jerk_search_candidates.argtypes = [vp, vp, C.c_float, vp, i64, vp, vp, u64, vp]
    lib.jerk_search_candidates_range.argtypes = [vp, vp, C.c_float, i32, i32, i32, i32, vp, i64, vp, vp, u64, vp]
    lib.jerk_search_candidates_templates.argtypes = [vp, vp, C.c_float, i32, i32, vp, i64, vp, vp, u64, vp]
    lib.jerk_search_candidates_batch.argtypes = [vp, C.POINTER(vp), i32, C.c_float, vp, i64, vp, vp, u64, vp]
    lib.jerk_search_candidates_stats.argtypes = [vp, vp, C.c_float, vp, i64, vp, vp, u64, vp, u64, vp]
    lib.jerk_snr_filter.argtypes = [vp, vp, vp, vp, i64, C.c_float, vp, i64, vp, vp]
    lib.jerk_sift_candidates.argtypes = [vp, vp, vp, i64, i32, i32, i32, vp, i64, vp, vp]
    lib.jerk_search_candidates_host.argtypes = [vp, vp, C.c_float, vp, i64, vp, vp, vp, vp, vp, u64, vp]
    lib.jerk_search_series_host.argtypes = [vp, vp, i64, i32, C.c_float, vp, i64, vp, vp, vp, vp, u64, vp, vp, vp, u64, vp]
    lib.jerk_harmonic_scratch_bytes.argtypes = [vp]
    lib.jerk_harmonic_scratch_bytes.restype = u64
    lib.jerk_harmonic_sum.argtypes = [vp, vp, i32, C.POINTER(i32), C.POINTER(C.c_float), vp, vp, u64, vp, u64, vp]
    lib.jerk_harmonic_sum_range.argtypes = [vp, vp, i32, C.POINTER(i32), C.POINTER(C.c_float), i64, i64, vp, vp, u64, vp, u64, vp]
    lib.jerk_harmonic_plane.argtypes = [vp, vp, i32, i64, i64, i32, i32, i32, i32, vp, u64, vp, u64, vp, u64, vp]
    lib.jerk_spectrum_scratch_bytes.argtypes = [i64]
    lib.jerk_spectrum_scratch_bytes.restype = u64
    lib.jerk_prepare_spectrum.argtypes = [vp, i64, i32, vp, vp, u64, vp]
    lib.jerk_prepare_spectrum_mode.argtypes = [vp, i64, i32, i32, vp, vp, u64, vp]
    lib.jerk_prepare_spectrum_static.argtypes = [vp, i64, i32, vp, vp]
    lib.jerk_strerror.argtypes = [i32]
    lib.jerk_strerror.restype = C.c_char_p
    lib.jerk_last_error.argtypes = [vp]
    lib.jerk_last_error.restype = C.c_char_p
    _lib = lib
    return lib


def _stream_ptr(stream=None):
    import torch
    s = stream if stream is not None else torch.cuda.current_stream()
    return C.c_void_p(s.cuda_stream)


class Plan:
    """jerk_plan_create(nbins, zmax, dz, wmax, dw, numbetween, seg_len) and the calls that take a plan."""

    def __init__(self, nbins, zmax, dz, wmax, dw, numbetween=2, seg_len=4096, extra_seams=0):
        self._lib = load_library()
        self.extra_seams = extra_seams
        self._h = C.c_void_p()
        rc = self._lib.jerk_plan_create(C.byref(self._h), int(nbins), float(zmax), float(dz), float(wmax), float(dw),
                                        int(numbetween), int(seg_len))
        if rc != JERK_OK:
            raise JerkError(rc, self._lib.jerk_strerror(rc).decode())
        info = PlanInfo()
        self._check(self._lib.jerk_plan_info(self._h, C.byref(info)))
        self.info = info
        self.bank = None
        self.work = None

    def __del__(self):
        try:
            if getattr(self, "_h", None):
                self._lib.jerk_plan_destroy(self._h)
                self._h = None
        except Exception:
            pass

    def _check(self, rc):
        if rc != JERK_OK:
            raise JerkError(rc, self._lib.jerk_strerror(rc).decode() + " | " + self._lib.jerk_last_error(self._h).decode())

    # ---- host-only queries
    def template_geometry(self, iz, iw):
        c, hw = C.c_int(), C.c_int()
        self._check(self._lib.jerk_template_geometry(self._h, int(iz), int(iw), C.byref(c), C.byref(hw)))
        return c.value, hw.value

    def template_units(self):
        """jerk_template_units: int64[ntemplates], the (segment, template-phase) units a candidate search runs per template."""
        n = int(self.info.ntemplates)
        buf = (C.c_int64 * n)()
        self._check(self._lib.jerk_template_units(self._h, buf, n))
        return np.frombuffer(buf, dtype=np.int64).copy()

    def plane_bytes(self, r_cnt, iz_cnt, iw_cnt):
        return int(self._lib.jerk_plane_bytes(int(r_cnt), int(iz_cnt), int(iw_cnt)))

    # ---- device calls (torch supplies memory and the stream)
    def _ensure_work(self, device):
        """The plan's d_work (caller-owned scratch).  One plan + work buffer serves one call at a time (include/jerk.h);
        `extra_seams` at construction time adds room for more seam records than the 2^20 of info.work_bytes."""
        import torch
        if self.work is None:
            self.work = torch.empty(int(self.info.work_bytes) + 16 * int(self.extra_seams), dtype=torch.uint8, device=device)
        return self.work

    def templates(self, device="cuda", stream=None):
        """jerk_templates: allocates the caller-owned bank as a torch tensor and builds it."""
        import torch
        if self.bank is None:
            self.bank = torch.empty(int(self.info.bank_bytes), dtype=torch.uint8, device=device)
        self._check(self._lib.jerk_templates(self._h, C.c_void_p(self.bank.data_ptr()), int(self.info.bank_bytes),
                                             _stream_ptr(stream)))
        return self.bank

    def templates_range(self, ti_lo, ti_cnt, device="cuda", stream=None):
        """jerk_templates_range: build and hold only templates [ti_lo, ti_lo + ti_cnt) (one rank's share of the bank)."""
        import torch
        nbytes = int(self._lib.jerk_bank_bytes_range(self._h, int(ti_cnt)))
        self.bank = torch.empty(max(nbytes, 256), dtype=torch.uint8, device=device)
        self._check(self._lib.jerk_templates_range(self._h, int(ti_lo), int(ti_cnt), C.c_void_p(self.bank.data_ptr()), nbytes,
                                                   _stream_ptr(stream)))
        return self.bank

    def templates_taps(self, iz, iw, stream=None):
        import torch
        c, hw = self.template_geometry(iz, iw)
        out = torch.empty((4 * hw + 1, 2), dtype=torch.float32, device="cuda")
        self._check(self._lib.jerk_templates_taps(self._h, int(iz), int(iw), C.c_void_p(out.data_ptr()),
                                                  out.numel() * 4, _stream_ptr(stream)))
        return out

    def search_plane(self, d_spec, r_lo, r_cnt, iz_lo=0, iz_cnt=None, iw_lo=0, iw_cnt=None, out=None, stream=None):
        """jerk_search_plane: returns P[iw_cnt][iz_cnt][2*r_cnt] float32 (torch, device)."""
        import torch
        iz_cnt = self.info.nz - iz_lo if iz_cnt is None else iz_cnt
        iw_cnt = self.info.nw - iw_lo if iw_cnt is None else iw_cnt
        if out is None:
            out = torch.empty((iw_cnt, iz_cnt, 2 * r_cnt), dtype=torch.float32, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        self._check(self._lib.jerk_search_plane(
            self._h, C.c_void_p(d_spec.data_ptr()), int(r_lo), int(r_cnt), int(iz_lo), int(iz_cnt), int(iw_lo),
            int(iw_cnt), C.c_void_p(out.data_ptr()), out.numel() * 4, C.c_void_p(work.data_ptr()), work.numel(),
            _stream_ptr(stream)))
        return out

    def search_candidates(self, d_spec, threshold, max_cands=1 << 20, d_cands=None, d_count=None, stream=None):
        """jerk_search_candidates: returns (d_cands uint8[max_cands*16], d_count int64[1]) device tensors (async)."""
        import torch
        if d_cands is None:
            d_cands = torch.empty(max_cands * 16, dtype=torch.uint8, device=d_spec.device)
        if d_count is None:
            d_count = torch.zeros(1, dtype=torch.int64, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        self._check(self._lib.jerk_search_candidates(
            self._h, C.c_void_p(d_spec.data_ptr()), float(threshold), C.c_void_p(d_cands.data_ptr()), int(max_cands),
            C.c_void_p(d_count.data_ptr()), C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return d_cands, d_count

    def search_candidates_range(self, d_spec, threshold, iz_lo, iz_cnt, iw_lo, iw_cnt, max_cands=1 << 20, d_cands=None,
                                d_count=None, stream=None):
        """jerk_search_candidates_range: candidate mode over one template box (the unit of multi-GPU sharding)."""
        import torch
        if d_cands is None:
            d_cands = torch.empty(max_cands * 16, dtype=torch.uint8, device=d_spec.device)
        if d_count is None:
            d_count = torch.zeros(1, dtype=torch.int64, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        self._check(self._lib.jerk_search_candidates_range(
            self._h, C.c_void_p(d_spec.data_ptr()), float(threshold), int(iz_lo), int(iz_cnt), int(iw_lo), int(iw_cnt),
            C.c_void_p(d_cands.data_ptr()), int(max_cands), C.c_void_p(d_count.data_ptr()), C.c_void_p(work.data_ptr()),
            work.numel(), _stream_ptr(stream)))
        return d_cands, d_count

    def search_candidates_templates(self, d_spec, threshold, ti_lo, ti_cnt, max_cands=1 << 20, d_cands=None, d_count=None, stream=None):
        """jerk_search_candidates_templates: candidate mode over the flat template range [ti_lo, ti_lo + ti_cnt)."""
        import torch
        if d_cands is None:
            d_cands = torch.empty(max_cands * 16, dtype=torch.uint8, device=d_spec.device)
        if d_count is None:
            d_count = torch.zeros(1, dtype=torch.int64, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        self._check(self._lib.jerk_search_candidates_templates(
            self._h, C.c_void_p(d_spec.data_ptr()), float(threshold), int(ti_lo), int(ti_cnt), C.c_void_p(d_cands.data_ptr()),
            int(max_cands), C.c_void_p(d_count.data_ptr()), C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return d_cands, d_count

    def search_candidates_batch(self, d_specs, threshold, max_cands=1 << 18, d_cands=None, d_counts=None, stream=None):
        """jerk_search_candidates_batch: a list of device spectra against the one bank; returns (d_cands uint8
        [nspec, max_cands*16], d_counts int64[nspec])."""
        import torch
        n = len(d_specs)
        dev = d_specs[0].device
        if d_cands is None:
            d_cands = torch.empty((n, max_cands * 16), dtype=torch.uint8, device=dev)
        if d_counts is None:
            d_counts = torch.zeros(n, dtype=torch.int64, device=dev)
        work = self._ensure_work(dev)
        ptrs = (C.c_void_p * n)(*[C.c_void_p(x.data_ptr()) for x in d_specs])
        self._check(self._lib.jerk_search_candidates_batch(
            self._h, ptrs, n, float(threshold), C.c_void_p(d_cands.data_ptr()), int(max_cands), C.c_void_p(d_counts.data_ptr()),
            C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return d_cands, d_counts

    def search_candidates_stats(self, d_spec, threshold, max_cands=1 << 20, stream=None):
        """jerk_search_candidates_stats: (d_cands, d_count, d_rowstats float64[T, 2] = {sum P, sum P^2} per (z,w) row)."""
        import torch
        d_cands = torch.empty(max_cands * 16, dtype=torch.uint8, device=d_spec.device)
        d_count = torch.zeros(1, dtype=torch.int64, device=d_spec.device)
        d_stats = torch.empty((self.info.ntemplates, 2), dtype=torch.float64, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        self._check(self._lib.jerk_search_candidates_stats(
            self._h, C.c_void_p(d_spec.data_ptr()), float(threshold), C.c_void_p(d_cands.data_ptr()), int(max_cands),
            C.c_void_p(d_count.data_ptr()), C.c_void_p(d_stats.data_ptr()), d_stats.numel() * 8, C.c_void_p(work.data_ptr()),
            work.numel(), _stream_ptr(stream)))
        return d_cands, d_count, d_stats

    def snr_filter(self, d_stats, d_cands, d_count, snr_threshold, max_out=1 << 20, stream=None):
        """jerk_snr_filter: (d_out, d_count_out); records carry the snr as float bits in `flags`."""
        import torch
        d_out = torch.empty(max_out * 16, dtype=torch.uint8, device=d_cands.device)
        d_nout = torch.zeros(1, dtype=torch.int64, device=d_cands.device)
        self._check(self._lib.jerk_snr_filter(
            self._h, C.c_void_p(d_stats.data_ptr()), C.c_void_p(d_cands.data_ptr()), C.c_void_p(d_count.data_ptr()),
            d_cands.numel() // 16, float(snr_threshold), C.c_void_p(d_out.data_ptr()), int(max_out),
            C.c_void_p(d_nout.data_ptr()), _stream_ptr(stream)))
        return d_out, d_nout

    def sift_candidates(self, d_cands, d_count, wj, wz, ww, max_out=1 << 20, stream=None):
        """jerk_sift_candidates: non-maximum suppression across (j, iz, iw); returns (d_out, d_count_out)."""
        import torch
        d_out = torch.empty(max_out * 16, dtype=torch.uint8, device=d_cands.device)
        d_nout = torch.zeros(1, dtype=torch.int64, device=d_cands.device)
        self._check(self._lib.jerk_sift_candidates(
            self._h, C.c_void_p(d_cands.data_ptr()), C.c_void_p(d_count.data_ptr()), d_cands.numel() // 16, int(wj), int(wz),
            int(ww), C.c_void_p(d_out.data_ptr()), int(max_out), C.c_void_p(d_nout.data_ptr()), _stream_ptr(stream)))
        return d_out, d_nout

    def search_candidates_host(self, h_spec, threshold, h_cands, h_count, d_spec, d_cands, d_count, stream=None):
        """jerk_search_candidates_host: pinned host tensors in/out, device staging caller-owned; synchronous."""
        work = self._ensure_work(d_spec.device)
        max_cands = d_cands.numel() // 16
        self._check(self._lib.jerk_search_candidates_host(
            self._h, C.c_void_p(h_spec.data_ptr()), float(threshold), C.c_void_p(h_cands.data_ptr()), int(max_cands),
            C.c_void_p(h_count.data_ptr()), C.c_void_p(d_spec.data_ptr()), C.c_void_p(d_cands.data_ptr()),
            C.c_void_p(d_count.data_ptr()), C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return int(h_count.item())

    def search_series_host(self, h_series, threshold, h_cands, h_count, d_series, d_spec, d_scratch, d_cands, d_count, block=1000,
                           stream=None):
        """jerk_search_series_host: pinned host time series in, candidates out; device staging caller-owned; synchronous."""
        work = self._ensure_work(d_spec.device)
        max_cands = d_cands.numel() // 16
        self._check(self._lib.jerk_search_series_host(
            self._h, C.c_void_p(h_series.data_ptr()), int(h_series.numel()), int(block), float(threshold),
            C.c_void_p(h_cands.data_ptr()), int(max_cands), C.c_void_p(h_count.data_ptr()), C.c_void_p(d_series.data_ptr()),
            C.c_void_p(d_spec.data_ptr()), C.c_void_p(d_scratch.data_ptr()), d_scratch.numel(), C.c_void_p(d_cands.data_ptr()),
            C.c_void_p(d_count.data_ptr()), C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return int(h_count.item())

    # ---- harmonic stage (row a-6)
    def harmonic_scratch_bytes(self):
        return int(self._lib.jerk_harmonic_scratch_bytes(self._h))

    def _ensure_scratch(self, device, nbytes=None):
        import torch
        nbytes = self.harmonic_scratch_bytes() if nbytes is None else int(nbytes)
        if getattr(self, "scratch", None) is None or self.scratch.numel() < nbytes:
            self.scratch = torch.empty(nbytes, dtype=torch.uint8, device=device)
        return self.scratch

    def harmonic_sum(self, d_spec, harms=(1, 2, 4, 8), thresholds=(25.0, 35.0, 50.0, 75.0), scratch_bytes=None, stream=None,
                     r_lo=0, r_cnt=None):
        """jerk_harmonic_sum (or jerk_harmonic_sum_range when r_lo / r_cnt restrict the top-harmonic positions): returns a
        structured numpy array (CAND_DTYPE) with one record per stage (synchronises)."""
        import torch
        n = len(harms)
        r_cnt = int(self.info.nbins) - int(r_lo) if r_cnt is None else int(r_cnt)
        d_top = torch.zeros(n * 16, dtype=torch.uint8, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        scratch = self._ensure_scratch(d_spec.device, scratch_bytes)
        nbytes = scratch.numel() if scratch_bytes is None else int(scratch_bytes)
        self._check(self._lib.jerk_harmonic_sum_range(
            self._h, C.c_void_p(d_spec.data_ptr()), n, (C.c_int * n)(*[int(h) for h in harms]),
            (C.c_float * n)(*[float(t) for t in thresholds]), int(r_lo), r_cnt, C.c_void_p(d_top.data_ptr()), C.c_void_p(scratch.data_ptr()),
            nbytes, C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return d_top.cpu().numpy().view(CAND_DTYPE).copy()

    def harmonic_plane(self, d_spec, h, r_lo, r_cnt, iz_lo=0, iz_cnt=None, iw_lo=0, iw_cnt=None, stream=None):
        """jerk_harmonic_plane: S_h[iw_cnt][iz_cnt][2*r_cnt] float32 (torch, device) for a box of top-harmonic positions."""
        import torch
        iz_cnt = self.info.nz - iz_lo if iz_cnt is None else iz_cnt
        iw_cnt = self.info.nw - iw_lo if iw_cnt is None else iw_cnt
        out = torch.empty((iw_cnt, iz_cnt, 2 * r_cnt), dtype=torch.float32, device=d_spec.device)
        work = self._ensure_work(d_spec.device)
        scratch = self._ensure_scratch(d_spec.device)
        self._check(self._lib.jerk_harmonic_plane(
            self._h, C.c_void_p(d_spec.data_ptr()), int(h), int(r_lo), int(r_cnt), int(iz_lo), int(iz_cnt), int(iw_lo),
            int(iw_cnt), C.c_void_p(out.data_ptr()), out.numel() * 4, C.c_void_p(scratch.data_ptr()), scratch.numel(),
            C.c_void_p(work.data_ptr()), work.numel(), _stream_ptr(stream)))
        return out

    def work_counters(self):
        """Diagnostic counters the last search left in d_work (item counter, seam records, seam overflow, settled at seams)."""
        return self.work[:64].view(dtype=__import__("torch").int64).cpu().numpy().copy()


NORM_MODES = {"mean": 0, "median": 1, "rednoise": 2}


def prepare_spectrum(d_series, block=1000, d_spec=None, d_scratch=None, stream=None, mode="mean"):
    """jerk_prepare_spectrum_mode: float32 device time series (2^11..2^25 samples) -> complex64 device spectrum of N/2 bins,
    block-normalised (mode "mean", "median" or "rednoise"); returns the spectrum as a float32 tensor of shape (N/2, 2)
    (the d_spec layout of the search calls)."""
    import torch
    lib = load_library()
    n = d_series.numel()
    if d_spec is None:
        d_spec = torch.empty((n // 2, 2), dtype=torch.float32, device=d_series.device)
    nbytes = int(lib.jerk_spectrum_scratch_bytes(n))
    if d_scratch is None:
        d_scratch = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=d_series.device)
    rc = lib.jerk_prepare_spectrum_mode(C.c_void_p(d_series.data_ptr()), int(n), int(block), int(NORM_MODES[mode]),
                                        C.c_void_p(d_spec.data_ptr()), C.c_void_p(d_scratch.data_ptr()), d_scratch.numel(),
                                        _stream_ptr(stream))
    if rc != 0:
        raise JerkError(rc, lib.jerk_strerror(rc).decode())
    return d_spec


def prepare_spectrum_static(d_series, block=1000, d_spec=None, stream=None):
    """jerk_prepare_spectrum_static: prepare_spectrum(mode="mean") for callers that must not allocate device memory (a
    host framework that owns the GPU's memory pool, a latency-critical loop, a plug-in given only its input and output).
    The library keeps the transform's intermediate data in an 8 MiB array of its own, so there is no d_scratch argument
    and the C call allocates nothing; pass d_spec (float32 (N/2, 2) on the series' device) to keep this wrapper from
    allocating the output either.  At most STATIC_SPECTRUM_MAX_SAMPLES (2^21) samples: longer series raise JerkError
    (JERK_ELIMIT).  All calls on a GPU share that one array: keep them on one stream (overlapping calls race), and make
    the first call on each device before any stream capture (it does a one-time address look-up)."""
    import torch
    lib = load_library()
    n = d_series.numel()
    if n > STATIC_SPECTRUM_MAX_SAMPLES:     # refused by the library as well; checked first so that no output is allocated for nothing
        raise JerkError(JERK_ELIMIT, lib.jerk_strerror(JERK_ELIMIT).decode())
    if d_spec is None:
        d_spec = torch.empty((n // 2, 2), dtype=torch.float32, device=d_series.device)
    rc = lib.jerk_prepare_spectrum_static(C.c_void_p(d_series.data_ptr()), int(n), int(block), C.c_void_p(d_spec.data_ptr()),
                                          _stream_ptr(stream))
    if rc != 0:
        raise JerkError(rc, lib.jerk_strerror(rc).decode())
    return d_spec


def candidates_to_numpy(d_cands, d_count):
    """Device candidate buffer -> (structured numpy array sorted by (iw, iz, j), total count).  Raises JerkError
    (JERK_EOVERFLOW) when the search reported a seam-record overflow: that result is incomplete (include/jerk.h)."""
    n = int(d_count.item()) & SEAM_OVERFLOW
    if n == SEAM_OVERFLOW:
        raise JerkError(JERK_EOVERFLOW, "seam records overflowed d_work: use a Plan with extra_seams or a higher threshold")
    cap = d_cands.numel() // 16
    arr = d_cands[: min(n, cap) * 16].cpu().numpy().view(CAND_DTYPE).copy()
    order = np.lexsort((arr["j"], arr["iz"], arr["iw"]))
    return arr[order], n


def spectrum_to_device(X: np.ndarray, device="cuda"):
    """complex64 numpy spectrum -> torch float32 [nbins, 2] tensor on the device."""
    import torch
    a = np.ascontiguousarray(X.astype(np.complex64)).view(np.float32).reshape(-1, 2)
    return torch.from_numpy(a).to(device)
