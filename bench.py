#!/usr/bin/env python
"""bench.py — headline measurement of the jerk-search hot path (BASELINE.json metric).

One "step" is one full candidate-mode search (all SURVEY.md 8(a) rows a-2..a-5 over the whole (r,z,w) volume) of the
zmax=200 / wmax=600 configuration (BASELINE.json configs[2], N = 2^23, seg_len 4096, threshold 25) on a seeded
synthetic spectrum already resident in HBM; the template bank (row a-1) is built once before the timed region, as in a
survey where one bank serves thousands of DM trials (reading S20), and its build time is reported separately.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..4] [--scaling weak|strong]

The default run (N = 1) also times every other row of the path and puts them in the same JSON line under "rows":
BASELINE configs 1, 2, 4 at their specified seg_len and at seg_len = 0 (the library's choice), config 5 (harmonic sum),
plane mode, the fused row statistics, the batched search and numbetween = 1; --no-rows skips them.

N > 1 (launched by torchrun, one rank per GPU).  --scaling weak (default): every rank searches its own independent
spectrum (another DM trial) with its own copy of the bank, no data-path collective; the only
collectives are the barrier and the max-over-ranks of the device time.  --scaling strong: ONE spectrum, every rank
builds, holds and searches 1/N of the template bank (jerk_templates_range + jerk_search_candidates_templates), the
spectrum is broadcast and the candidate lists gathered inside the timed step (shard.search_candidates_sharded), and the
gathered list is checked against rank 0's whole-grid search.

--impl reference times the oracle (oracle/jerk_oracle.py, as it stands) on this box's host cores on a bounded sample
of the same workload; it is a deliberately slow baseline, not the target.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

METRIC = "ffdot_points_per_sec"
UNIT = "points/s"
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12     # 74.45: SMs x FP32 lanes x 2 (FMA) x max SM clock
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "k_search64_traffic.json")   # written from the ncu capture it names
HARM_FLOP_FACTOR = sum(e ** 3 for e in range(1, 9)) / 512.0                # eight sub-volumes of fractions e/8: 2.53 base searches


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return None


def _ncu_traffic(config_index):
    """DRAM bytes per launch of the headline kernel from the committed ncu capture (profiles/k_search64_traffic.json)."""
    try:
        with open(TRAFFIC_FILE) as f:
            t = json.load(f)
        if t.get("config") != config_index:
            return None, None
        return int(t["dram_bytes_read"]) + int(t["dram_bytes_write"]), f"bytes per launch (ncu dram read+write, capture {t['capture']})"
    except Exception:
        return None, None


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.samples = []
        self.reasons = set()
        self.max_mhz = None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4),
            "hw_power_brake": getattr(nv, "nvmlClocksThrottleReasonHwPowerBrakeSlowdown", 0x80),
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop_evt.wait(0.05)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------ the oracle, timed
def _oracle_row_job(args):
    from oracle import jerk_oracle as orc
    Xs, z, w, b_rel, b_cnt = args
    return orc.power_row(Xs, z, w, b_rel, b_cnt).size


def _nproc():
    try:
        return len(os.sched_getaffinity(0))
    except Exception:
        return os.cpu_count() or 1


def oracle_sample(cfg, X, seconds_target=8.0, seed=7, workers=1, pool=None):
    """Time the oracle as it stands on a bounded sample of the workload: random (z,w) rows x a 4000-bin range, one row
    per task, `workers` processes.  Returns (points_per_s, description, points, seconds).  Template quadrature is part of
    the oracle's work."""
    from oracle import jerk_oracle as orc
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    rng = np.random.default_rng(seed)
    b_cnt = min(cfg.nbins, 4000)
    b_lo = int(rng.integers(0, cfg.nbins - b_cnt + 1))
    pad = 700
    lo, hi = max(0, b_lo - pad), min(cfg.nbins, b_lo + b_cnt + pad)
    Xs = np.asarray(X[lo:hi])

    def job():
        iz, iw = int(rng.integers(0, zs.size)), int(rng.integers(0, ws.size))
        return (Xs, float(zs[iz]), float(ws[iw]), b_lo - lo, b_cnt)

    rows = 0
    t0 = time.perf_counter()
    if workers <= 1 or pool is None:
        while True:
            _oracle_row_job(job())
            rows += 1
            el = time.perf_counter() - t0
            if el >= seconds_target or rows >= 4096:
                break
    else:
        while True:                                   # waves of 2 rows per worker until the time target is reached
            wave = [job() for _ in range(2 * workers)]
            list(pool.map(_oracle_row_job, wave))
            rows += len(wave)
            el = time.perf_counter() - t0
            if el >= seconds_target or rows >= 65536:
                break
    pts = rows * 2 * b_cnt
    return pts / el, f"{rows} random (z,w) rows x {b_cnt} bins ({pts} points) of {cfg.name}, templates included, {workers} process(es)", pts, el


def oracle_pool(workers):
    import multiprocessing as mp
    from concurrent.futures import ProcessPoolExecutor
    pool = ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn"))
    list(pool.map(_oracle_row_job, [(np.zeros(64, np.complex64), 0.0, 0.0, 8, 4)] * (2 * workers)))    # start the workers (imports) outside the timed region
    return pool


def cpu_baseline(cfg, X):
    """The oracle on ALL host cores of this box (a process pool over rows) plus the 1-core figure."""
    n = _nproc()
    v1, d1, p1, s1 = oracle_sample(cfg, X, seconds_target=6.0, workers=1)
    out = {"value": v1, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": d1, "seconds": s1,
           "value_1core": v1, "extrapolated_seconds_per_search": cfg.points / v1, "host_cores": n}
    if n > 1:
        pool = oracle_pool(n)
        try:
            v, d, p, s = oracle_sample(cfg, X, seconds_target=10.0, seed=8, workers=n, pool=pool)
        finally:
            pool.shutdown()
        out.update({"value": v, "cores": n, "sample": d, "seconds": s, "extrapolated_seconds_per_search": cfg.points / v,
                    "sample_1core": d1, "seconds_1core": s1})
    return out


def run_reference(args, cfg_index):
    """--impl reference: the oracle on the host cores, same metric/config; each step is a bounded sample."""
    import workloads as synth
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = synth.config(cfg_index)
    X = synth.make_spectrum(cfg)
    n = _nproc()
    pool = oracle_pool(n) if n > 1 else None
    per_step = max(2.0, min(12.0, 90.0 / max(1, args.steps + args.warmup)))
    try:
        for _ in range(args.warmup):
            oracle_sample(cfg, X, seconds_target=per_step, workers=n, pool=pool)
        pts, secs, desc = 0, 0.0, ""
        for s in range(args.steps):
            v, desc, p, el = oracle_sample(cfg, X, seconds_target=per_step, seed=100 + s, workers=n, pool=pool)
            pts += p
            secs += el
    finally:
        if pool is not None:
            pool.shutdown()
    value = pts / secs
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": secs * 1e3 / max(1, args.steps), "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(cfg),
        "note": "each step is a bounded sample of the workload (ms_per_step is the sample's own time); a full search at this rate is extrapolated_ms_per_search",
        "points_per_step": pts / max(1, args.steps), "extrapolated_ms_per_search": cfg.points / value * 1e3,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": n, "kind": "oracle", "sample": desc + f", x{args.steps} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def _config_dict(cfg, seg_len=None, mode="candidate mode"):
    L = cfg.seg_len if seg_len is None else seg_len
    return {
        # kept under 120 characters: the driver's parser cuts longer strings
        "workload": f"configs[{cfg.index - 1}] N=2^{cfg.log2n} zmax={cfg.zmax:g} dz={cfg.dz:g} wmax={cfg.wmax:g} dw={cfg.dw:g} "
                    f"nb=2 seg_len={L} {mode} thr={cfg.threshold:g}",
        "workload_name": cfg.name,
        "nbins": cfg.nbins, "nz": cfg.nz, "nw": cfg.nw, "points_per_search": cfg.points,
        "cache": "inputs larger than L2: the 0.8 GB template bank is streamed every step (no L2 flush needed)",
        "parallelism": "one independent spectrum (DM trial) per GPU, bank replicated; no data-path collective",
    }


# ------------------------------------------------------------------------------------------------ measurement probes
# bench_probes.cu (beside this file) holds two measurement kernels that are not part of the library: built here into
# bench_probes.so (nvcc, sm_100a) and called through ctypes.
_PROBE_SRC = os.path.join(ROOT, "bench_probes.cu")
_PROBE_LIB = os.path.join(ROOT, "bench_probes.so")
_probes = None


def build_probes(force=False):
    """nvcc bench_probes.cu -> bench_probes.so (skipped when the library is newer than the source)."""
    import subprocess
    from paper_1911_01353_b200 import build as _build
    if not force and os.path.exists(_PROBE_LIB) and os.path.getmtime(_PROBE_LIB) >= os.path.getmtime(_PROBE_SRC):
        return _PROBE_LIB
    cmd = [_build.nvcc_path(), "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17", "-Xcompiler", "-fPIC",
           "-shared", "-o", _PROBE_LIB, _PROBE_SRC]
    res = subprocess.run(cmd, capture_output=True, text=True)
    if res.returncode != 0:
        sys.stderr.write(res.stdout + res.stderr)
        raise RuntimeError("nvcc failed building bench_probes.so")
    return _PROBE_LIB


def _load_probes():
    global _probes
    if _probes is None:
        import ctypes as C
        lib = C.CDLL(build_probes())
        lib.bench_probe_fma.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        lib.bench_probe_issue.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_double), C.c_void_p]
        _probes = lib
    return _probes


def _cur_stream():
    import ctypes as C
    import torch
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def probe_fp32_tflops(iters=1 << 15, reps=5):
    """Measured FP32 FMA throughput of the current device in TFLOP/s (bench_probe_fma timed with CUDA events, best of reps)."""
    import torch
    import ctypes as C
    lib = _load_probes()
    d = torch.zeros(4, dtype=torch.float32, device="cuda")
    fl = C.c_double(0.0)
    best = None
    for i in range(reps + 1):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        rc = lib.bench_probe_fma(C.c_void_p(d.data_ptr()), int(iters), C.byref(fl), _cur_stream())
        b.record()
        torch.cuda.synchronize()
        if rc != 0:
            raise RuntimeError(f"bench probe failed with status {rc}")
        ms = a.elapsed_time(b)
        if i > 0:
            best = ms if best is None else min(best, ms)
    return fl.value / (best * 1e-3) / 1e12


def probe_issue_slots(iters=2000):
    """bench_probe_issue: scheduler cycles per round of 8 packed FMAs + 4 companion instructions, by companion kind."""
    import torch
    import ctypes as C
    lib = _load_probes()
    d = torch.zeros(64, dtype=torch.int64, device="cuda")
    out = (C.c_double * 6)()
    rc = lib.bench_probe_issue(C.c_void_p(d.data_ptr()), int(iters), out, _cur_stream())
    if rc != 0:
        raise RuntimeError(f"bench probe failed with status {rc}")
    kinds = ("none", "int_prmt", "lds128", "fmnmx3_abs", "ffma_scalar", "shfl")
    base = out[0]
    return {"cycles_per_round": {k: out[i] for i, k in enumerate(kinds)},
            "packed_fma_cycles": base / 8.0,
            "companion_cost_cycles": {k: (out[i] - base) / 4.0 for i, k in enumerate(kinds) if i}}


# ------------------------------------------------------------------------------------------------ timing helpers
def _time_steps(fn, warmup, steps):
    """Per-step CUDA-event times (ms) of fn on the current stream after `warmup` (>= 3) untimed calls."""
    import torch
    for _ in range(max(3, warmup)):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    return ts


def _row_entry(ts, points, flops, extra=None, flops_nominal=None):
    """`flops` = SURVEY.md 8(d) per-unit flops x the (segment, template-phase) units the timed launches EXECUTE;
    `flops_nominal` (optional) = the same per-unit figure x the nominal ceil(nbins/step) * 2T units of the workload."""
    ms = float(np.median(ts))
    e = {"ms": ms, "ms_best": float(min(ts)), "steps": len(ts), "points_per_s": points / (ms * 1e-3) if points else None}
    if flops:
        e["tflops_executed"] = flops / (ms * 1e-3) / 1e12
        e["frac_fp32_peak"] = e["tflops_executed"] / FP32_PEAK_TFLOPS
    if flops_nominal:
        e["frac_nominal_workload"] = flops_nominal / (ms * 1e-3) / 1e12 / FP32_PEAK_TFLOPS
    if extra:
        e.update(extra)
    return e


def _plane_flops(info):
    """Plane mode runs every template on the hw_max segmentation: nseg * numbetween * T units of 5 L log2 L + 6 L + 3 step flops."""
    L = int(info.seg_len)
    return float(info.nseg) * info.numbetween * info.ntemplates * (5.0 * L * np.log2(L) + 6.0 * L + 3.0 * info.step)


def cufft_unfused_block(cfg, warmup=3, steps=3, check_templates=(0, 100, 255)):
    """SURVEY.md 8(f) N4; PAPER.md:45 compares its shared-memory FFT with a cuFFT-based convolution: the UNFUSED pipeline on
    the same GPU, built from library calls only (torch.fft = cuFFT, torch elementwise kernels): for a block of segments x
    template-phases  Y = F * G  ->  batched inverse FFT  ->  |y|^2 over the valid window  ->  row max.
    It is a comparator, not a product path: it uses this library's bank (re-ordered to natural order), is checked against
    jerk_search_plane on the rows of `check_templates` (flat template indices < 256, both phases), is timed on a bounded
    sample of the workload and extrapolated.  Returns the row's dict."""
    import torch
    from paper_1911_01353_b200 import binding
    import workloads as synth
    L = 4096                                         # the comparator re-orders the seg_len-4096 bank layout
    X = synth.make_spectrum(cfg)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, L)
    plan.templates()
    info = plan.info
    d_spec = binding.spectrum_to_device(X)
    spec = torch.view_as_complex(d_spec)
    # bank -> natural order.  Element k = 64*k1 + t of a (template, phase), k1 = 16 a + b, sits at float2 slot
    # 2*((2 b + a/2)*64 + t) + (a & 1), in the mixed form of the fused first radix-4 layer (csrc/jerk.cu bank_slot<4096>):
    # a = 0 plain (re, im); a = 1, 2: (c, t) with g = c (1 + i t); a = 3: (c3 / c1, t3)
    k = torch.arange(L, device="cuda")
    k1, t = k >> 6, k & 63
    a, b = k1 >> 4, k1 & 15
    slot = 2 * ((2 * b + (a >> 1)) * 64 + t) + (a & 1)
    slot_c1 = 2 * ((2 * b) * 64 + t) + 1                      # the a = 1 entry of the same butterfly
    geom_bytes = (info.ntemplates * 8 + 255) // 256 * 256
    bank = plan.bank[geom_bytes:geom_bytes + info.ntemplates * 2 * L * 8].view(torch.float32).view(-1, L, 2)
    ntp_blk = min(512, 2 * int(info.ntemplates))     # 512 template-phases x 64 segments per block: 1 GB of complex64
    nseg_blk = min(64, int(info.nseg))
    raw = bank[:ntp_blk][:, slot, :]                                             # [ntp, L, 2] in natural element order
    c1 = bank[:ntp_blk][:, slot_c1, 0]
    c = torch.where(a[None, :] == 3, raw[..., 0] * c1, raw[..., 0])
    G = torch.where(a[None, :] == 0, torch.complex(raw[..., 0], raw[..., 1]), torch.complex(c, c * raw[..., 1]))   # [ntp, L]
    seg0 = (int(info.nseg) - nseg_blk) // 2
    starts = info.seg_base + (seg0 + torch.arange(nseg_blk, device="cuda")) * info.step
    idx = starts[:, None] + torch.arange(L, device="cuda")[None, :]
    inside = (idx >= 0) & (idx < cfg.nbins)                                     # X[k] = 0 outside the spectrum
    idx_c = idx.clamp(0, cfg.nbins - 1)
    lo, hi = info.hw_max, info.hw_max + info.step

    def block():
        F = torch.fft.fft(torch.where(inside, spec[idx_c], torch.zeros((), dtype=spec.dtype, device="cuda")), dim=1)   # [nseg, L]   (a-2)
        Y = F[:, None, :] * G[None, :, :]                                      # [nseg, ntp, L]   (a-3, written to HBM)
        y = torch.fft.ifft(Y, dim=2, norm="forward")                           # unnormalised inverse FFT (cuFFT, batched)
        P = (y.real * y.real + y.imag * y.imag)[:, :, lo:hi]                   # (a-4)
        return P, P.amax(dim=2)                                                # (a-5, reduced to a row maximum)

    P, mx = block()
    # check template rows of the block (all its segments, both phases) against the fused kernel's plane output
    err = 0.0
    for ti in check_templates:
        if 2 * ti + 1 >= ntp_blk:
            continue
        iz, iw = ti % int(info.nz), ti // int(info.nz)
        geom_c = int(plan.template_geometry(iz, iw)[0])
        b_first = int(starts[0].item()) + lo - geom_c
        b_lo, b_hi = max(b_first, 0), min(b_first + nseg_blk * int(info.step), cfg.nbins)
        ours = plan.search_plane(d_spec, b_lo, b_hi - b_lo, iz, 1, iw, 1)[0, 0]     # P[j], j = 2*(b - b_lo) + p
        theirs = torch.stack([P[:, 2 * ti].reshape(-1), P[:, 2 * ti + 1].reshape(-1)], dim=1)     # [bins of the block, phase]
        theirs = theirs[b_lo - b_first:b_hi - b_first].reshape(-1)
        err = max(err, float(((ours - theirs).abs() / torch.clamp(ours, min=1.0)).max()))
    ts = _time_steps(block, warmup, steps)
    units = ntp_blk * nseg_blk
    total_units = 2 * info.ntemplates * info.nseg
    ms = float(np.median(ts))
    return {"ms": ms, "ms_block": ts, "units_per_block": units, "max_rel_diff_vs_fused_plane": err, "checked_templates": list(check_templates),
            "extrapolated_ms_per_search": float(min(ts)) * total_units / units,
            "note": "library-only unfused pipeline (cuFFT through torch.fft + elementwise kernels); comparator, not a product path"}


def run_cufft_comparator(args, cfg, out):
    """--row cufft: cufft_unfused_block on the chosen config, one JSON line."""
    out.update(cufft_unfused_block(cfg, args.warmup, args.steps))
    assert out["max_rel_diff_vs_fused_plane"] < 1e-3, out["max_rel_diff_vs_fused_plane"]
    print(json.dumps(out))
    return 0


def harmonic_scratch_bytes(plan, free_bytes):
    """Scratch for the harmonic row: 8x the library's default (a 524288-bin r-chunk, the longest the library uses: fewest
    segment-edge recomputations; 80 GB of the 180 GB of a B200) when the device has room, else 4x, else the default."""
    base = plan.harmonic_scratch_bytes()
    for mult in (8, 4):
        if free_bytes > mult * base + (8 << 30):
            return mult * base
    return base


def run_row(args):
    """--row harmonic|spectrum|stats|plane|batch|cufft: time ONE of the other rows of the path and print its own line."""
    import torch
    from paper_1911_01353_b200 import binding, build
    import workloads as synth
    build.build()
    binding.load_library()
    torch.cuda.set_device(0)
    idx = {"harmonic": 5, "plane": 2}.get(args.row, args.config)
    cfg = synth.config(idx)
    out = {"row": args.row, "config": _config_dict(cfg)["workload"], "steps": args.steps, "warmup": args.warmup, "data": "synthetic"}
    if args.row == "cufft":
        return run_cufft_comparator(args, cfg, out)
    points = flops = None
    if args.row == "spectrum":
        d_series = torch.from_numpy(synth.make_series(cfg)).cuda()
        d_spec = torch.empty((cfg.nbins, 2), dtype=torch.float32, device="cuda")
        d_scr = torch.empty(cfg.n * 4, dtype=torch.uint8, device="cuda")
        fn = lambda: binding.prepare_spectrum(d_series, 1000, d_spec, d_scr)
        out["algorithmic_bytes"] = cfg.n * 4 + 5 * cfg.nbins * 8
    else:
        X = synth.make_spectrum(cfg)
        plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
        plan.templates()
        d_spec = binding.spectrum_to_device(X)
        points, flops = cfg.points, plan.info.flops_per_search_executed      # stats / batch: candidate searches on the overlap classes
        if args.row == "harmonic":
            flops = plan.info.flops_per_search
            nbytes = args.scratch_gb << 30 if args.scratch_gb else harmonic_scratch_bytes(plan, torch.cuda.mem_get_info()[0])
            out["scratch_bytes"] = nbytes
            flops *= HARM_FLOP_FACTOR
            fn = lambda: plan.harmonic_sum(d_spec, scratch_bytes=nbytes)
        elif args.row == "stats":
            def fn():
                d_c, d_n, d_s = plan.search_candidates_stats(d_spec, cfg.threshold)
                return plan.snr_filter(d_s, d_c, d_n, 20.0)
        elif args.row == "batch":
            specs = [d_spec] + [binding.spectrum_to_device(synth.make_spectrum(synth.config(idx), trial=b)) for b in range(1, args.batch)]
            points, flops = points * args.batch, flops * args.batch
            out["nspec"] = args.batch
            fn = lambda: plan.search_candidates_batch(specs, cfg.threshold)
        else:
            plane = torch.empty((cfg.nw, cfg.nz, 2 * cfg.nbins), dtype=torch.float32, device="cuda")
            fn = lambda: plan.search_plane(d_spec, 0, cfg.nbins, out=plane)
            flops = _plane_flops(plan.info)
            out["algorithmic_bytes"] = plane.numel() * 4
    ts = _time_steps(fn, args.warmup, args.steps)
    out.update(_row_entry(ts, points, flops))
    out["ms_all"] = ts
    if "algorithmic_bytes" in out:
        out["GBps_algorithmic"] = out["algorithmic_bytes"] / min(ts) / 1e6
    print(json.dumps(out))
    return 0


def other_rows(steps=3):
    """Every other row of the path, timed in the same run (CUDA events, >= 3 warm-ups each): BASELINE configs 1, 2, 4 at
    their specified seg_len and at seg_len = 0 (the library's choice; results do not depend on seg_len, pin P9), plane
    mode, fused statistics, batched spectra, numbetween = 1, and config 5 (harmonic sum)."""
    import torch
    from paper_1911_01353_b200 import binding
    import workloads as synth
    rows = {}
    for idx in (1, 2, 4):
        cfg = synth.config(idx)
        X = synth.make_spectrum(cfg)
        d_spec = binding.spectrum_to_device(X)
        for L in (cfg.seg_len, 0):
            plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, L)
            plan.templates()
            n_steps = 2 if idx == 4 else steps
            ts = _time_steps(lambda: plan.search_candidates(d_spec, cfg.threshold), 3, n_steps)
            n = int(plan.search_candidates(d_spec, cfg.threshold)[1].item())
            rows[f"config{idx}_candidates_seg{L if L else '0(%d)' % int(plan.info.seg_len)}"] = _row_entry(
                ts, cfg.points, plan.info.flops_per_search_executed, {"seg_len": int(plan.info.seg_len), "candidates": n},
                flops_nominal=plan.info.flops_per_search)
            if idx == 2:
                plane = torch.empty((cfg.nw, cfg.nz, 2 * cfg.nbins), dtype=torch.float32, device="cuda")
                ts = _time_steps(lambda: plan.search_plane(d_spec, 0, cfg.nbins, out=plane), 3, steps)
                rows[f"config2_plane_mode_seg{L if L else '0(%d)' % int(plan.info.seg_len)}"] = _row_entry(ts, cfg.points, _plane_flops(plan.info),
                                                                {"plane_bytes": plane.numel() * 4, "plane_GBps": plane.numel() * 4 / np.median(ts) / 1e6},
                                                                flops_nominal=plan.info.flops_per_search)
                del plane
            del plan
        del d_spec
        torch.cuda.empty_cache()
    cfg = synth.config(3)
    X = synth.make_spectrum(cfg)
    d_spec = binding.spectrum_to_device(X)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    plan.templates()

    def stats():
        d_c, d_n, d_s = plan.search_candidates_stats(d_spec, cfg.threshold)
        return plan.snr_filter(d_s, d_c, d_n, 20.0)

    rows["config3_candidates_with_row_statistics"] = _row_entry(_time_steps(stats, 3, steps), cfg.points, plan.info.flops_per_search_executed,
                                                                flops_nominal=plan.info.flops_per_search)
    # threshold sensitivity of the rare candidate path (a warp with a power above the threshold stashes its powers and
    # runs the local-max test): the S/N front end of 8(f) N2 works at powers of 8-12, not 25
    for thr in (12.0, 9.0):
        pt = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len, extra_seams=1 << 24)
        try:
            pt.templates()
            max_c = 1 << 26
            d_c = torch.empty(max_c * 16, dtype=torch.uint8, device="cuda")
            d_n = torch.zeros(1, dtype=torch.int64, device="cuda")
            ts = _time_steps(lambda: pt.search_candidates(d_spec, thr, max_c, d_c, d_n), 3, steps)
            n = int(d_n.item())
            rows[f"config3_candidates_thr{thr:g}"] = _row_entry(
                ts, cfg.points, pt.info.flops_per_search_executed,
                {"threshold": thr, "candidates": n if n >= 0 else "seam records overflowed d_work", "max_cands": max_c},
                flops_nominal=pt.info.flops_per_search)
            del d_c, d_n
        except Exception as exc:      # noqa: BLE001 -- a row, not the headline: report and go on
            rows[f"config3_candidates_thr{thr:g}"] = {"error": repr(exc)}
        del pt
        torch.cuda.empty_cache()
    nspec = 4
    specs = [d_spec] + [binding.spectrum_to_device(synth.make_spectrum(synth.config(3), trial=b)) for b in range(1, nspec)]
    ts = _time_steps(lambda: plan.search_candidates_batch(specs, cfg.threshold), 3, 2)
    rows["config3_batch_of_4_spectra"] = _row_entry(ts, nspec * cfg.points, nspec * plan.info.flops_per_search_executed,
                                                    {"nspec": nspec, "ms_per_spectrum": float(np.median(ts)) / nspec},
                                                    flops_nominal=nspec * plan.info.flops_per_search)
    del specs
    plan1 = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 1, cfg.seg_len)
    plan1.templates()
    ts = _time_steps(lambda: plan1.search_candidates(d_spec, cfg.threshold), 3, steps)
    rows["config3_numbetween1"] = _row_entry(ts, cfg.points // 2, plan1.info.flops_per_search_executed, flops_nominal=plan1.info.flops_per_search)
    del plan1, d_spec
    torch.cuda.empty_cache()
    try:
        rows["cufft_unfused_block"] = cufft_unfused_block(cfg, 3, steps)
    except Exception as exc:          # noqa: BLE001
        rows["cufft_unfused_block"] = {"error": repr(exc)}
    torch.cuda.empty_cache()
    cfg = synth.config(5)
    X = synth.make_spectrum(cfg)
    d_spec = binding.spectrum_to_device(X)
    nbytes = harmonic_scratch_bytes(plan, torch.cuda.mem_get_info()[0])
    ts = _time_steps(lambda: plan.harmonic_sum(d_spec, scratch_bytes=nbytes), 3, 2)
    top = plan.harmonic_sum(d_spec, scratch_bytes=nbytes)
    rows["config5_harmonic_sum_1_2_4_8"] = _row_entry(
        ts, cfg.points, plan.info.flops_per_search * HARM_FLOP_FACTOR,
        {"scratch_bytes": nbytes,
         # the method's own work is ONE search plus seven adds per point (the sub-planes are the same plane on nested boxes):
         "frac_fp32_peak_one_search": plan.info.flops_per_search / (float(np.median(ts)) * 1e-3) / 1e12 / FP32_PEAK_TFLOPS, "stage_tops": [{"h": h, "j": int(r["j"]), "iz": int(r["iz"]), "iw": int(r["iw"]), "S": float(r["power"])}
                                                  for h, r in zip((1, 2, 4, 8), top)],
         "flops_note": "frac_fp32_peak credits the 2.53 base searches this design executes ((1^3 + ... + 8^3)/512: the eight sub-volumes "
                       "of fractions e/8 are recomputed); frac_fp32_peak_one_search counts the one search the method needs"})
    # the same stage with the scratch size the library itself asks for (jerk_harmonic_scratch_bytes: 65536-bin r-chunks)
    try:
        base = int(plan.harmonic_scratch_bytes())
        plan.scratch = None
        torch.cuda.empty_cache()
        ts = _time_steps(lambda: plan.harmonic_sum(d_spec, scratch_bytes=base), 3, 2)
        top_d = plan.harmonic_sum(d_spec, scratch_bytes=base)
        rows["config5_harmonic_sum_default_scratch"] = _row_entry(
            ts, cfg.points, plan.info.flops_per_search * HARM_FLOP_FACTOR,
            {"scratch_bytes": base, "same_stage_tops_as_large_scratch": bool(top_d.tobytes() == top.tobytes()),
             "frac_fp32_peak_one_search": plan.info.flops_per_search / (float(np.median(ts)) * 1e-3) / 1e12 / FP32_PEAK_TFLOPS})
    except Exception as exc:          # noqa: BLE001
        rows["config5_harmonic_sum_default_scratch"] = {"error": repr(exc)}
    return rows


def run_strong(args, torch, dist, rank, local_rank, world):
    """--scaling strong: one spectrum, the template bank sharded over the ranks."""
    from paper_1911_01353_b200 import binding, shard
    import workloads as synth
    cfg = synth.config(args.config)
    X = synth.make_spectrum(cfg)                         # every rank can make it; only rank 0's copy is used (broadcast)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    ti_lo, ti_cnt = shard.build_bank_shard(plan)
    # the split is cut at equal executed units (jerk_template_units), not equal template counts: host-only, same on every rank
    units = plan.template_units()
    ranges = [shard.template_range(int(plan.info.ntemplates), world, r, units) for r in range(world)]
    units_per_rank = [int(units[lo:lo + cnt].sum()) for lo, cnt in ranges]
    d_spec = binding.spectrum_to_device(X if rank == 0 else np.zeros_like(X))
    step = lambda: shard.search_candidates_sharded(plan, d_spec, cfg.threshold)
    merged = step()
    check = None
    if rank == 0:                                        # the gathered list == the whole-grid search of a full bank
        full = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
        full.templates()
        ref, _ = binding.candidates_to_numpy(*full.search_candidates(d_spec, cfg.threshold))
        check = bool(merged.tobytes() == np.sort(ref, order=["iw", "iz", "j"]).tobytes())
        del full
    for _ in range(max(3, args.warmup) - 1):
        step()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local_rank)
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop()
    total_ms = e0.elapsed_time(e1)
    if world > 1:
        total_ms = shard.max_over_ranks(total_ms)
    if rank == 0:
        ms = total_ms / args.steps
        cd = _config_dict(cfg)
        cd["parallelism"] = (f"tp{world} over the template bank: rank r builds and searches a contiguous template range cut at equal executed units; spectrum "
                             "broadcast + candidate all-gather inside the timed step; no collective inside the search")
        print(json.dumps({
            "metric": METRIC, "value": cfg.points / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
            "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": cd, "clocks": clocks, "gathered_equals_whole_grid_search": check, "templates_per_rank": [int(c) for _, c in ranges],
            # imbalance is visible apart from overhead: the slowest rank sets the step time
            "units_per_rank": units_per_rank, "units_imbalance_max_over_mean": max(units_per_rank) / (sum(units_per_rank) / world),
            "bank_bytes_per_rank": int(plan.bank.numel()), "candidates": int(merged.size),
            "gpu_launches": (6 if int(plan.info.nclasses) > 1 else 5) * args.steps,
        }))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..4 (default 3: the headline)")
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-rows", action="store_true", help="skip the other rows of the path (configs 1, 2, 4, 5, plane, statistics, batch)")
    ap.add_argument("--row", default="search", choices=["search", "harmonic", "spectrum", "stats", "plane", "batch", "cufft"],
                    help="search (default) = the headline bench line; the others time another row of the path and print their own line")
    ap.add_argument("--batch", type=int, default=4, help="--row batch: spectra per call")
    ap.add_argument("--scratch-gb", type=int, default=0, help="--row harmonic: scratch buffer size in GiB (default: 8x the library's default chunk when the device has room)")
    ap.add_argument("--log2n", type=int, default=0,
                    help="profiling aid: shorten the time series to 2^LOG2N samples (same grid, same kernel); not the headline")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                       # timing rule: at least 3 warm-up steps

    if args.row != "search":
        return run_row(args)
    if args.impl == "reference":
        return run_reference(args, args.config)

    import torch
    import torch.distributed as dist
    from paper_1911_01353_b200 import binding, build
    import workloads as synth

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback for the product path)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    if rank == 0:
        build.build()
    if world > 1:
        dist.barrier()
    binding.load_library()
    if args.scaling == "strong":
        rc = run_strong(args, torch, dist, rank, local_rank, world)
        if world > 1:
            dist.destroy_process_group()
        return rc

    cfg = synth.config(args.config)
    if args.log2n:
        cfg.log2n = args.log2n
        cfg.name += f"-reduced-2^{args.log2n}"
    X = synth.make_spectrum(cfg, trial=rank)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    info = plan.info
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    plan.templates()                      # first build: includes the lazy load of the CUDA module
    torch.cuda.synchronize()
    ev0.record()
    plan.templates()
    ev1.record()
    torch.cuda.synchronize()
    bank_ms = ev0.elapsed_time(ev1)

    max_cands = 1 << 20
    d_spec = binding.spectrum_to_device(X)
    d_cands = torch.empty(max_cands * 16, dtype=torch.uint8, device="cuda")
    d_count = torch.zeros(1, dtype=torch.int64, device="cuda")

    def step():
        plan.search_candidates(d_spec, cfg.threshold, max_cands, d_cands, d_count)

    def sync_all():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    sync_all()
    n_found = int(d_count.item())

    sampler = ClockSampler(local_rank)
    sampler.start()
    starts = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ends = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    sync_all()
    for i in range(args.steps):
        starts[i].record()
        step()
        ends[i].record()
    sync_all()
    clocks = sampler.stop()
    total_ms = starts[0].elapsed_time(ends[-1])
    step_ms = [s.elapsed_time(e) for s, e in zip(starts, ends)]

    # ---- e2e: the same search through the host-buffer entry point (pinned H2D of the spectrum + D2H of the result inside)
    h_spec = torch.from_numpy(np.ascontiguousarray(X).view(np.float32).reshape(-1, 2)).pin_memory()
    h_cands = torch.empty(max_cands * 16, dtype=torch.uint8).pin_memory()
    h_count = torch.zeros(1, dtype=torch.int64).pin_memory()
    d_spec2 = torch.empty_like(d_spec)
    for _ in range(2):
        plan.search_candidates_host(h_spec, cfg.threshold, h_cands, h_count, d_spec2, d_cands, d_count)
    sync_all()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_host0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        n_e2e = plan.search_candidates_host(h_spec, cfg.threshold, h_cands, h_count, d_spec2, d_cands, d_count)
    e1.record()
    sync_all()
    e2e_ms = max(e0.elapsed_time(e1), (time.perf_counter() - t_host0) * 1e3)

    # ---- upstream stage, reported beside the search: time series -> normalised spectrum on the device
    prep_ms = series_ms = None
    if world == 1 and not args.log2n:
        d_series = torch.from_numpy(synth.make_series(synth.config(args.config), trial=rank)).cuda()
        d_scr = torch.empty(d_series.numel() * 4, dtype=torch.uint8, device="cuda")
        for _ in range(3):
            binding.prepare_spectrum(d_series, 1000, d_spec2, d_scr)
        p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        p0.record()
        for _ in range(10):
            binding.prepare_spectrum(d_series, 1000, d_spec2, d_scr)
        p1.record()
        torch.cuda.synchronize()
        prep_ms = p0.elapsed_time(p1) / 10
        # the whole pipeline from a pinned host time series (H2D series, spectrum preparation, search, D2H candidates)
        h_series = torch.from_numpy(synth.make_series(synth.config(args.config), trial=rank)).pin_memory()
        for _ in range(2):
            plan.search_series_host(h_series, cfg.threshold, h_cands, h_count, d_series, d_spec2, d_scr, d_cands, d_count)
        t_s0 = time.perf_counter()
        for _ in range(args.steps):
            plan.search_series_host(h_series, cfg.threshold, h_cands, h_count, d_series, d_spec2, d_scr, d_cands, d_count)
        torch.cuda.synchronize()
        series_ms = (time.perf_counter() - t_s0) * 1e3 / args.steps
        del d_series, d_scr

    t = torch.tensor([total_ms, e2e_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    total_ms, e2e_ms = float(t[0]), float(t[1])

    if rank == 0:
        ms_per_step = total_ms / args.steps
        value = world * cfg.points / (ms_per_step * 1e-3)
        e2e_value = world * cfg.points / (e2e_ms / args.steps * 1e-3)
        kernel_ms = float(np.mean(step_ms))                   # k_search is > 99.9 % of a step (profiles/)
        # SURVEY.md 8(d) per-unit flops x the units ONE launch executes (the overlap classes run fewer units than the nominal
        # ceil(nbins/step) * 2T of the workload; the nominal figure is kept beside it)
        achieved = info.flops_per_search_executed / (kernel_ms * 1e-3) / 1e12
        achieved_nominal = info.flops_per_search / (kernel_ms * 1e-3) / 1e12
        peaks = _measured_peaks()
        try:
            measured_fp32 = probe_fp32_tflops()
        except Exception:
            measured_fp32 = None
        try:
            issue = probe_issue_slots()
        except Exception:
            issue = None
        traffic, traffic_unit = (None, None) if args.log2n else _ncu_traffic(args.config)
        roofline = {
            "bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
            "traffic": traffic, "traffic_unit": traffic_unit,
            "kernel": "k_search64<cand>" if cfg.seg_len == 4096 else f"k_search<{cfg.seg_len},cand>", "kernel_ms": kernel_ms,
            # what the launch executes: the overlap classes give narrow templates longer steps, i.e. fewer (segment,
            # template-phase) units than the nominal ceil(nbins/step) * 2T of SURVEY.md 8(d) for the same points
            "executed_units_per_launch": int(info.units_per_search), "executed_flops_per_launch": info.flops_per_search_executed,
            "nominal_flops_per_search": info.flops_per_search,
            "achieved_nominal_workload": achieved_nominal, "frac_nominal_workload": achieved_nominal / FP32_PEAK_TFLOPS,
            "note": "achieved/frac = SURVEY.md 8(d) flops per unit (5L log2 L + 6L + 3 step) x executed_units_per_launch / kernel_ms; "
                    "*_nominal_workload uses the workload's nominal ceil(nbins/step) * 2T units at step = L - 2 hw_max (DESIGN.md 6.2)",
            "issue_probe": issue,      # bench_probe_issue: what a non-FMA instruction costs next to packed FP32
            "peak_measured_ffma": measured_fp32, "frac_of_measured_ffma": (achieved / measured_fp32) if measured_fp32 else None,
            "peak_source": "FP32 FMA nominal: 148 SMs x 128 lanes x 2 x 1.965 GHz (DESIGN.md); MEASURED_PEAKS.json has no fp32 entry"
                           + (f"; hbm_gbs={peaks.get('hbm_gbs')} (not the bound here)" if peaks else ""),
        }
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "seconds_per_search": ms_per_step * 1e-3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic", "config": _config_dict(cfg),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(cfg.nbins * 8),
                    "d2h_bytes_per_step": int(8 + min(n_e2e, max_cands) * 16), "ms_per_step": e2e_ms / args.steps},
            "gpu_launches": (6 if int(info.nclasses) > 1 else 5) * args.steps,   # k_reset, (k_order,) k_search64, k_seam_clear, k_seam_insert, k_seam_resolve per search
            "roofline": roofline,
            "bank_build_ms": bank_ms, "spectrum_prep_ms": prep_ms, "e2e_from_series_ms": series_ms, "candidates_found": n_found, "step_ms": step_ms,
        }
        del d_cands, d_spec2
        if world == 1 and not args.no_rows and not args.log2n and args.config == 3:
            del plan, d_spec
            torch.cuda.empty_cache()
            line["rows"] = other_rows()
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = cpu_baseline(cfg, X)
        elif world > 1:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
