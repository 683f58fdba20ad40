#!/usr/bin/env python
"""bench.py — headline measurement of the jerk-search hot path (BASELINE.json metric).

One "step" is one full candidate-mode search (all SURVEY.md 8(a) rows a-2..a-5 over the whole (r,z,w) volume) of the
zmax=200 / wmax=600 configuration (BASELINE.json configs[2], N = 2^23, seg_len 4096, threshold 25) on a seeded
synthetic spectrum already resident in HBM; the template bank (row a-1) is built once before the timed region, as in a
survey where one bank serves thousands of DM trials (reading S20), and its build time is reported separately.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 1..4]

N > 1 (launched by torchrun, one rank per GPU): every rank searches its own independent spectrum (another DM trial)
with its own copy of the bank: weak scaling, no data-path collective; the only collectives are the
barrier and the max-over-ranks of the device time.

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
# dram__bytes_read.sum + dram__bytes_write.sum of one full-size config-3 k_search64<cand> launch (profiles/r1_05_k_search64_cand_full.md);
# algorithmic minimum = bank + spectrum once = 0.837 GB
NCU_DRAM_BYTES_PER_LAUNCH = {3: 1055630080 + 8592896}


def _measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f)
    except Exception:
        return None


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


def oracle_sample(cfg, X, seconds_target=15.0, seed=7):
    """Time the oracle as it stands on a bounded sample of the workload: random (z,w) rows x a bin range.

    Returns (points_per_s, description, points, seconds).  Template quadrature is part of the oracle's work."""
    from oracle import jerk_oracle as orc
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    rng = np.random.default_rng(seed)
    b_cnt = min(cfg.nbins, 4000)
    b_lo = int(rng.integers(0, cfg.nbins - b_cnt + 1))
    pad = 700
    lo, hi = max(0, b_lo - pad), min(cfg.nbins, b_lo + b_cnt + pad)
    Xs = np.asarray(X[lo:hi])
    rows = 0
    t0 = time.perf_counter()
    while True:
        iz, iw = int(rng.integers(0, zs.size)), int(rng.integers(0, ws.size))
        orc.power_row(Xs, float(zs[iz]), float(ws[iw]), b_lo - lo, b_cnt)
        rows += 1
        el = time.perf_counter() - t0
        if el >= seconds_target or rows >= 4096:
            break
    pts = rows * 2 * b_cnt
    return pts / el, f"{rows} random (z,w) rows x {b_cnt} bins ({pts} points) of {cfg.name}, templates included", pts, el


def run_reference(args, cfg_index):
    """--impl reference: the oracle on host cores, same metric/config; each step is a bounded sample."""
    from paper_1911_01353_b200 import synth
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg = synth.config(cfg_index)
    X = synth.make_spectrum(cfg)
    per_step = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(cfg, X, seconds_target=per_step)
    pts = 0
    secs = 0.0
    desc = ""
    for s in range(args.steps):
        v, desc, p, el = oracle_sample(cfg, X, seconds_target=per_step, seed=100 + s)
        pts += p
        secs += el
    value = pts / secs
    ms_per_step_full = cfg.points / value * 1e3        # extrapolated time of one full search at the oracle's rate
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step_full, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(cfg, note="oracle timed on a bounded sample per step; ms_per_step is extrapolated to a full search"),
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc + f", x{args.steps} steps"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def _config_dict(cfg, note=None):
    d = {
        "workload": f"BASELINE.json configs[{cfg.index - 1}] '{cfg.name}': N=2^{cfg.log2n}, zmax={cfg.zmax:g} dz={cfg.dz:g}, "
                    f"wmax={cfg.wmax:g} dw={cfg.dw:g}, numbetween=2, seg_len={cfg.seg_len}, candidate mode thr={cfg.threshold:g}",
        "nbins": cfg.nbins, "nz": cfg.nz, "nw": cfg.nw, "points_per_search": cfg.points,
        "cache": "inputs larger than L2: the 0.8 GB template bank is streamed every step (no L2 flush needed)",
        "parallelism": "one independent spectrum (DM trial) per GPU, bank replicated; no data-path collective",
    }
    if note:
        d["note"] = note
    return d


def run_cufft_comparator(args, cfg, out):
    """--row cufft (PAPER.md:45 compares its shared-memory FFT with a cuFFT-based convolution): the
    UNFUSED pipeline on the same GPU, built from library calls only (torch.fft = cuFFT, torch elementwise kernels): for a
    block of segments x template-phases  Y = F * G  ->  batched inverse FFT  ->  |y|^2 over the valid window  ->  row max.
    It is a comparator, not a product path: it uses this library's bank (re-ordered to natural order), is checked
    against jerk_search_plane on one block, is timed on a bounded sample of the config-3 workload and extrapolated."""
    import torch
    from paper_1911_01353_b200 import binding, synth
    L = cfg.seg_len
    assert L == 4096, "the comparator re-orders the seg_len-4096 bank layout"
    X = synth.make_spectrum(cfg)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, L)
    plan.templates()
    info = plan.info
    d_spec = binding.spectrum_to_device(X)
    spec = torch.view_as_complex(d_spec)
    # bank in natural order: element k = 64*k1 + t of a (template, phase) sits at float2 slot 2*((k1>>1)*64 + t) + (k1&1)
    k = torch.arange(L, device="cuda")
    k1, t = k >> 6, k & 63
    slot = 2 * ((k1 >> 1) * 64 + t) + (k1 & 1)
    geom_bytes = (info.ntemplates * 8 + 255) // 256 * 256
    bank = plan.bank[geom_bytes:geom_bytes + info.ntemplates * 2 * L * 8].view(torch.float32).view(-1, L, 2)
    ntp_blk, nseg_blk = 512, 64                      # 512 template-phases x 64 segments per block: 1 GB of complex64
    G = torch.view_as_complex(bank[:ntp_blk][:, slot, :].contiguous())           # [ntp, L] natural order
    seg0 = info.nseg // 2
    starts = info.seg_base + (seg0 + torch.arange(nseg_blk, device="cuda")) * info.step
    idx = starts[:, None] + torch.arange(L, device="cuda")[None, :]
    lo, hi = info.hw_max, info.hw_max + info.step

    def block():
        F = torch.fft.fft(spec[idx], dim=1)                                    # [nseg, L]   (a-2)
        Y = F[:, None, :] * G[None, :, :]                                      # [nseg, ntp, L]   (a-3, written to HBM)
        y = torch.fft.ifft(Y, dim=2, norm="forward")                           # unnormalised inverse FFT (cuFFT, batched)
        P = (y.real * y.real + y.imag * y.imag)[:, :, lo:hi]                   # (a-4)
        return P, P.amax(dim=2)                                                # (a-5, reduced to a row maximum)

    P, mx = block()
    # check one template-phase row of the block against the fused kernel's plane output
    geom_c = int(plan.template_geometry(0, 0)[0])
    b_first = int(starts[0].item()) + lo - geom_c
    ours = plan.search_plane(d_spec, b_first, info.step, 0, 1, 0, 1)[0, 0]     # P[j], j = 2*(b - b_first) + p
    theirs = torch.stack([P[0, 0], P[0, 1]], dim=1).reshape(-1)
    err = float(((ours - theirs).abs() / torch.clamp(ours, min=1.0)).max())
    assert err < 1e-3, err
    for _ in range(max(1, args.warmup)):
        block()
    torch.cuda.synchronize()
    ts = []
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        block()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    units = ntp_blk * nseg_blk
    total_units = 2 * info.ntemplates * info.nseg
    out.update({"ms_block": ts, "units_per_block": units, "max_rel_diff_vs_fused_plane": err,
                "extrapolated_ms_per_search": min(ts) * total_units / units,
                "note": "library-only unfused pipeline (cuFFT through torch.fft + elementwise kernels); comparator, not a product path"})
    print(json.dumps(out))
    return 0


def run_row(args):
    """--row harmonic|spectrum|stats|plane: time one of the OTHER rows of the path (not the headline line; one GPU).

    harmonic: jerk_harmonic_sum on BASELINE config 5; spectrum: jerk_prepare_spectrum on the config's time series;
    stats: jerk_search_candidates_stats + jerk_snr_filter on config 3; plane: jerk_search_plane of the whole config-2 volume."""
    import torch
    from paper_1911_01353_b200 import binding, build, synth
    build.build()
    binding.load_library()
    torch.cuda.set_device(0)
    idx = {"harmonic": 5, "plane": 2}.get(args.row, args.config)
    cfg = synth.config(idx)
    out = {"row": args.row, "config": _config_dict(cfg)["workload"], "steps": args.steps, "warmup": args.warmup, "data": "synthetic"}
    if args.row == "cufft":
        return run_cufft_comparator(args, cfg, out)
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
        if args.row == "harmonic":
            fn = lambda: plan.harmonic_sum(d_spec)
        elif args.row == "stats":
            def fn():
                d_c, d_n, d_s = plan.search_candidates_stats(d_spec, cfg.threshold)
                return plan.snr_filter(d_s, d_c, d_n, 20.0)
        else:
            plane = torch.empty((cfg.nw, cfg.nz, 2 * cfg.nbins), dtype=torch.float32, device="cuda")
            fn = lambda: plan.search_plane(d_spec, 0, cfg.nbins, out=plane)
            out["algorithmic_bytes"] = plane.numel() * 4
        out["algorithmic_flops"] = plan.info.flops_per_search
    for _ in range(args.warmup):
        fn()
    torch.cuda.synchronize()
    ts = []
    for _ in range(args.steps):
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        fn()
        b.record()
        torch.cuda.synchronize()
        ts.append(a.elapsed_time(b))
    out["ms"] = ts
    out["ms_best"] = min(ts)
    if "algorithmic_bytes" in out:
        out["GBps_algorithmic"] = out["algorithmic_bytes"] / min(ts) / 1e6
    print(json.dumps(out))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config number 1..4 (default 3: the headline)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--row", default="search", choices=["search", "harmonic", "spectrum", "stats", "plane", "cufft"],
                    help="search (default) = the headline bench line; the others time another row of the path and print their own line")
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
    from paper_1911_01353_b200 import binding, build, synth

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
        achieved = info.flops_per_search / (kernel_ms * 1e-3) / 1e12
        peaks = _measured_peaks()
        try:
            measured_fp32 = binding.probe_fp32_tflops()
        except Exception:
            measured_fp32 = None
        roofline = {
            "bound": "alu", "achieved": achieved, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s", "frac": achieved / FP32_PEAK_TFLOPS,
            "traffic": None if args.log2n else NCU_DRAM_BYTES_PER_LAUNCH.get(args.config),
            "traffic_unit": "bytes per launch (ncu dram read+write, profiles/r1_05)",
            "kernel": "k_search64<cand>" if cfg.seg_len == 4096 else f"k_search<{cfg.seg_len},cand>", "kernel_ms": kernel_ms,
            "algorithmic_flops_per_launch": info.flops_per_search,
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
            "gpu_launches": 3 * args.steps,
            "roofline": roofline,
            "bank_build_ms": bank_ms, "spectrum_prep_ms": prep_ms, "e2e_from_series_ms": series_ms, "candidates_found": n_found, "step_ms": step_ms,
        }
        if not args.no_cpu_baseline and world == 1:
            v, desc, pts, el = oracle_sample(cfg, X, seconds_target=15.0)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": desc,
                                    "seconds": el, "extrapolated_seconds_per_search": cfg.points / v}
        elif world > 1:
            line["cpu_baseline"] = None
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
