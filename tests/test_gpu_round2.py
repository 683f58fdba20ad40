"""GPU parity tests added in round 2 (all through the C-ABI):

 * every candidate / stage top that the FULL-SIZE searches of BASELINE configs 3, 4, 5 return is checked against the oracle
   on its own neighbourhood (power, threshold, local-max rule);
 * the headline kernel instantiation k_search64<cand, PRUNE> (hw_max >= 256) at a low threshold on short / ragged spectra;
 * config 4 at its specified seg_len 8192: random plane rows;
 * seam handling: long seam lists (hash path), seam overflow reported, never silent;
 * batched spectra, bank shards + flat template ranges, numbetween = 1.
"""
import ctypes as C

import numpy as np
import pytest

from oracle import jerk_oracle as orc
from paper_1911_01353_b200 import binding, build, shard
import workloads as synth
from tests import helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    binding.load_library()


_cache = {}


def _setup(idx, seg_len=None):
    key = (idx, seg_len)
    if key not in _cache:
        cfg = synth.config(idx)
        X = synth.make_spectrum(cfg)
        plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len if seg_len is None else seg_len)
        plan.templates()
        d_spec = binding.spectrum_to_device(X)
        torch.cuda.synchronize()
        _cache[key] = (cfg, X, plan, d_spec)
    return _cache[key]


# ------------------------------------------------------------------------------------------------ every candidate, full size
def _verify_every_candidate(cfg, X, cands, thr):
    """Each record (j, iz, iw, P) against the oracle on b-2 .. b+2: the power within tolerance, above the threshold and a
    local maximum (P > P[j-1], P >= P[j+1]), the last two up to the tolerance / near-tie reading S11."""
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    by_row = {}
    for c in cands:
        by_row.setdefault((int(c["iz"]), int(c["iw"])), []).append(c)
    jobs = [(np.asarray(X), float(zs[iz]), float(ws[iw]), sorted({max(0, int(c["j"]) // 2 - 2) for c in cs})) for (iz, iw), cs in by_row.items()]
    res = H.oracle_point_rows(jobs)
    worst = 0.0
    for ((iz, iw), cs), rows in zip(by_row.items(), res):
        for c in cs:
            j, p = int(c["j"]), float(c["power"])
            b_lo = max(0, j // 2 - 2)
            P = rows[b_lo]                                  # oracle powers, half-bin indices 2 b_lo .. 2 b_lo + 9
            k = j - 2 * b_lo
            pr = P[k]
            tol = H.POWER_TOL * max(1.0, pr)
            assert abs(p - pr) <= tol, (c, pr)
            worst = max(worst, abs(p - pr) / max(1.0, pr))
            assert pr > thr - 2 * tol, (c, pr)
            left = P[k - 1] if k >= 1 else -np.inf
            right = P[k + 1] if j + 1 < 2 * cfg.nbins else -np.inf
            assert pr - left > -2e-3 * pr and pr - right > -2e-3 * pr, (c, left, pr, right)
    return worst


@pytest.mark.parametrize("idx", [3, 4])
def test_every_full_size_candidate_against_oracle(idx):
    """BASELINE.json north_star: "candidate (r,z,w) indices must match ... on all five configs": ALL records the
    full-size search returns (the launch configuration bench.py times), not only those near the injections."""
    cfg, X, plan, d_spec = _setup(idx)
    cands, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, cfg.threshold))
    assert n == cands.size and n > 0 and plan.work_counters()[2] == 0
    assert len({(c["j"], c["iz"], c["iw"]) for c in cands}) == n
    _verify_every_candidate(cfg, X, cands, cfg.threshold)
    # config 4 also through the library's own choice of segment length (4096, the two-pass kernel): same records
    if idx == 4:
        plan0 = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, 0)
        plan0.templates()
        c0, n0 = binding.candidates_to_numpy(*plan0.search_candidates(d_spec, cfg.threshold))
        key = lambda a: [(int(c["iw"]), int(c["iz"]), int(c["j"])) for c in a]
        far = lambda a: [k for k, c in zip(key(a), a) if c["power"] > 1.05 * cfg.threshold]
        assert far(c0) == far(cands)
        _verify_every_candidate(cfg, X, c0, cfg.threshold)


def test_config5_stage_tops_against_oracle_neighbourhoods():
    """Config 5: every stage top the full-size harmonic search returns, checked on ITS OWN neighbourhood: the sum at the
    point and at its 26 neighbours in (j, iz, iw) from oracle powers; nothing there beats it beyond tolerance."""
    cfg, X, plan, d_spec = _setup(5)
    thr = (25.0, 35.0, 50.0, 75.0)
    top = plan.harmonic_sum(d_spec, (1, 2, 4, 8), thr)
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    cz, cw = (zs.size - 1) // 2, (ws.size - 1) // 2
    tmpl, rows = {}, {}

    def Pref(j, a, b):
        if (a, b) not in tmpl:
            tmpl[(a, b)] = orc.template(float(zs[a + cz]), float(ws[b + cw]))
        blk = (j // 2) // 16
        if (a, b, blk) not in rows:
            rows[(a, b, blk)] = orc.power_row(X, float(zs[a + cz]), float(ws[b + cw]), blk * 16, 16, tmpl=tmpl[(a, b)])
        return rows[(a, b, blk)][j - 32 * blk]

    for s, h in enumerate((1, 2, 4, 8)):
        rec = top[s]
        assert rec["j"] >= 0 and rec["power"] > thr[s]
        j0, a0, b0 = int(rec["j"]), int(rec["iz"]) - cz, int(rec["iw"]) - cw
        s_at = orc.harmonic_sum_point(Pref, j0, a0, b0, h)
        tol = H.POWER_TOL * (h + s_at)
        assert abs(rec["power"] - s_at) <= tol, (h, rec, s_at)
        S_gpu = plan.harmonic_plane(d_spec, h, j0 // 2 - 1, 3, max(0, a0 + cz - 1), min(cfg.nz, a0 + cz + 2) - max(0, a0 + cz - 1),
                                    max(0, b0 + cw - 1), min(cfg.nw, b0 + cw + 2) - max(0, b0 + cw - 1)).cpu().numpy()
        assert S_gpu.max() <= rec["power"]                         # the GPU's own plane: nothing around beats its top
        for da in (-1, 0, 1):
            for db in (-1, 0, 1):
                if not (0 <= a0 + da + cz < cfg.nz and 0 <= b0 + db + cw < cfg.nw):
                    continue
                for dj in (-1, 0, 1):
                    ref = orc.harmonic_sum_point(Pref, j0 + dj, a0 + da, b0 + db, h)
                    assert ref <= s_at + 2 * tol, (h, rec, (dj, da, db), ref, s_at)


# ------------------------------------------------------------------------------------------------ the PRUNE instantiation
class _Cfg:
    def __init__(self, nbins, zmax, dz, wmax, dw):
        self.nbins, self.zmax, self.dz, self.wmax, self.dw = nbins, zmax, dz, wmax, dw


@pytest.mark.parametrize("nbins", [100, 3579, 3581, 9000])
@pytest.mark.parametrize("dz,dw,nclasses", [(2.0, 20.0, 16), (20.0, 100.0, 1)])
def test_wide_grid_low_threshold_seams_and_edges(nbins, dz, dw, nclasses):
    """The zmax 200 / wmax 600 grid (hw_max = 258) on spectra shorter than a segment, one bin either side of one step
    (3580) and several ragged segments, threshold 5: sampled plane rows and ALL candidates of those rows (seams and both
    spectrum edges included) against the oracle.  dz 2 / dw 20 is the headline grid: candidate mode runs on the 16
    overlap classes (k_search64<cand, PRUNE = false>, every class with its own step and seams), plane mode on the
    PRUNE = true instantiation.  dz 20 / dw 100 (273 templates: one class) keeps the candidate-mode PRUNE = true
    instantiation (hw >= 256 in every job) under the same test."""
    X = synth.random_spectrum(nbins, 2000 + nbins)
    plan = binding.Plan(nbins, 200, dz, 600, dw, 2, 4096)
    assert plan.info.hw_max == 258 and plan.info.nclasses == nclasses
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    zs, ws = orc.grid_values(200, dz), orc.grid_values(600, dw)
    nz1, nw1 = zs.size - 1, ws.size - 1
    rows = sorted({(0, 0), (nz1, nw1), (nz1 // 2, nw1 // 2), (37 * nz1 // 200, 55 * nw1 // 60), (170 * nz1 // 200, 3 * nw1 // 60),
                   (nz1, 0), (0, nw1), (nz1 // 2 + 1, nw1 // 2 + 1)})
    ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], 0, nbins)
    for (iz, iw), r in zip(rows, ref):
        P = plan.search_plane(d_spec, 0, nbins, iz, 1, iw, 1).cpu().numpy()[0, 0]
        H.assert_power_close(P, r, f"nbins={nbins} row {(iz, iw)}")
    thr = 5.0
    cands, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, thr, max_cands=1 << 22))
    assert n == cands.size and plan.work_counters()[2] == 0 and plan.work_counters()[1] > 0
    zs_l, ws_l = list(zs), list(ws)
    tot_m = tot_s = 0
    for (iz, iw), r in zip(rows, ref):
        rj, rp, rm = orc.row_candidates(r, thr)
        sel = (cands["iz"] == iz) & (cands["iw"] == iw)
        m, s = H.compare_row_candidates(cands["j"][sel], cands["power"][sel], rj, rp, rm, r, 0, thr)
        tot_m += m
        tot_s += s
    assert tot_m == tot_s and (tot_s > 0 or nbins < 1000)
    assert cands["j"].min() >= 0 and cands["j"].max() <= 2 * nbins - 1
    # the candidate list agrees with the local-max rule applied to the plane the same kernel family writes
    z0, zc, w0, wc = 9 * nz1 // 20, min(20, zs.size - 9 * nz1 // 20), 5 * nw1 // 12, min(10, ws.size - 5 * nw1 // 12)
    box = plan.search_plane(d_spec, 0, nbins, z0, zc, w0, wc)
    neg = torch.full_like(box[..., :1], -float("inf"))
    left, right = torch.cat((neg, box[..., :-1]), -1), torch.cat((box[..., 1:], neg), -1)
    want = int(((box > thr) & (box > left) & (box >= right)).sum().item())
    got = int(((cands["iz"] >= z0) & (cands["iz"] < z0 + zc) & (cands["iw"] >= w0) & (cands["iw"] < w0 + wc)).sum())
    assert abs(got - want) <= max(2, want // 2000)       # (plane and candidate powers differ in the last bit where the segmentations differ)


def test_config4_plane_rows_at_seg_len_8192():
    """BASELINE.json configs[3] at its specified seg_len 8192: 16 random (z,w) rows x a 20000-bin range vs the oracle."""
    cfg, X, plan, d_spec = _setup(4)
    assert plan.info.seg_len == 8192
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    rng = np.random.default_rng(44)
    rows = sorted({(int(rng.integers(0, zs.size)), int(rng.integers(0, ws.size))) for _ in range(16)})
    b_cnt = 20000
    b_lo = int(rng.integers(0, cfg.nbins - b_cnt))
    ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], b_lo, b_cnt)
    for (iz, iw), r in zip(rows, ref):
        P = plan.search_plane(d_spec, b_lo, b_cnt, iz, 1, iw, 1).cpu().numpy()[0, 0]
        H.assert_power_close(P, r, f"config 4 row {(iz, iw)}")


# ------------------------------------------------------------------------------------------------ seams
def _rule_count(box, thr):
    neg = torch.full_like(box[..., :1], -float("inf"))
    left, right = torch.cat((neg, box[..., :-1]), -1), torch.cat((box[..., 1:], neg), -1)
    return int(((box > thr) & (box > left) & (box >= right)).sum().item())


def test_long_seam_list_hash_path_and_overflow_is_never_silent():
    """Threshold 0 on 2^18 bins x 147 templates: every point is above threshold, ~2.4 M seam records.
    (a) with room for them (a larger d_work) the hash-table path settles them: the candidate count equals the rule applied
        to the plane; (b) with the default d_work (2^20 records) the list overflows: the call reports UINT64_MAX in
        *d_count, candidates_to_numpy raises and the host entry point returns JERK_EOVERFLOW."""
    nbins = 1 << 18
    X = synth.random_spectrum(nbins, 77)
    d_spec = binding.spectrum_to_device(X)
    big = binding.Plan(nbins, 20, 2, 60, 20, 2, 4096, extra_seams=3_000_000)
    big.templates()
    d_c, d_n = big.search_candidates(d_spec, 0.0, max_cands=1 << 16)
    ctr = big.work_counters()
    assert ctr[2] == 0 and ctr[1] > (1 << 21)
    plane = big.search_plane(d_spec, 0, nbins)
    assert int(d_n.item()) == _rule_count(plane, 0.0)
    del plane
    small = binding.Plan(nbins, 20, 2, 60, 20, 2, 4096)
    small.bank = big.bank
    lib = binding.load_library()
    assert lib.jerk_templates(small._h, C.c_void_p(small.bank.data_ptr()), int(small.info.bank_bytes), None) == 0
    d_c, d_n = small.search_candidates(d_spec, 0.0, max_cands=1 << 16)
    assert small.work_counters()[2] == 1
    assert int(d_n.item()) & binding.SEAM_OVERFLOW == binding.SEAM_OVERFLOW
    with pytest.raises(binding.JerkError) as e:
        binding.candidates_to_numpy(d_c, d_n)
    assert e.value.status == binding.JERK_EOVERFLOW
    h_spec = torch.from_numpy(np.ascontiguousarray(X).view(np.float32).reshape(-1, 2)).pin_memory()
    h_c = torch.empty((1 << 16) * 16, dtype=torch.uint8).pin_memory()
    h_n = torch.zeros(1, dtype=torch.int64).pin_memory()
    d_spec2 = torch.empty_like(d_spec)
    with pytest.raises(binding.JerkError) as e:
        small.search_candidates_host(h_spec, 0.0, h_c, h_n, d_spec2, d_c, d_n)
    assert e.value.status == binding.JERK_EOVERFLOW
    # count > max_cands is JERK_EOVERFLOW from the host entry point as well (records still copied)
    with pytest.raises(binding.JerkError) as e:
        big.search_candidates_host(h_spec, 12.0, h_c[:16 * 10], h_n, d_spec2, d_c[:16 * 10], d_n)
    assert e.value.status == binding.JERK_EOVERFLOW and int(h_n.item()) > 10


# ------------------------------------------------------------------------------------------------ batched spectra (N3)
def test_batched_search_equals_single_searches():
    """jerk_search_candidates_batch: B spectra against one bank in one launch (per 32) == B single searches, record for
    record (bit-exact), including the seam-settled ones; one member is the oracle-checked config-1 spectrum."""
    cfg = synth.config(1)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, 4096)
    plan.templates()
    nspec = 35                                             # two launches: 32 + 3
    specs = [binding.spectrum_to_device(synth.make_spectrum(synth.config(1), trial=b)) for b in range(nspec)]
    thr = 7.0
    d_c, d_n = plan.search_candidates_batch(specs, thr, max_cands=1 << 16)
    counts = d_n.cpu().numpy()
    for b in range(nspec):
        got, n = binding.candidates_to_numpy(d_c[b], d_n[b:b + 1])
        ref, k = binding.candidates_to_numpy(*plan.search_candidates(specs[b], thr, max_cands=1 << 16))
        assert n == k == counts[b] and n > 100
        assert got.tobytes() == ref.tobytes(), b
    # member 0 is the parity-pinned config-1 spectrum: its strongest record is the injection at the oracle's grid point
    got, _ = binding.candidates_to_numpy(d_c[0], d_n[0:1])
    best = got[np.argmax(got["power"])]
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    assert (zs[best["iz"]], ws[best["iw"]]) == (10.0, 40.0) and best["j"] / 2.0 in (5000.0, 5000.5)
    ref_row = orc.power_row(synth.make_spectrum(synth.config(1)), 10.0, 40.0, 4990, 20)
    assert abs(best["power"] - ref_row.max()) <= 1e-3 * ref_row.max()


# ------------------------------------------------------------------------------------------------ bank shards (8(e))
@pytest.mark.parametrize("idx,world,seg_len", [(1, 3, 1024), (1, 8, 4096), (2, 4, 4096), (1, 150, 1024)])
def test_bank_shards_and_flat_template_ranges(idx, world, seg_len):
    """Every "rank" builds ONLY its flat range of templates (jerk_templates_range) and searches it
    (jerk_search_candidates_templates): the union equals the whole-grid search of a full bank, record for record; a
    search outside the built range is refused (JERK_ESTATE).  world 150 > 147 templates: the last ranks hold an empty
    range (tables only) and return no candidates instead of failing before the collectives of a sharded search."""
    cfg, X, plan, d_spec = _setup(idx, seg_len)
    thr = 8.0 if idx == 1 else cfg.threshold
    full, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, thr))
    T = plan.info.ntemplates
    parts = []
    for r in range(world):
        lo, cnt = shard.template_range(T, world, r)
        p = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, seg_len)
        bank = p.templates_range(lo, cnt)
        assert bank.numel() < plan.info.bank_bytes // world + 2 * plan.info.seg_len * 16 + (1 << 20)
        c, k = binding.candidates_to_numpy(*p.search_candidates_templates(d_spec, thr, lo, cnt))
        ti = c["iw"].astype(np.int64) * cfg.nz + c["iz"]
        assert k == c.size and np.all((ti >= lo) & (ti < lo + cnt))
        assert cnt > 0 or k == 0
        parts.append(c)
        if r == 0 and world > 1:
            with pytest.raises(binding.JerkError) as e:
                p.search_candidates(d_spec, thr)
            assert e.value.status == binding.JERK_ESTATE
    merged = np.sort(np.concatenate(parts), order=["iw", "iz", "j"])
    assert merged.tobytes() == np.sort(full, order=["iw", "iz", "j"]).tobytes()


# ------------------------------------------------------------------------------------------------ numbetween = 1 (N4)
@pytest.mark.parametrize("seg_len,zmax,wmax", [(4096, 50.0, 0.0), (1024, 20.0, 60.0), (4096, 200.0, 600.0), (8192, 20.0, 60.0)])
def test_numbetween_one(seg_len, zmax, wmax):
    """numbetween = 1 (FDAS-only mode with numbetween options; also on jerk grids): the plane has one
    float per bin and equals the oracle's phase-0 rows; candidates follow the same rule along integer bins."""
    nbins = 9000
    X = synth.random_spectrum(nbins, 31).astype(np.complex128)
    z0, w0, r0 = (36.0, 0.0, 4000) if wmax == 0 else (10.0, 40.0, 4000)
    c, hw, lat = orc.template(z0, w0)
    m, taps = orc.phase_taps(c, hw, lat, 0)
    X[r0 + m] += 8.0 * taps
    X = X.astype(np.complex64)
    dz, dw = (2.0, 20.0) if zmax < 200 else (20.0, 100.0)
    plan = binding.Plan(nbins, zmax, dz, wmax, dw, 1, seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    info = plan.info
    zs, ws = orc.grid_values(zmax, dz), orc.grid_values(wmax, dw)
    out = torch.empty((info.nw, info.nz, nbins), dtype=torch.float32, device="cuda")
    plan.search_plane(d_spec, 0, nbins, out=out)
    P = out.cpu().numpy()
    rng = np.random.default_rng(5)
    rows = {(int(rng.integers(0, info.nz)), int(rng.integers(0, info.nw))) for _ in range(5)} | {(0, 0), (info.nz - 1, info.nw - 1)}
    if wmax == 0 or zmax < 200:
        rows.add((list(zs).index(z0), list(ws).index(w0)))
    thr = 6.0
    cands, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, thr))
    assert n == cands.size and cands["j"].max() < nbins
    for iz, iw in sorted(rows):
        ref = orc.power_row(X, float(zs[iz]), float(ws[iw]))[0::2]                  # phase-0 points of the oracle row
        H.assert_power_close(P[iw, iz], ref, f"numbetween=1 row {(iz, iw)}")
        rj, rp, rm = orc.row_candidates(ref, thr)
        sel = (cands["iz"] == iz) & (cands["iw"] == iw)
        mm, ss = H.compare_row_candidates(cands["j"][sel], cands["power"][sel], rj, rp, rm, ref, 0, thr)
        assert mm == ss
    # the two definitions of the oracle agree (section I written out per tap vs the phase-0 slice) on a short range
    assert np.abs(orc.power_row_nb1(X, float(zs[0]), float(ws[0]), 3990, 12) - orc.power_row(X, float(zs[0]), float(ws[0]), 3990, 12)[0::2]).max() < 1e-9
    # whole-list count == the rule on the plane; the injected signal is the strongest record at its grid point
    assert n == _rule_count(out, thr)
    if wmax == 0 or zmax < 200:
        best = cands[np.argmax(cands["power"])]
        assert (zs[best["iz"]], ws[best["iw"]], int(best["j"])) == (z0, w0, r0)
    with pytest.raises(binding.JerkError):
        plan.harmonic_sum(d_spec)


# ------------------------------------------------------------------------------------------------ strong scaling under NCCL
def test_strong_scaling_two_ranks_nccl():
    """the template-sharded search on TWO GPUs under NCCL (bench.py --scaling strong through torchrun):
    every rank builds and searches half of the bank, the gathered list must equal rank 0's whole-grid search.  Skipped
    when fewer than two GPUs are visible (nothing in this build run has more than one)."""
    import json
    import os
    import subprocess
    import sys
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", "2", "--master-addr", "127.0.0.1",
           "--master-port", "29517", os.path.join(root, "bench.py"), "--gpus", "2", "--scaling", "strong", "--config", "2",
           "--steps", "1", "--warmup", "3"]
    res = subprocess.run(cmd, capture_output=True, text=True, timeout=900, cwd=root)
    assert res.returncode == 0, res.stderr[-2000:]
    line = json.loads([l for l in res.stdout.splitlines() if l.startswith("{")][-1])
    assert line["n_gpus"] == 2 and line["scaling"] == "strong"
    assert line["gathered_equals_whole_grid_search"] is True


# ------------------------------------------------------------------------------------------------ out-of-bounds canaries
def _padded(nbytes, device="cuda", pad=1 << 16):
    """A uint8 view of `nbytes` bytes (256-byte aligned) inside a buffer with 64 KB canary bands on both sides."""
    full = torch.full((nbytes + 2 * pad + 256,), 0xA5, dtype=torch.uint8, device=device)
    off = pad + (-(full.data_ptr() + pad)) % 256
    return full, full[off:off + nbytes], off


def _canaries_intact(full, off, nbytes):
    return bool((full[:off] == 0xA5).all().item()) and bool((full[off + nbytes:] == 0xA5).all().item())


@pytest.mark.parametrize("seg_len,zmax,wmax", [(4096, 60.0, 180.0), (1024, 20.0, 60.0)])
def test_no_write_outside_caller_buffers(seg_len, zmax, wmax):
    """compute-sanitizer is closed on this pool, so the memcheck substitute is explicit: every caller-owned buffer the
    library writes (bank, d_work, candidates, count, plane, harmonic scratch, stage tops) sits between 64 KB canary bands
    that must be untouched after bank build, candidate search (low threshold: seams, overlap classes for the first grid),
    a plane box that starts and ends inside segments, and a harmonic-summed search with chunking."""
    nbins = 23456
    X = synth.random_spectrum(nbins, 909)
    plan = binding.Plan(nbins, zmax, 2, wmax, 20, 2, seg_len)
    lib = binding.load_library()
    bank_full, plan.bank, bank_off = _padded(int(plan.info.bank_bytes))
    assert lib.jerk_templates(plan._h, C.c_void_p(plan.bank.data_ptr()), int(plan.info.bank_bytes), None) == 0
    work_full, plan.work, work_off = _padded(int(plan.info.work_bytes))
    d_spec = binding.spectrum_to_device(X)
    max_cands = 5000                                        # smaller than the number of candidates: the excess must be dropped, not written
    cand_full, d_cands, cand_off = _padded(max_cands * 16)
    cnt_full, d_cnt8, cnt_off = _padded(8)
    d_count = d_cnt8.view(torch.int64)
    plan.search_candidates(d_spec, 4.0, max_cands=max_cands, d_cands=d_cands, d_count=d_count)
    assert int(d_count.item()) > max_cands
    r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt = 777, 9001, 3, 5, 1, 2
    plane_full, plane8, plane_off = _padded(iw_cnt * iz_cnt * 2 * r_cnt * 4)
    out = plane8.view(torch.float32).view(iw_cnt, iz_cnt, 2 * r_cnt)
    plan.search_plane(d_spec, r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt, out=out)
    nscr = int(plan.harmonic_scratch_bytes()) // 3          # a third of the default: several r-chunks
    nscr -= nscr % 256
    scr_full, plan.scratch, scr_off = _padded(nscr)
    top = plan.harmonic_sum(d_spec, (1, 2, 4, 8), (8.0, 12.0, 18.0, 28.0), scratch_bytes=nscr)
    torch.cuda.synchronize()
    assert (top["j"] >= 0).all()
    for name, full, off, n in (("bank", bank_full, bank_off, int(plan.info.bank_bytes)), ("work", work_full, work_off, int(plan.info.work_bytes)),
                               ("cands", cand_full, cand_off, max_cands * 16), ("count", cnt_full, cnt_off, 8),
                               ("plane", plane_full, plane_off, plane8.numel()), ("scratch", scr_full, scr_off, nscr)):
        assert _canaries_intact(full, off, n), f"write outside the {name} buffer"
    assert np.isfinite(out.cpu().numpy()).all()


# ------------------------------------------------------------------------------------------------ measurement aids
def test_probes_report_sane_numbers():
    """bench.py's bench_probe_fma / bench_probe_issue (bench_probes.cu, outside the library; the denominators and the issue-slot model of DESIGN.md 6.2): a packed FP32
    instruction takes about two scheduler cycles, no companion instruction is free, the FFMA probe is near the nominal peak."""
    import bench
    p = bench.probe_issue_slots(iters=500)
    assert 1.9 < p["packed_fma_cycles"] < 2.3
    assert all(c > 0.5 for c in p["companion_cost_cycles"].values())
    tf = bench.probe_fp32_tflops(iters=1 << 13, reps=3)
    assert 50.0 < tf < 80.0


def test_cufft_comparator_agrees_with_the_fused_plane():
    """SURVEY.md 8(f) N4 / PAPER.md:45: the unfused cuFFT pipeline of bench.py (library calls only: torch.fft + elementwise
    kernels on this library's bank) gives the powers of jerk_search_plane to 1e-3 * max(1, P) -- on config 2 (the whole
    1 GB block path: 512 template-phases x 64 segments) for three templates, all segments of the block, both phases."""
    import bench
    row = bench.cufft_unfused_block(synth.config(2), warmup=1, steps=1, check_templates=(0, 100, 255))
    assert row["units_per_block"] == 512 * 64
    assert row["max_rel_diff_vs_fused_plane"] < 1e-3, row
    assert row["extrapolated_ms_per_search"] > 0


def test_config3_candidate_list_is_complete_on_random_windows():
    """Completeness at full size (reading S11): the tests above check every RETURNED record; here the
    oracle decides what must be there.  Config 3 at threshold 9 (1.1e7 candidates: the rare path, the seam records and the
    hash table of the full-size launch are all busy; threshold 12 would leave ~0.2 candidates per window), 64 random (z,w)
    rows x a 20 000-bin window -- one window at bin 0, one ending at nbins - 1, the rest
    at random places (each spans five or more segments of its overlap class): the GPU's records of that row and window
    and orc.row_candidates agree as sets, up to the near-threshold / near-tie allowances of compare_row_candidates."""
    cfg, X, plan0, d_spec = _setup(3)
    thr = 9.0
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len, extra_seams=1 << 24)
    plan.bank = plan0.bank                 # the same caller-owned bank (rebuilt in place with identical contents)
    plan.templates()
    max_c = 1 << 24
    d_c, d_n = plan.search_candidates(d_spec, thr, max_cands=max_c)
    n = int(d_n.item())
    assert 5e6 < n <= max_c, n               # neither the candidate buffer nor the seam records overflowed (-1)
    cands = d_c[: n * 16].cpu().numpy().view(binding.CAND_DTYPE)
    zs, ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
    rng = np.random.default_rng(1911)
    wlen = 20000
    jobs, keys = [], []
    for k in range(64):
        iz, iw = int(rng.integers(0, cfg.nz)), int(rng.integers(0, cfg.nw))
        if k == 0:
            iz, iw = 0, 0                                   # widest templates (first class boundary), window at the start
        if k == 1:
            iz, iw = cfg.nz - 1, cfg.nw - 1
        b_lo = 0 if k % 8 == 0 else (cfg.nbins - wlen if k % 8 == 1 else int(rng.integers(0, cfg.nbins - wlen)))
        jobs.append((zs[iz], ws[iw], b_lo, wlen))
        keys.append((iz, iw, b_lo))
    refs = H.oracle_candidates_for_rows(X, jobs, thr)
    ti_all = cands["iw"].astype(np.int64) * cfg.nz + cands["iz"]
    cands = cands[np.isin(ti_all, [iw * cfg.nz + iz for iz, iw, _ in keys])]      # the 64 rows only, before sorting
    order = np.lexsort((cands["j"], cands["iz"], cands["iw"]))
    cs = cands[order]
    ti_sorted = cs["iw"].astype(np.int64) * cfg.nz + cs["iz"]
    total_ref = total_strong = 0
    for (iz, iw, b_lo), (rj, rp, rm, P_ref, j0) in zip(keys, refs):
        a, b = np.searchsorted(ti_sorted, [iw * cfg.nz + iz, iw * cfg.nz + iz + 1])
        row = cs[a:b]
        sel = (row["j"] >= 2 * b_lo) & (row["j"] < 2 * (b_lo + wlen))
        if b_lo > 0:
            sel &= row["j"] > j0                            # the window's artificial edges, as in oracle_candidates_for_row
        if b_lo + wlen < cfg.nbins:
            sel &= row["j"] < j0 + P_ref.size - 1
        matched, strong = H.compare_row_candidates(row["j"][sel], row["power"][sel], rj, rp, rm, P_ref, j0, thr)
        assert matched == strong
        total_ref += rj.size
        total_strong += strong
    assert total_ref > 100 and total_strong > 40, (total_ref, total_strong)
