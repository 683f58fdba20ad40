"""GPU parity tests: the CUDA path (through the C-ABI) against the oracle, element by element on the same
seeded inputs (BASELINE.json north_star: |P_gpu - P_ref| <= 1e-3*max(1,P_ref); candidate indices bit-exact
for candidates more than 5 % above threshold; injected signals recovered at the exact grid point)."""
import ctypes as C

import numpy as np
import pytest

from oracle import jerk_oracle as orc
from paper_1911_01353_b200 import binding, build
import workloads as synth
from tests import helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    binding.load_library()


_cache = {}


def _setup(idx):
    """(cfg, X complex64, plan with bank built, d_spec) for BASELINE config idx, cached per module."""
    if idx not in _cache:
        cfg = synth.config(idx)
        X = synth.make_spectrum(cfg)
        plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
        plan.templates()
        d_spec = binding.spectrum_to_device(X)
        torch.cuda.synchronize()
        _cache[idx] = (cfg, X, plan, d_spec)
    return _cache[idx]


def _grid(cfg):
    return orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)


# ------------------------------------------------------------------------------------------------ a-1 template bank
@pytest.mark.parametrize("zw", [(0, 0), (2, 0), (10, 40), (-20, 60), (200, 600), (200, -600), (-150, 600), (50, -600), (0, 600)])
def test_template_taps_match_oracle(zw):
    cfg = synth.config(3)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    zs, ws = _grid(cfg)
    iz, iw = list(zs).index(zw[0]), list(ws).index(zw[1])
    taps = plan.templates_taps(iz, iw).cpu().numpy()
    c, hw, lat = orc.template(float(zw[0]), float(zw[1]))
    assert (c, hw) == plan.template_geometry(iz, iw)
    got = taps[:, 0] + 1j * taps[:, 1]
    assert np.abs(got - lat).max() < 1e-6      # fp32 storage of an fp64 quadrature


# ------------------------------------------------------------------------------------------------ config 1: everything
def test_config1_full_plane():
    cfg, X, plan, d_spec = _setup(1)
    P = plan.search_plane(d_spec, 0, cfg.nbins).cpu().numpy()
    ref = orc.plane(X, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw)
    assert P.shape == ref.shape == (7, 21, 65536)
    H.assert_power_close(P, ref, "config 1 plane")
    # injected signal recovered at the exact grid point the oracle finds (reading S18)
    assert np.unravel_index(np.argmax(P), P.shape) == np.unravel_index(np.argmax(ref), ref.shape)
    iw, iz, j = np.unravel_index(np.argmax(ref), ref.shape)
    zs, ws = _grid(cfg)
    assert (zs[iz], ws[iw]) == (10.0, 40.0) and j / 2.0 in (5000.0, 5000.5)


def _check_candidates(cfg, X, cands, rows, b_lo, b_cnt, thr):
    zs, ws = _grid(cfg)
    tot_m = tot_s = 0
    for iz, iw in rows:
        rj, rp, rm, Pref, j0 = H.oracle_candidates_for_row(X, float(zs[iz]), float(ws[iw]), thr, b_lo, b_cnt, cfg.nbins)
        sel = (cands["iz"] == iz) & (cands["iw"] == iw) & (cands["j"] >= 2 * b_lo) & (cands["j"] < 2 * (b_lo + b_cnt))
        if b_lo > 0:
            sel &= cands["j"] > 2 * max(0, b_lo - 1)
        if b_lo + b_cnt < cfg.nbins:
            sel &= cands["j"] < 2 * min(cfg.nbins, b_lo + b_cnt + 1) - 1
        m, s = H.compare_row_candidates(cands["j"][sel], cands["power"][sel], rj, rp, rm, Pref, j0, thr)
        tot_m += m
        tot_s += s
    return tot_m, tot_s


def test_config1_candidates_all_rows():
    cfg, X, plan, d_spec = _setup(1)
    d_c, d_n = plan.search_candidates(d_spec, cfg.threshold)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert n == cands.size and n > 0
    assert np.all(cands["flags"] == 0)
    assert len({(c["j"], c["iz"], c["iw"]) for c in cands}) == n          # no duplicates
    rows = [(iz, iw) for iw in range(7) for iz in range(21)]
    m, s = _check_candidates(cfg, X, cands, rows, 0, cfg.nbins, cfg.threshold)
    assert m == s and s > 0
    best = cands[np.argmax(cands["power"])]
    zs, ws = _grid(cfg)
    assert (zs[best["iz"]], ws[best["iw"]]) == (10.0, 40.0) and best["j"] / 2.0 in (5000.0, 5000.5)


def test_config1_low_threshold_seams():
    """Threshold 6: ~25k candidates, hundreds of them on warp/segment seams -> exercises the resolve kernel."""
    cfg, X, plan, d_spec = _setup(1)
    thr = 6.0
    d_c, d_n = plan.search_candidates(d_spec, thr, max_cands=1 << 18)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    ctr = plan.work_counters()
    assert ctr[1] > 0 and ctr[2] == 0 and ctr[3] > 0                        # seam records seen, no overflow, some resolved
    assert len({(c["j"], c["iz"], c["iw"]) for c in cands}) == n
    rows = [(iz, iw) for iw in range(7) for iz in range(21)]
    m, s = _check_candidates(cfg, X, cands, rows, 0, cfg.nbins, thr)
    assert m == s and s > 1000
    # exact set equality away from near-ties / near-threshold powers
    ref = orc.plane(X, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw)
    nref = 0
    for iw in range(7):
        for iz in range(21):
            j, p, mg = orc.row_candidates(ref[iw, iz], thr)
            nref += j.size
    assert abs(nref - n) <= max(5, int(2e-3 * nref))


def test_candidate_overflow_is_reported():
    cfg, X, plan, d_spec = _setup(1)
    d_c, d_n = plan.search_candidates(d_spec, 6.0, max_cands=100)
    assert int(d_n.item()) > 100                                            # count keeps counting, excess dropped
    arr = d_c.cpu().numpy().view(binding.CAND_DTYPE)
    assert arr.size == 100 and np.all(arr["power"] > 6.0)


# ------------------------------------------------------------------------------------------------ invariances (P8, P9)
def test_seg_len_invariance_and_edges():
    """Same plane for seg_len 1024/2048/4096/8192 (several tiles + ragged tail), spectrum edges included."""
    nbins = 9000
    X = synth.random_spectrum(nbins, 17)
    d_spec = binding.spectrum_to_device(X)
    zs, ws = orc.grid_values(20, 2), orc.grid_values(60, 20)
    rows = [(0, 0), (20, 6), (10, 3), (3, 5), (17, 1)]
    ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], 0, nbins)
    for L in (1024, 2048, 4096, 8192):
        plan = binding.Plan(nbins, 20, 2, 60, 20, 2, L)
        plan.templates()
        P = plan.search_plane(d_spec, 0, nbins).cpu().numpy()
        for (iz, iw), r in zip(rows, ref):
            H.assert_power_close(P[iw, iz], r, f"L={L} row {(iz, iw)}")


def test_plane_subrange_equals_full_plane():
    cfg, X, plan, d_spec = _setup(1)
    full = plan.search_plane(d_spec, 0, cfg.nbins).cpu().numpy()
    for (r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt) in [(0, 1, 0, 1, 0, 1), (4990, 37, 3, 5, 2, 3), (32700, 68, 20, 1, 6, 1),
                                                        (0, 3000, 0, 21, 0, 7), (957, 2, 10, 2, 3, 1)]:
        sub = plan.search_plane(d_spec, r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt).cpu().numpy()
        want = full[iw_lo:iw_lo + iw_cnt, iz_lo:iz_lo + iz_cnt, 2 * r_lo:2 * (r_lo + r_cnt)]
        assert np.array_equal(sub, want)


def test_shift_invariance_gpu():
    nbins, k = 6000, 41
    X = synth.random_spectrum(nbins, 23)
    Xs = np.concatenate((np.zeros(k, dtype=X.dtype), X))[:nbins]
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, 1024)
    plan.templates()
    a = plan.search_plane(binding.spectrum_to_device(X), 1000, 3000).cpu().numpy()
    b = plan.search_plane(binding.spectrum_to_device(Xs), 1000 + k, 3000).cpu().numpy()
    assert np.abs(a - b).max() <= 1e-3 * max(1.0, a.max())


def test_tiny_spectrum_shorter_than_a_segment():
    nbins = 100
    X = synth.random_spectrum(nbins, 5)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, 1024)
    plan.templates()
    P = plan.search_plane(binding.spectrum_to_device(X), 0, nbins).cpu().numpy()
    ref = orc.plane(X, 20, 2, 60, 20)
    H.assert_power_close(P, ref, "nbins=100")


def test_empty_ranges_and_errors():
    cfg, X, plan, d_spec = _setup(1)
    out = plan.search_plane(d_spec, 10, 0)                               # empty r range: no-op
    assert out.numel() == 0
    with pytest.raises(binding.JerkError) as e:
        plan.search_plane(d_spec, cfg.nbins - 5, 10)                     # range past the spectrum
    assert e.value.status == binding.JERK_EINVAL
    small = torch.empty(16, dtype=torch.float32, device="cuda")
    with pytest.raises(binding.JerkError) as e:
        plan.search_plane(d_spec, 0, 100, out=small)                     # plane buffer too small
    assert e.value.status == binding.JERK_ENOMEM
    lib = binding.load_library()
    rc = lib.jerk_search_candidates(plan._h, C.c_void_p(d_spec.data_ptr() + 8), 20.0, C.c_void_p(small.data_ptr()), 1,
                                    C.c_void_p(small.data_ptr()), C.c_void_p(plan.work.data_ptr()), plan.work.numel(), None)
    assert rc == binding.JERK_EINVAL                                     # misaligned spectrum pointer


# ------------------------------------------------------------------------------------------------ configs 2-4: sampled rows
def _rows_around(cfg, signals, dz_steps=1, dw_steps=1):
    zs, ws = _grid(cfg)
    rows = set()
    for (r0, z0, w0, p) in signals:
        iz0, iw0 = list(zs).index(z0), list(ws).index(w0)
        for a in range(-dz_steps, dz_steps + 1):
            for b in range(-dw_steps, dw_steps + 1):
                if 0 <= iz0 + a < zs.size and 0 <= iw0 + b < ws.size:
                    rows.add((iz0 + a, iw0 + b))
    return sorted(rows)


def _sampled_plane_check(idx, n_random_rows, b_cnt, seed):
    cfg, X, plan, d_spec = _setup(idx)
    zs, ws = _grid(cfg)
    rng = np.random.default_rng(seed)
    rows = {(int(rng.integers(0, zs.size)), int(rng.integers(0, ws.size))) for _ in range(n_random_rows)}
    rows |= {(0, 0), (zs.size - 1, ws.size - 1), (zs.size - 1, 0), (0, ws.size - 1)}
    rows = sorted(rows)
    b_lo = int(rng.integers(0, cfg.nbins - b_cnt))
    ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], b_lo, b_cnt)
    worst = 0.0
    for (iz, iw), r in zip(rows, ref):
        P = plan.search_plane(d_spec, b_lo, b_cnt, iz, 1, iw, 1).cpu().numpy()[0, 0]
        worst = max(worst, H.assert_power_close(P, r, f"config {idx} row {(iz, iw)}"))
    return worst


def _injection_check(idx, half_range=600):
    """Rows around each injection: plane parity, candidate parity, and recovery at the oracle's grid point."""
    cfg, X, plan, d_spec = _setup(idx)
    zs, ws = _grid(cfg)
    d_c, d_n = plan.search_candidates(d_spec, cfg.threshold)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert n == cands.size and plan.work_counters()[2] == 0
    assert len({(c["j"], c["iz"], c["iw"]) for c in cands}) == n
    tot_m = tot_s = 0
    for sig in cfg.signals:
        r0, z0, w0, p = sig
        rows = _rows_around(cfg, [sig])
        b_lo = max(0, int(r0) - half_range)
        b_cnt = min(cfg.nbins, int(r0) + half_range) - b_lo
        ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], b_lo, b_cnt)
        best_ref = (-1.0, None)
        best_gpu = (-1.0, None)
        for (iz, iw), r in zip(rows, ref):
            P = plan.search_plane(d_spec, b_lo, b_cnt, iz, 1, iw, 1).cpu().numpy()[0, 0]
            H.assert_power_close(P, r, f"config {idx} injection row {(iz, iw)}")
            if r.max() > best_ref[0]:
                best_ref = (float(r.max()), (iz, iw, 2 * b_lo + int(np.argmax(r))))
            if P.max() > best_gpu[0]:
                best_gpu = (float(P.max()), (iz, iw, 2 * b_lo + int(np.argmax(P))))
        assert best_gpu[1] == best_ref[1]                                   # GPU == oracle (readings S18/S19)
        m, s = _check_candidates(cfg, X, cands, rows, b_lo, b_cnt, cfg.threshold)
        tot_m += m
        tot_s += s
        if best_ref[0] > 1.05 * cfg.threshold:
            iz, iw, j = best_ref[1]
            hit = cands[(cands["iz"] == iz) & (cands["iw"] == iw) & (cands["j"] == j)]
            assert hit.size == 1
    assert tot_m == tot_s
    return tot_s


def test_config2_sampled_rows():
    _sampled_plane_check(2, 24, 20000, seed=2)


def test_config2_injections_and_candidates():
    assert _injection_check(2) > 0


def test_config3_sampled_rows():
    """BASELINE.json configs[2]: the oracle spot-checks 64 random (z,w) rows over a 20000-bin range."""
    _sampled_plane_check(3, 64, 20000, seed=3)


def test_config3_injections_and_candidates():
    assert _injection_check(3) > 0


def test_config4_injections_and_candidates():
    """BASELINE.json configs[3]: N = 2^25, seg_len 8192; rows around each injection (two near threshold)."""
    assert _injection_check(4, half_range=400) > 0


# ------------------------------------------------------------------------------------------------ template-box sharding (8(e))
@pytest.mark.gpu
@pytest.mark.parametrize("idx,world,thr", [(1, 2, 8.0), (1, 3, 8.0), (3, 2, 25.0)])
def test_candidates_range_union(idx, world, thr):
    """The union of jerk_search_candidates_range over the template boxes of shard.template_box is, record for record
    (bit-exact j, iz, iw and power), the result of the whole-grid search: the property multi-GPU template sharding rests on."""
    from paper_1911_01353_b200 import shard
    cfg, X, plan, d_spec = _setup(idx)
    d_c, d_n = plan.search_candidates(d_spec, thr)
    full, n = binding.candidates_to_numpy(d_c, d_n)
    assert n == full.size and n > 0
    parts = []
    for r in range(world):
        iz_lo, iz_cnt, iw_lo, iw_cnt = shard.template_box(cfg.nz, cfg.nw, world, r)
        d_c, d_n = plan.search_candidates_range(d_spec, thr, iz_lo, iz_cnt, iw_lo, iw_cnt)
        c, k = binding.candidates_to_numpy(d_c, d_n)
        assert k == c.size
        assert np.all((c["iz"] >= iz_lo) & (c["iz"] < iz_lo + iz_cnt) & (c["iw"] >= iw_lo) & (c["iw"] < iw_lo + iw_cnt))
        parts.append(c)
    merged = np.sort(np.concatenate(parts), order=["iw", "iz", "j"])
    assert np.array_equal(merged, np.sort(full, order=["iw", "iz", "j"]))
    # empty box: count 0, no launch error
    d_c, d_n = plan.search_candidates_range(d_spec, thr, 0, 0, 0, cfg.nw)
    assert int(d_n.item()) == 0


# ------------------------------------------------------------------------------------------------ FDAS-only mode (8(f) N4)
@pytest.mark.gpu
@pytest.mark.parametrize("seg_len", [1024, 4096])
def test_fdas_only_mode_w0(seg_len):
    """wmax = 0: the acceleration-only (FDAS) search the paper extends: one w-row, templates are the
    Fresnel responses; full plane rows and candidates against the oracle."""
    nbins = 40000
    X = synth.random_spectrum(nbins, seed=424242)
    # inject one accelerated signal: X += A * R_{z0,0}(k - r0) (the response itself), amplitude 9
    z0, r0 = 36.0, 20000
    c, hw, lattice = orc.template(z0, 0.0)
    m, p0_taps = orc.phase_taps(c, hw, lattice, 0)
    X = X.astype(np.complex128)
    X[r0 + m] += 9.0 * p0_taps
    X = X.astype(np.complex64)
    plan = binding.Plan(nbins, 50.0, 2.0, 0.0, 20.0, 2, seg_len)
    assert plan.info.nw == 1 and plan.info.nz == 51
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    zs = orc.grid_values(50.0, 2.0)
    b_lo, b_cnt = 19000, 2000
    rows = [0, 7, 25, 43, 50]
    refs = H.oracle_rows(X, [(zs[iz], 0.0) for iz in rows], b_lo, b_cnt)
    for iz, ref in zip(rows, refs):
        P = plan.search_plane(d_spec, b_lo, b_cnt, iz, 1, 0, 1).cpu().numpy()[0, 0]
        H.assert_power_close(P, ref, f"fdas row iz={iz}")
    d_c, d_n = plan.search_candidates(d_spec, 30.0)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    best = cands[np.argmax(cands["power"])]
    assert (zs[best["iz"]], best["iw"], best["j"]) == (z0, 0, 2 * r0)


# ------------------------------------------------------------------------------------------------ run-to-run reproducibility
@pytest.mark.gpu
def test_repeated_searches_are_bit_identical():
    """The work items are handed out dynamically (atomic counter) and every FFT group synchronises through mbarriers and a
    TMA-refilled exchange buffer: a race there would show up as run-to-run differences.  Candidate records (sorted) and
    plane values must be bit-identical over repeated launches (compute-sanitizer is not available on this pool)."""
    cfg, X, plan, d_spec = _setup(3)
    ref = None
    for _ in range(4):
        c, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, cfg.threshold))
        c = np.sort(c, order=["iw", "iz", "j"])
        if ref is None:
            ref = c
        assert n == ref.size and c.tobytes() == ref.tobytes()
    p_ref = None
    for _ in range(3):
        P = plan.search_plane(d_spec, 2_000_000, 40_000, 90, 8, 28, 3).cpu().numpy()
        if p_ref is None:
            p_ref = P
        assert P.tobytes() == p_ref.tobytes()


# ------------------------------------------------------------------------------------------------ k_search64 edge cases
class _Cfg:
    """Minimal stand-in for synth.Config in _check_candidates (grid + nbins)."""
    def __init__(self, nbins, zmax, dz, wmax, dw):
        self.nbins, self.zmax, self.dz, self.wmax, self.dw = nbins, zmax, dz, wmax, dw


@pytest.mark.gpu
@pytest.mark.parametrize("nbins", [100, 3579, 3581, 9000])
def test_seg_len_4096_low_threshold_seams_and_edges(nbins):
    """The two-pass kernel (seg_len 4096) on spectra shorter than a segment, one bin either side of one step (3580), and
    several ragged segments: full plane of sampled rows and ALL low-threshold candidates (hundreds on warp/segment seams
    and at both spectrum edges) against the oracle."""
    X = synth.random_spectrum(nbins, 1000 + nbins)
    cfg = _Cfg(nbins, 20.0, 2.0, 60.0, 20.0)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, 4096)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    zs, ws = orc.grid_values(20, 2), orc.grid_values(60, 20)
    rows = [(0, 0), (20, 6), (10, 3), (3, 5), (17, 1), (20, 0), (0, 6)]
    ref = H.oracle_rows(X, [(zs[iz], ws[iw]) for iz, iw in rows], 0, nbins)
    P = plan.search_plane(d_spec, 0, nbins).cpu().numpy()
    for (iz, iw), r in zip(rows, ref):
        H.assert_power_close(P[iw, iz], r, f"nbins={nbins} row {(iz, iw)}")
    # sub-box == slice of the full plane, bit for bit
    r_lo, r_cnt = nbins // 3, max(1, nbins // 5)
    sub = plan.search_plane(d_spec, r_lo, r_cnt, 5, 4, 2, 3).cpu().numpy()
    assert np.array_equal(sub, P[2:5, 5:9, 2 * r_lo:2 * (r_lo + r_cnt)])
    thr = 5.0
    d_c, d_n = plan.search_candidates(d_spec, thr, max_cands=1 << 18)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert n == cands.size and len({(c["j"], c["iz"], c["iw"]) for c in cands}) == n
    assert plan.work_counters()[2] == 0                                       # no seam overflow
    m, s = _check_candidates(cfg, X, cands, rows, 0, nbins, thr)
    assert m == s and (s > 0 or nbins < 1000)
    # first and last half-bin of a row can be candidates (P[-1] = P[2 nbins] = -inf)
    assert cands["j"].min() >= 0 and cands["j"].max() <= 2 * nbins - 1


@pytest.mark.gpu
def test_sharded_search_entry_point_single_rank():
    """shard.search_candidates_sharded without a process group == the whole-grid search (the N = 1 end of SURVEY.md 8(e);
    the multi-rank host logic runs under gloo in tests/test_shard_gloo.py, the box property in test_candidates_range_union)."""
    from paper_1911_01353_b200 import shard
    cfg, X, plan, d_spec = _setup(1)
    got = shard.search_candidates_sharded(plan, d_spec, 8.0)
    full, n = binding.candidates_to_numpy(*plan.search_candidates(d_spec, 8.0))
    assert np.array_equal(got, np.sort(full, order=["iw", "iz", "j"]))
