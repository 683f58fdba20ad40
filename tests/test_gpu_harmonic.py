"""GPU parity of the harmonic-sum stage (BASELINE.json configs[4]) against the oracle's
definition S_h(j,iz',iw') = sum_k P[rnd(j k/h); rnd(iz' k/h), rnd(iw' k/h)] (oracle/jerk_oracle.py, section F)."""
import numpy as np
import pytest

from oracle import jerk_oracle as orc
from paper_1911_01353_b200 import binding, build
import workloads as synth
from tests import helpers as H

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

STAGES = (1, 2, 4, 8)


@pytest.fixture(scope="module", autouse=True)
def _built():
    build.build()
    binding.load_library()


def _harm_tol(h, s_ref):
    # every term obeys |P_gpu - P_ref| <= 1e-3*max(1, P_ref)  =>  |S_gpu - S_ref| <= 1e-3*(h + S_ref)
    return H.POWER_TOL * (h + s_ref)


def _small_case(nbins=3000, seed=41):
    """Config-1 grid on a short spectrum: noise plus an 8-harmonic signal whose harmonics stay on the grid."""
    rng = np.random.Generator(np.random.PCG64(seed))
    n = 2 * nbins
    x = rng.standard_normal(n)
    r0, z0, w0 = 300.5, 2.0, 0.0
    a = np.sqrt(4.0 * 40.0 / n)
    for k in range(1, 9):
        x += synth.chirp_series(n, k * r0, k * z0, k * w0, a / k)
    X = synth.block_normalise(np.fft.rfft(x)[:nbins]).astype(np.complex64)
    return X


@pytest.mark.parametrize("seg_len", [1024, 4096])
def test_harmonic_plane_and_top_match_oracle_on_full_small_volume(seg_len):
    """seg_len 1024: eight stored sub-planes + k_harm; seg_len 4096: the sums are formed inside the top-harmonic search
    pass (k_search64<MODE_HARM>), seven stored sub-planes."""
    nbins = 3000 if seg_len == 1024 else 9000
    X = _small_case(nbins)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    P = orc.plane(X, 20, 2, 60, 20)                                    # [7][21][6000] float64
    top = plan.harmonic_sum(d_spec, STAGES, (0.0, 0.0, 0.0, 0.0))
    for s, h in enumerate(STAGES):
        S_ref = orc.harmonic_sum_volume(P, h)
        S_gpu = plan.harmonic_plane(d_spec, h, 0, nbins).cpu().numpy().astype(np.float64)
        assert S_gpu.shape == S_ref.shape
        err = np.abs(S_gpu - S_ref) - _harm_tol(h, S_ref)
        assert err.max() <= 0, f"h={h}: worst excess {err.max()}"
        # arg-max: same point as the oracle unless the runner-up is within tolerance (then the GPU value must still match)
        iw, iz, j = np.unravel_index(np.argmax(S_ref), S_ref.shape)
        best = S_ref[iw, iz, j]
        second = np.partition(S_ref.ravel(), -2)[-2]
        rec = top[s]
        assert abs(rec["power"] - S_ref[rec["iw"], rec["iz"], rec["j"]]) <= _harm_tol(h, best)
        if best - second > 2 * _harm_tol(h, best):
            assert (rec["iw"], rec["iz"], rec["j"]) == (iw, iz, j), (h, rec, (iw, iz, j))
        # the fp32 plane the kernel itself produces and its own arg-max agree bit-exactly (ties -> first in row-major order)
        g = plan.harmonic_plane(d_spec, h, 0, nbins).cpu().numpy()
        assert np.unravel_index(np.argmax(g), g.shape) == (rec["iw"], rec["iz"], rec["j"])
        assert g.max() == rec["power"]
    # h = 1 is the plane itself
    S1 = plan.harmonic_plane(d_spec, 1, 0, nbins).cpu().numpy()
    assert np.array_equal(S1, plan.search_plane(d_spec, 0, nbins).cpu().numpy())


@pytest.mark.parametrize("seg_len", [1024, 4096])
def test_harmonic_plane_subbox_is_bit_exact_slice(seg_len):
    nbins = 3000
    X = _small_case(nbins)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    for h in (2, 8):
        full = plan.harmonic_plane(d_spec, h, 0, nbins).cpu().numpy()
        for (r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt) in [(0, 1, 0, 1, 0, 1), (2397, 603, 20, 1, 6, 1), (1000, 517, 3, 11, 1, 4)]:
            sub = plan.harmonic_plane(d_spec, h, r_lo, r_cnt, iz_lo, iz_cnt, iw_lo, iw_cnt).cpu().numpy()
            assert np.array_equal(sub, full[iw_lo:iw_lo + iw_cnt, iz_lo:iz_lo + iz_cnt, 2 * r_lo:2 * (r_lo + r_cnt)])


@pytest.mark.parametrize("seg_len", [1024, 4096])
def test_harmonic_chunking_is_invisible_and_thresholds_apply(seg_len):
    """A scratch buffer that forces many r-chunks gives the same tops; stages under threshold report j = -1."""
    nbins = 3000
    X = _small_case(nbins)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    a = plan.harmonic_sum(d_spec, STAGES, (0.0,) * 4)
    small = plan.harmonic_scratch_bytes() // 8
    b = plan.harmonic_sum(d_spec, STAGES, (0.0,) * 4, scratch_bytes=small)
    assert np.array_equal(a, b)
    c = plan.harmonic_sum(d_spec, (8, 1), (1e9, 0.0))
    assert c[0]["j"] == -1 and c[0]["power"] == 0.0 and c[1]["j"] == a[0]["j"] and c[1]["power"] == a[0]["power"]
    with pytest.raises(binding.JerkError) as e:
        plan.harmonic_sum(d_spec, (3,), (0.0,))
    assert e.value.status == binding.JERK_EINVAL
    with pytest.raises(binding.JerkError) as e:
        plan.harmonic_sum(d_spec, (1,), (0.0,), scratch_bytes=4096)
    assert e.value.status == binding.JERK_ENOMEM


def test_harmonic_prune_kernel_small_volume():
    """The PRUNE instantiation (hw_max = 258) of the fused top-harmonic pass on a coarse zmax 200 / wmax 600 grid
    (21 x 13 templates) over a short spectrum with ragged segments: the whole S_h volume and the stage tops vs the oracle."""
    nbins = 5000
    rng = np.random.Generator(np.random.PCG64(43))
    n = 2 * nbins
    x = rng.standard_normal(n)
    r0, z0, w0 = 310.5, 20.0, 0.0
    a = np.sqrt(4.0 * 60.0 / n)
    for k in range(1, 9):
        x += synth.chirp_series(n, k * r0, k * z0, k * w0, a / k)
    X = synth.block_normalise(np.fft.rfft(x)[:nbins]).astype(np.complex64)
    plan = binding.Plan(nbins, 200, 20, 600, 100, 2, 4096)
    assert plan.info.hw_max == 258 and plan.info.ntemplates == 21 * 13
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    P = orc.plane(X, 200, 20, 600, 100)
    top = plan.harmonic_sum(d_spec, STAGES, (0.0,) * 4)
    for s, h in enumerate(STAGES):
        S_ref = orc.harmonic_sum_volume(P, h)
        g = plan.harmonic_plane(d_spec, h, 0, nbins).cpu().numpy()
        err = np.abs(g.astype(np.float64) - S_ref) - _harm_tol(h, S_ref)
        assert err.max() <= 0, f"h={h}: worst excess {err.max()}"
        rec = top[s]
        assert np.unravel_index(np.argmax(g), g.shape) == (rec["iw"], rec["iz"], rec["j"]) and g.max() == rec["power"]
        iw, iz, j = np.unravel_index(np.argmax(S_ref), S_ref.shape)
        second = np.partition(S_ref.ravel(), -2)[-2]
        if S_ref[iw, iz, j] - second > 2 * _harm_tol(h, S_ref[iw, iz, j]):
            assert (rec["iw"], rec["iz"], rec["j"]) == (iw, iz, j)


def test_harmonic_wide_templates_seg_len_4096():
    """hw_max = 708 > 512 at seg_len 4096 (zmax 1200, wmax 400): the edge blocks of a unit are shorter than a pair's source
    range, so the block-maxima bound of the fused pass does not hold and the library must take the stored-sub-plane path.
    Whole S_h volume and stage tops vs the oracle, at thresholds 0 and at thresholds just under the true maxima (the
    setting in which a wrongly pruned pair loses the arg-max)."""
    nbins = 9000
    rng = np.random.Generator(np.random.PCG64(47))
    n = 2 * nbins
    x = rng.standard_normal(n)
    r0, z0, w0 = 410.5, 50.0, 25.0
    a = np.sqrt(4.0 * 60.0 / n)
    for k in range(1, 9):
        x += synth.chirp_series(n, k * r0, k * z0, k * w0, a / k)
    X = synth.block_normalise(np.fft.rfft(x)[:nbins]).astype(np.complex64)
    plan = binding.Plan(nbins, 1200, 400, 400, 200, 2, 4096)
    assert plan.info.hw_max == 708 and plan.info.ntemplates == 7 * 5
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    P = orc.plane(X, 1200, 400, 400, 200)
    top = plan.harmonic_sum(d_spec, STAGES, (0.0,) * 4)
    maxima = []
    for s, h in enumerate(STAGES):
        S_ref = orc.harmonic_sum_volume(P, h)
        g = plan.harmonic_plane(d_spec, h, 0, nbins).cpu().numpy()
        err = np.abs(g.astype(np.float64) - S_ref) - _harm_tol(h, S_ref)
        assert err.max() <= 0, f"h={h}: worst excess {err.max()}"
        rec = top[s]
        assert np.unravel_index(np.argmax(g), g.shape) == (rec["iw"], rec["iz"], rec["j"]) and g.max() == rec["power"]
        iw, iz, j = np.unravel_index(np.argmax(S_ref), S_ref.shape)
        second = np.partition(S_ref.ravel(), -2)[-2]
        if S_ref[iw, iz, j] - second > 2 * _harm_tol(h, S_ref[iw, iz, j]):
            assert (rec["iw"], rec["iz"], rec["j"]) == (iw, iz, j)
        maxima.append(float(g.max()))
    near = plan.harmonic_sum(d_spec, STAGES, tuple(0.999 * m for m in maxima))
    assert np.array_equal(near, top)


@pytest.mark.parametrize("seg_len,world", [(4096, 3), (1024, 2), (4096, 7)])
def test_harmonic_r_ranges_fold_to_the_single_call(seg_len, world):
    """jerk_harmonic_sum_range (the harmonic stage shards by r-range): the stage tops of `world` disjoint
    blocks of the top-harmonic axis, folded with the tie rule (shard.fold_stage_records), equal the single call bit for bit;
    every block's record lies inside its block; an empty block reports nothing; one rank is the whole call."""
    from paper_1911_01353_b200 import shard
    nbins = 9000
    X = _small_case(nbins)
    plan = binding.Plan(nbins, 20, 2, 60, 20, 2, seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    thr = (0.0, 0.0, 30.0, 1e9)
    whole = plan.harmonic_sum(d_spec, STAGES, thr)
    recs = []
    for r in range(world):
        lo, cnt = shard.block_range(nbins, world, r)
        part = plan.harmonic_sum(d_spec, STAGES, thr, r_lo=lo, r_cnt=cnt)
        for c in part:
            assert c["j"] == -1 or 2 * lo <= c["j"] < 2 * (lo + cnt)
        recs.append(part)
    folded = shard.fold_stage_records(np.stack(recs))
    assert folded.tobytes() == whole.tobytes()
    assert whole[3]["j"] == -1 and whole[0]["j"] >= 0
    empty = plan.harmonic_sum(d_spec, STAGES, thr, r_lo=100, r_cnt=0)
    assert (empty["j"] == -1).all() and (empty["power"] == 0).all()
    assert shard.harmonic_sum_sharded(plan, d_spec, STAGES, thr).tobytes() == whole.tobytes()      # no process group: this rank does it all
    with pytest.raises(binding.JerkError) as e:
        plan.harmonic_sum(d_spec, STAGES, thr, r_lo=nbins - 10, r_cnt=11)
    assert e.value.status == binding.JERK_EINVAL


class _OraclePowers:
    """P_ref(j, iz', iw') on demand (signed grid indices), one oracle row segment per request, cached."""

    def __init__(self, X, cfg):
        self.X, self.cfg = X, cfg
        self.zs, self.ws = orc.grid_values(cfg.zmax, cfg.dz), orc.grid_values(cfg.wmax, cfg.dw)
        self.cz, self.cw = (self.zs.size - 1) // 2, (self.ws.size - 1) // 2
        self.tmpl, self.rows = {}, {}

    def __call__(self, j, a, b):
        key = (a, b)
        if key not in self.tmpl:
            self.tmpl[key] = orc.template(float(self.zs[a + self.cz]), float(self.ws[b + self.cw]))
        blk = (j // 2) // 64
        if (key, blk) not in self.rows:
            self.rows[(key, blk)] = orc.power_row(self.X, float(self.zs[a + self.cz]), float(self.ws[b + self.cw]), blk * 64, 64,
                                                  tmpl=self.tmpl[key])
        return self.rows[(key, blk)][j - 128 * blk]


def test_config5_harmonic_search():
    """BASELINE.json configs[4]: N = 2^23, 4 signals x 8 harmonics, stages 1/2/4/8 with thresholds 25/35/50/75."""
    cfg = synth.config(5)
    X = synth.make_spectrum(cfg)
    plan = binding.Plan(cfg.nbins, cfg.zmax, cfg.dz, cfg.wmax, cfg.dw, 2, cfg.seg_len)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    thr = (25.0, 35.0, 50.0, 75.0)
    top = plan.harmonic_sum(d_spec, STAGES, thr)
    Pref = _OraclePowers(X, cfg)
    cz, cw = Pref.cz, Pref.cw
    for s, h in enumerate(STAGES):
        rec = top[s]
        assert rec["j"] >= 0 and rec["power"] > thr[s], (h, rec)
        # (1) the sum the GPU reports at its point is the oracle's sum at that point
        s_at = orc.harmonic_sum_point(Pref, int(rec["j"]), int(rec["iz"]) - cz, int(rec["iw"]) - cw, h)
        assert abs(rec["power"] - s_at) <= _harm_tol(h, s_at), (h, rec, s_at)
        # (2) nothing in the neighbourhoods of the injected top harmonics beats it, and the box around the strongest
        #     injection agrees element by element with jerk_harmonic_plane
        best_nb = (-1.0, None)
        for (r0, z0, w0, p1) in cfg.signals:
            j0, a0, b0 = int(round(2 * h * r0)), int(round(h * z0 / cfg.dz)), int(round(h * w0 / cfg.dw))
            r_lo = j0 // 2 - 2
            iz_lo, iw_lo = max(0, a0 + cz - 1), max(0, b0 + cw - 1)
            iz_cnt, iw_cnt = min(cfg.nz, a0 + cz + 2) - iz_lo, min(cfg.nw, b0 + cw + 2) - iw_lo
            S_gpu = plan.harmonic_plane(d_spec, h, r_lo, 5, iz_lo, iz_cnt, iw_lo, iw_cnt).cpu().numpy()
            for iwr in range(iw_cnt):
                for izr in range(iz_cnt):
                    for jr in range(10):
                        ref = orc.harmonic_sum_point(Pref, 2 * r_lo + jr, iz_lo + izr - cz, iw_lo + iwr - cw, h)
                        assert abs(S_gpu[iwr, izr, jr] - ref) <= _harm_tol(h, ref)
                        if ref > best_nb[0]:
                            best_nb = (ref, (2 * r_lo + jr, iz_lo + izr, iw_lo + iwr))
        assert rec["power"] >= best_nb[0] - 2 * _harm_tol(h, best_nb[0]), (h, rec, best_nb)
        # (3) the top candidate is an injected signal's h-th harmonic (within one grid step; S18/S19: what the oracle finds)
        hit = any(abs(rec["j"] - 2 * h * r0) <= 2 and abs(rec["iz"] - cz - h * z0 / cfg.dz) <= 1 and
                  abs(rec["iw"] - cw - h * w0 / cfg.dw) <= 1 for (r0, z0, w0, p1) in cfg.signals)
        if hit:
            assert rec["power"] >= best_nb[0] - 2 * _harm_tol(h, best_nb[0])
            if best_nb[0] - rec["power"] > 0 or (int(rec["j"]), int(rec["iz"]), int(rec["iw"])) != best_nb[1]:
                # a different point than the oracle's neighbourhood maximum is only acceptable as a near tie
                assert abs(best_nb[0] - s_at) <= 2 * _harm_tol(h, s_at)
