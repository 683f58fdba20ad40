"""GPU parity of the fused row statistics + S/N candidate filter against oracle/jerk_oracle.py section G."""
import numpy as np
import pytest

from oracle import jerk_oracle as orc
from paper_1911_01353_b200 import binding, build
import workloads as synth
from tests import helpers as H

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

NBINS, ZMAX, DZ, WMAX, DW, THR, SNR_THR = 30000, 20.0, 2.0, 60.0, 20.0, 8.0, 9.0


@pytest.fixture(scope="module")
def setup():
    build.build()
    binding.load_library()
    X = synth.random_spectrum(NBINS, seed=20251104).astype(np.complex128)
    c, hw, lattice = orc.template(10.0, 40.0)
    m, taps = orc.phase_taps(c, hw, lattice, 0)
    X[12345 + m] += 8.0 * taps                      # one strong jerk signal at (r, z, w) = (12345, 10, 40)
    X[:1500] *= 3.0                                 # and a loud band: S/N must be judged against the row's own statistics
    X = X.astype(np.complex64)
    plan = binding.Plan(NBINS, ZMAX, DZ, WMAX, DW, 2, 4096)
    plan.templates()
    d_spec = binding.spectrum_to_device(X)
    zs, ws = orc.grid_values(ZMAX, DZ), orc.grid_values(WMAX, DW)
    zw = [(zs[iz], ws[iw]) for iw in range(ws.size) for iz in range(zs.size)]
    rows = H.oracle_rows(X, zw, 0, NBINS)            # every row of the plane: 147 x 60000 points
    return X, plan, d_spec, zs, ws, rows


def test_row_statistics_match_the_oracle(setup):
    X, plan, d_spec, zs, ws, rows = setup
    d_c, d_n, d_stats = plan.search_candidates_stats(d_spec, THR)
    stats = d_stats.cpu().numpy()
    want = np.array([orc.row_stats(P) for P in rows])
    # every power is within 1e-3 * max(1, P) (north_star); the sums of 60000 of them average the error down
    assert np.abs(stats[:, 0] / want[:, 0] - 1.0).max() < 2e-5
    assert np.abs(stats[:, 1] / want[:, 1] - 1.0).max() < 1e-4
    # the candidates of the fused pass are those of the plain candidate search, record for record
    plain, n0 = binding.candidates_to_numpy(*plan.search_candidates(d_spec, THR))
    fused, n1 = binding.candidates_to_numpy(d_c, d_n)
    assert n0 == n1 and np.array_equal(np.sort(plain, order=["iw", "iz", "j"]), np.sort(fused, order=["iw", "iz", "j"]))


def test_snr_filter_matches_the_oracle(setup):
    X, plan, d_spec, zs, ws, rows = setup
    d_c, d_n, d_stats = plan.search_candidates_stats(d_spec, THR)
    d_o, d_no = plan.snr_filter(d_stats, d_c, d_n, SNR_THR)
    kept, nk = binding.candidates_to_numpy(d_o, d_no)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert 0 < nk < n
    kept_keys = {(int(c["iw"]), int(c["iz"]), int(c["j"])): c for c in kept}
    nz = zs.size
    strong = 0
    for c in cands:
        P = rows[int(c["iw"]) * nz + int(c["iz"])]
        mean, std = orc.row_mean_std(P)
        s_ref = float(orc.snr(P[int(c["j"])], mean, std))
        key = (int(c["iw"]), int(c["iz"]), int(c["j"]))
        if s_ref > 1.02 * SNR_THR:
            strong += 1
            assert key in kept_keys, (key, s_ref)
        if s_ref < 0.98 * SNR_THR:
            assert key not in kept_keys, (key, s_ref)
        if key in kept_keys:
            s_gpu = float(np.array(kept_keys[key]["flags"], dtype=np.uint32).view(np.float32))
            assert abs(s_gpu - s_ref) <= 2e-3 * max(1.0, abs(s_ref))
    assert strong > 0
    # the injected signal survives at its grid point
    iz0, iw0 = int(np.argmin(np.abs(zs - 10.0))), int(np.argmin(np.abs(ws - 40.0)))
    assert (iw0, iz0, 2 * 12345) in kept_keys


@pytest.mark.parametrize("seg_len", [1024, 2048, 8192])
def test_row_statistics_on_every_seg_len(setup, seg_len):
    """The fused statistics in the three-pass kernels k_search<L, MODE_CAND_STATS>: the same sums and candidates as the oracle rows."""
    X, plan, d_spec, zs, ws, rows = setup
    p2 = binding.Plan(NBINS, ZMAX, DZ, WMAX, DW, 2, seg_len)
    p2.templates()
    d_c, d_n, d_stats = p2.search_candidates_stats(d_spec, THR)
    stats = d_stats.cpu().numpy()
    want = np.array([orc.row_stats(P) for P in rows])
    assert np.abs(stats[:, 0] / want[:, 0] - 1.0).max() < 2e-5
    assert np.abs(stats[:, 1] / want[:, 1] - 1.0).max() < 1e-4
    plain, n0 = binding.candidates_to_numpy(*p2.search_candidates(d_spec, THR))
    fused, n1 = binding.candidates_to_numpy(d_c, d_n)
    assert n0 == n1 and np.array_equal(np.sort(plain, order=["iw", "iz", "j"]), np.sort(fused, order=["iw", "iz", "j"]))


@pytest.mark.parametrize("seg_len", [4096, 2048])
def test_row_statistics_and_snr_with_numbetween_one(setup, seg_len):
    """numbetween = 1 (SURVEY.md 8(f) N4 with N2): a row holds nbins points, not 2 nbins -- the sums, and the mean and
    sigma the S/N filter derives from them, are those of the oracle's phase-0 points (oracle section I = even j of section C)."""
    X, plan, d_spec, zs, ws, rows = setup
    p1 = binding.Plan(NBINS, ZMAX, DZ, WMAX, DW, 1, seg_len)
    p1.templates()
    rows1 = [P[0::2] for P in rows]
    assert np.abs(orc.power_row_nb1(X, float(zs[3]), float(ws[2]), 12000, 64) - rows1[2 * zs.size + 3][12000:12064]).max() < 1e-9
    d_c, d_n, d_stats = p1.search_candidates_stats(d_spec, THR)
    stats = d_stats.cpu().numpy()
    want = np.array([orc.row_stats(P) for P in rows1])
    assert np.abs(stats[:, 0] / want[:, 0] - 1.0).max() < 2e-5
    assert np.abs(stats[:, 1] / want[:, 1] - 1.0).max() < 1e-4
    d_o, d_no = p1.snr_filter(d_stats, d_c, d_n, SNR_THR)
    kept, nk = binding.candidates_to_numpy(d_o, d_no)
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert 0 < nk < n
    kept_keys = {(int(c["iw"]), int(c["iz"]), int(c["j"])): c for c in kept}
    nz = zs.size
    strong = 0
    for c in cands:
        P = rows1[int(c["iw"]) * nz + int(c["iz"])]
        mean, std = orc.row_mean_std(P)
        s_ref = float(orc.snr(P[int(c["j"])], mean, std))
        key = (int(c["iw"]), int(c["iz"]), int(c["j"]))
        if s_ref > 1.02 * SNR_THR:
            strong += 1
            assert key in kept_keys, (key, s_ref)
        if s_ref < 0.98 * SNR_THR:
            assert key not in kept_keys, (key, s_ref)
        if key in kept_keys:
            s_gpu = float(np.array(kept_keys[key]["flags"], dtype=np.uint32).view(np.float32))
            assert abs(s_gpu - s_ref) <= 2e-3 * max(1.0, abs(s_ref))
    assert strong > 0
    iz0, iw0 = int(np.argmin(np.abs(zs - 10.0))), int(np.argmin(np.abs(ws - 40.0)))
    assert (iw0, iz0, 12345) in kept_keys


# ------------------------------------------------------------------------------------------------ cross-row sifting
def _to_tuples(a):
    return [(int(c["j"]), int(c["iz"]), int(c["iw"]), float(c["power"])) for c in a]


@pytest.mark.parametrize("windows", [(4, 1, 1), (40, 3, 2), (0, 0, 0)])
def test_sift_matches_the_oracle_on_search_output(setup, windows):
    X, plan, d_spec, zs, ws, rows = setup
    d_c, d_n = plan.search_candidates(d_spec, 45.0)          # the loud band and the injected signal: ~1e3 candidates
    cands, n = binding.candidates_to_numpy(d_c, d_n)
    assert 100 < n < 5000, n
    d_o, d_no = plan.sift_candidates(d_c, d_n, *windows)
    kept, nk = binding.candidates_to_numpy(d_o, d_no)
    want = orc.sift(_to_tuples(cands), *windows)
    assert sorted(_to_tuples(kept), key=lambda c: (c[2], c[1], c[0])) == want     # bit-exact: index and byte work only
    if windows == (0, 0, 0):
        assert nk == n
    else:
        assert nk < n
    # the injected signal's cluster collapses to its grid point
    iz0, iw0 = int(np.argmin(np.abs(zs - 10.0))), int(np.argmin(np.abs(ws - 40.0)))
    assert (2 * 12345, iz0, iw0) in {(c[0], c[1], c[2]) for c in want}


def test_sift_ties_and_empty_list(setup):
    X, plan, d_spec, zs, ws, rows = setup
    rng = np.random.default_rng(8)
    n = 3000
    a = np.zeros(n, dtype=binding.CAND_DTYPE)
    keys = set()
    while len(keys) < n:
        keys.add((int(rng.integers(0, 3000)), int(rng.integers(0, 21)), int(rng.integers(0, 7))))
    for i, (j, iz, iw) in enumerate(sorted(keys)):
        a[i] = (j, iz, iw, float(rng.integers(4, 9)) * 5.0, 0)           # five distinct power values: many exact ties
    a = a[rng.permutation(n)]
    d_c = torch.from_numpy(a.view(np.uint8).reshape(-1).copy()).cuda()
    d_n = torch.tensor([n], dtype=torch.int64, device="cuda")
    d_o, d_no = plan.sift_candidates(d_c, d_n, 8, 2, 1)
    kept, nk = binding.candidates_to_numpy(d_o, d_no)
    assert sorted(_to_tuples(kept), key=lambda c: (c[2], c[1], c[0])) == orc.sift(_to_tuples(a), 8, 2, 1)
    d_n.zero_()
    d_o, d_no = plan.sift_candidates(d_c, d_n, 8, 2, 1)
    assert int(d_no.item()) == 0
