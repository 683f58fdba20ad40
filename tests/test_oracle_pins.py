"""Pins for oracle/jerk_oracle.py against what the mathematics fixes.

The paper prints no worked example, so the pins are closed forms, invariants, brute force on
tiny inputs, and regression values computed independently of the oracle (tests/golden/).
Each pin is chosen so that a plausible mistake (dropped term, sign, index, transposed operand)
fails it.  None of these tests touches the CUDA path.
"""
import math
import os
from fractions import Fraction

import numpy as np
import pytest
from scipy.special import fresnel

from oracle import jerk_oracle as orc
import workloads as synth

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---- P1: z = w = 0 closed form  R(q) = exp(-i pi q) sinc(pi q)   (BASELINE.json north_star)
def test_p1_sinc_closed_form():
    q = np.arange(-40, 60, 0.25)
    ref = np.exp(-1j * np.pi * q) * np.sinc(q)           # numpy sinc(x) = sin(pi x)/(pi x)
    assert np.abs(orc.response(0.0, 0.0, q) - ref).max() < 1e-13


# ---- P2: w = 0 Fresnel closed form
def _fresnel_response(z, q):
    q = np.asarray(q, dtype=np.float64)
    if z < 0:
        return np.conj(_fresnel_response(-z, -q))
    s0 = -q * np.sqrt(2.0 / z)
    s1 = (z - q) * np.sqrt(2.0 / z)
    S1, C1 = fresnel(s1)
    S0, C0 = fresnel(s0)
    return np.exp(-1j * np.pi * q * q / z) / np.sqrt(2 * z) * ((C1 - C0) + 1j * (S1 - S0))


@pytest.mark.parametrize("z", [2.0, -2.0, 10.0, -10.0, 37.0, 200.0, -200.0])
def test_p2_fresnel_closed_form(z):
    q = np.arange(-300, 300, 0.5)
    assert np.abs(orc.response(z, 0.0, q) - _fresnel_response(z, q)).max() < 1e-12


# ---- P3: conjugate symmetry R_{-z,-w}(-q) = conj R_{z,w}(q)   (no closed form exists for w != 0)
@pytest.mark.parametrize("z,w", [(10.0, 40.0), (-20.0, 60.0), (200.0, -600.0), (6.0, -40.0)])
def test_p3_conjugate_symmetry(z, w):
    q = np.arange(-60, 90, 0.5)
    assert np.abs(orc.response(-z, -w, -q) - np.conj(orc.response(z, w, q))).max() < 1e-13


# ---- quadrature refinement: doubling panels and raising the order changes nothing
def test_quadrature_converged():
    q = np.arange(-20, 520, 0.5)
    a = orc.response(200.0, 600.0, q)
    b = orc.response(200.0, 600.0, q, panels=4000, order=20)
    assert np.abs(a - b).max() < 1e-13


# ---- w != 0 pin that is not a self-comparison: brute-force midpoint rule with 2e6 points
def test_response_vs_midpoint_rule():
    z, w = 10.0, 40.0
    n = 2_000_000
    u = (np.arange(n) + 0.5) / n
    for q in (-3.0, 14.5, 31.0):
        ref = np.exp(2j * np.pi * (z * u * u / 2 + w * u ** 3 / 6 - q * u)).mean()
        assert abs(orc.response(z, w, [q])[0] - ref) < 1e-9


# ---- P4: Parseval: sum over all integer k of |R(k+delta)|^2 = 1 (unit-modulus function on [0,1])
def test_p4_unit_energy():
    k = np.arange(-3000, 3000)
    e = (np.abs(orc.response(10.0, 40.0, k + 0.37)) ** 2).sum()
    assert 0.9999 < e < 1.0            # 0.99996, tail ~ 1/k


# ---- template placement: centre / half-width / truncated energies against independently computed values
def _golden_rows(name):
    rows = []
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append(line.split())
    return rows


def test_template_centre_halfwidth_energy_golden():
    for z, w, c, hw, e0, e1 in _golden_rows("template_energy.txt"):
        z, w, c, hw, e0, e1 = float(z), float(w), int(c), int(hw), float(e0), float(e1)
        cc, hh, lat = orc.template(z, w)
        assert (cc, hh) == (c, hw), (z, w)
        assert lat.size == 4 * hw + 1
        m0, t0 = orc.phase_taps(cc, hh, lat, 0)
        m1, t1 = orc.phase_taps(cc, hh, lat, 1)
        assert m0.size == 2 * hw + 1 and m1.size == 2 * hw and m0[0] == c - hw and m1[-1] == c + hw
        assert abs((np.abs(t0) ** 2).sum() - e0) < 1.5e-5, (z, w)
        assert abs((np.abs(t1) ** 2).sum() - e1) < 1.5e-5, (z, w)
        # symmetric partner: c -> -c, same energies (exact symmetry P3)
        c2, h2, lat2 = orc.template(-z, -w)
        assert (c2, h2) == (-c, hw)


def test_excursion_brute_force():
    u = np.linspace(0, 1, 200001)
    for z, w in [(10, 40), (-20, 60), (200, -600), (50, -600), (-150, 600), (0, 600), (7, 0), (0, 0)]:
        g = z * u + w * u * u / 2
        lo, hi = orc.excursion(float(z), float(w))
        assert abs(lo - g.min()) < 1e-6 and abs(hi - g.max()) < 1e-6


def test_grid_values():
    zs = orc.grid_values(20, 2)
    ws = orc.grid_values(60, 20)
    assert zs.size == 21 and zs[0] == -20 and zs[-1] == 20 and zs[10] == 0
    assert ws.size == 7 and list(ws) == [-60, -40, -20, 0, 20, 40, 60]


# ---- P5: a noise-free unit-amplitude injection peaks at exactly its grid point with P = (sum |R|^2)^2
def _noise_free_spectrum(r0, z0, w0, n=1 << 16):
    x = synth.chirp_series(n, r0, z0, w0, 1.0)
    return (np.fft.rfft(x)[: n // 2] * (2.0 / n)).astype(np.complex128)


def test_p5_injection_recovered_at_exact_grid_point():
    gold = _golden_rows("injection_noise_free.txt")
    peaks = [g for g in gold if g[0] != "competitor"]
    comps = [g for g in gold if g[0] == "competitor"]
    b_lo, b_cnt = 4960, 100
    zs, ws = orc.grid_values(20, 2), orc.grid_values(60, 20)
    for r0, r_pk, z_pk, w_pk, p_pk in peaks:
        r0, r_pk, z_pk, w_pk, p_pk = map(float, (r0, r_pk, z_pk, w_pk, p_pk))
        X = _noise_free_spectrum(r0, 10.0, 40.0)
        vol = orc.plane(X, 20, 2, 60, 20, b_lo, b_cnt)
        iw, iz, j = np.unravel_index(np.argmax(vol), vol.shape)
        assert (ws[iw], zs[iz]) == (w_pk, z_pk)
        assert b_lo + j / 2.0 == r_pk
        assert abs(vol[iw, iz, j] - p_pk) < 3e-4           # discrete-vs-continuous response: O(1/N)
        if r0 == 5000.5:
            for _, z, w, r, p in comps:
                row = vol[list(ws).index(float(w)), list(zs).index(float(z))]
                jj = int(np.argmax(row))
                assert b_lo + jj / 2.0 == float(r)
                assert abs(row[jj] - float(p)) < 5e-4
    # on-grid peak power equals the squared truncated template energy (reading S6: no renormalisation)
    c, hw, lat = orc.template(10.0, 40.0)
    e1 = (np.abs(orc.phase_taps(c, hw, lat, 1)[1]) ** 2).sum()
    X = _noise_free_spectrum(5000.5, 10.0, 40.0)
    p = orc.power_row(X, 10.0, 40.0, 5000, 1)[1]
    assert abs(p - e1 ** 2) < 3e-4


# ---- P6: brute force on a tiny input: de-chirped DFT == spectral correlation with the discrete full-width template
def test_p6_bruteforce_dechirped_dft():
    n = 512
    rng = np.random.default_rng(5)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = np.fft.fft(x)                                            # forward DFT e^{-2 pi i k n / N} (S8)
    u = np.arange(n) / n
    z, w = 6.0, -20.0
    hw = n // 2 - 2
    c = 0
    # discrete template D(q) = (1/N) sum_n exp(2 pi i (z u^2/2 + w u^3/6 - q u)) on the half-bin lattice
    qs = c - hw + 0.5 * np.arange(4 * hw + 1)
    chirp = z * u * u / 2 + w * u ** 3 / 6
    D = np.array([np.exp(2j * np.pi * (chirp - q * u)).mean() for q in qs])
    # brute force: A(r) = sum_n x_n exp(-2 pi i (r u + z u^2/2 + w u^3/6)) with X periodic -> use wrapped spectrum
    Xw = np.concatenate((X, X, X))                               # periodic extension, bins -n..2n
    b_lo, b_cnt = n + 100, 40
    A = orc.amplitude_row(Xw, z, w, b_lo, b_cnt, tmpl=(c, hw, D))
    for i in range(2 * b_cnt):
        r = (b_lo - n) + i / 2.0
        ref = (x * np.exp(-2j * np.pi * (r * u + chirp))).sum()
        # taps cover 2hw+1 = n-3 of the n bins of the periodic spectrum: the remainder is O(|D| at the edge)
        assert abs(A[i] - ref) < 2e-2 * abs(ref) + 0.5


def test_p6_exact_with_full_period_taps():
    """Same as above but with an odd N so that 2hw+1 = N covers the period exactly: agreement to rounding."""
    n = 257
    rng = np.random.default_rng(6)
    x = rng.standard_normal(n) + 1j * rng.standard_normal(n)
    X = np.fft.fft(x)
    u = np.arange(n) / n
    z, w = 4.0, 12.0
    hw, c = (n - 1) // 2, 0
    qs = c - hw + 0.5 * np.arange(4 * hw + 1)
    chirp = z * u * u / 2 + w * u ** 3 / 6
    D = np.array([np.exp(2j * np.pi * (chirp - q * u)).mean() for q in qs])
    Xw = np.concatenate((X, X, X))
    b_lo, b_cnt = n + 30, 20
    A = orc.amplitude_row(Xw, z, w, b_lo, b_cnt, tmpl=(c, hw, D))
    for i in range(0, 2 * b_cnt, 2):                            # integer r: exact (phase-0 taps span one full period)
        r = (b_lo - n) + i // 2
        ref = (x * np.exp(-2j * np.pi * (r * u + chirp))).sum()
        assert abs(A[i] - ref) < 1e-10 * n


# ---- correlation routine against an independent library routine (np.correlate) with arbitrary taps
def test_amplitude_row_vs_np_correlate():
    rng = np.random.default_rng(11)
    X = rng.standard_normal(300) + 1j * rng.standard_normal(300)
    c, hw = -7, 12
    lat = rng.standard_normal(4 * hw + 1) + 1j * rng.standard_normal(4 * hw + 1)
    A = orc.amplitude_row(X, 0.0, 0.0, 0, 300, tmpl=(c, hw, lat))
    for p in (0, 1):
        ms, taps = orc.phase_taps(c, hw, lat, p)
        # A_p[b] = sum_m X[b+m] conj(t_m); np.correlate(a, v)[k] = sum_n a[n+k] conj(v[n])
        pad = 64
        Xp = np.concatenate((np.zeros(pad), X, np.zeros(pad)))
        full = np.correlate(Xp, taps, mode="valid")              # index k <-> first tap at Xp[k]
        ref = np.array([full[b + ms[0] + pad] for b in range(300)])
        assert np.abs(A[p::2] - ref).max() < 1e-11


def test_edges_are_zero_padded():
    X = np.ones(50, dtype=np.complex128)
    A = orc.amplitude_row(X, 0.0, 0.0)
    c, hw, lat = orc.template(0.0, 0.0)
    # bin 0, phase 0: only taps m >= 0 see data
    ms, taps = orc.phase_taps(c, hw, lat, 0)
    assert abs(A[0] - np.conj(taps[ms >= 0]).sum()) < 1e-12
    ms, taps = orc.phase_taps(c, hw, lat, 1)
    assert abs(A[99] - np.conj(taps[ms <= 0]).sum()) < 1e-12    # last bin, phase 1


# ---- P7: noise statistics: P is exponential with mean sum |h|^2
def test_p7_noise_statistics():
    X = synth.random_spectrum(60000, 99)
    P = orc.power_row(X, 10.0, 40.0)
    c, hw, lat = orc.template(10.0, 40.0)
    e0 = (np.abs(lat[0::2]) ** 2).sum()
    e1 = (np.abs(lat[1::2]) ** 2).sum()
    assert abs(P[0::2].mean() - e0) < 0.02 and abs(P[1::2].mean() - e1) < 0.02
    frac = (P > 5.0).mean()
    assert abs(frac - math.exp(-5.0 / 0.9925)) < 0.0012


# ---- P8: shift invariance: moving the spectrum by k bins moves the plane by 2k half-bins
def test_p8_shift_invariance():
    X = synth.random_spectrum(4000, 3)
    k = 37
    Xs = np.concatenate((np.zeros(k, dtype=X.dtype), X))
    a = orc.power_row(X, -12.0, 40.0, 500, 200)
    b = orc.power_row(Xs, -12.0, 40.0, 500 + k, 200)
    assert np.abs(a - b).max() < 1e-12


# ---- E: candidate rule, brute-force loop
def test_candidates_bruteforce():
    rng = np.random.default_rng(2)
    P = rng.exponential(size=500)
    P[100] = P[101] = 9.0                                        # exact tie: the right-hand one is not > left
    P[0] = 8.0
    P[-1] = 8.5
    j, pw, margin = orc.row_candidates(P, 3.0, j_offset=1000)
    want = []
    for i in range(500):
        l = P[i - 1] if i > 0 else -np.inf
        r = P[i + 1] if i < 499 else -np.inf
        if P[i] > 3.0 and P[i] > l and P[i] >= r:
            want.append(i + 1000)
    assert list(j) == want
    assert 1100 in want and 1101 not in want and 1000 in want and 1499 in want
    assert np.all(margin >= 0)


# ---- F / P10: harmonic sum rounding rule and volume routine against pure-Python brute force
def test_rnd_frac_is_round_half_away():
    for a in range(-40, 41):
        for h in (1, 2, 4, 8):
            for k in range(1, h + 1):
                f = Fraction(a * k, h)
                ref = int(math.floor(abs(f) + Fraction(1, 2))) * (1 if f >= 0 else -1)
                assert orc.rnd_frac(a, k, h) == ref


def test_p10_harmonic_volume_bruteforce():
    rng = np.random.default_rng(8)
    P = rng.exponential(size=(5, 7, 40))
    cz, cw = 3, 2
    for h in (1, 2, 4, 8):
        S = orc.harmonic_sum_volume(P, h)
        for iw in range(5):
            for iz in range(7):
                for j in range(40):
                    ref = orc.harmonic_sum_point(
                        lambda jj, a, b: P[b + cw, a + cz, jj], j, iz - cz, iw - cw, h)
                    assert abs(S[iw, iz, j] - ref) < 1e-12
    # h = 1 is the plane itself
    assert np.array_equal(orc.harmonic_sum_volume(P, 1), P)


def test_p10_harmonic_injection_noise_free():
    """8-harmonic noise-free injection: S_h peaks at h*(j0, iz0', iw0') (SURVEY 8(c)-F, Appendix values)."""
    n = 1 << 14
    r0, z0, w0 = 300.0, 2.0, 20.0
    x = np.zeros(n)
    for k in range(1, 9):
        x += synth.chirp_series(n, k * r0, k * z0, k * w0, 1.0 / k)
    X = np.fft.rfft(x)[: n // 2] * (2.0 / n)
    ideal = {1: 1.0, 2: 1.25, 4: 1.4236, 8: 1.5274}
    zmax, dz, wmax, dw = 20.0, 2.0, 180.0, 20.0
    zs, ws = orc.grid_values(zmax, dz), orc.grid_values(wmax, dw)
    cz, cw = (zs.size - 1) // 2, (ws.size - 1) // 2
    cache = {}

    def P_lookup(j, a, b):
        key = (a, b)
        if key not in cache:
            cache[key] = orc.power_row(X, float(zs[a + cz]), float(ws[b + cw]))
        return cache[key][j]

    j0, a0, b0 = int(2 * r0), int(z0 / dz), int(w0 / dw)
    for h in (1, 2, 4, 8):
        s = orc.harmonic_sum_point(P_lookup, h * j0, h * a0, h * b0, h)
        assert ideal[h] * 0.95 < s <= ideal[h] + 1e-3            # truncation energy loses a few per cent
        # moving the top harmonic off by one grid step in any coordinate lowers the sum
        for dj, da, db in ((2, 0, 0), (-2, 0, 0), (0, 1, 0), (0, 0, 1)):
            assert orc.harmonic_sum_point(P_lookup, h * j0 + dj, h * a0 + da, h * b0 + db, h) < s


# ------------------------------------------------------------------------------------------------ G: row statistics, S/N
def test_row_mean_std_against_textbook_routines():
    import statistics
    rng = np.random.default_rng(11)
    P = rng.exponential(1.0, 500)
    mean, std = orc.row_mean_std(P)
    assert abs(mean - statistics.fmean(P.tolist())) < 1e-12
    assert abs(std - statistics.pstdev(P.tolist())) < 1e-12
    s1, s2 = orc.row_stats(P)
    assert abs(s1 - math.fsum(P.tolist())) < 1e-9 and abs(s2 - math.fsum((P * P).tolist())) < 1e-9
    assert orc.row_mean_std(np.full(10, 3.0)) == (3.0, 0.0)


def test_noise_row_has_std_equal_to_mean():
    """Unit-variance complex Gaussian X: P is exponential (pin P7), whose standard deviation equals its mean = sum |h|^2."""
    X = synth.random_spectrum(60000, seed=99)
    P = orc.power_row(X, 10.0, 40.0, 0, 60000)
    mean, std = orc.row_mean_std(P)
    assert abs(mean - 0.9925) < 0.015            # mean 0.9925 for (10, 40)
    assert abs(std / mean - 1.0) < 0.03


def test_snr_is_scale_invariant_and_filter_is_a_plain_comparison():
    X = synth.random_spectrum(8000, seed=5)
    P = orc.power_row(X, 4.0, 20.0, 0, 8000)
    P9 = orc.power_row(X.astype(np.complex128) * 3.0, 4.0, 20.0, 0, 8000)
    m1, s1 = orc.row_mean_std(P)
    m9, s9 = orc.row_mean_std(P9)
    assert abs(m9 / m1 - 9.0) < 1e-9 and abs(s9 / s1 - 9.0) < 1e-9
    assert np.allclose(orc.snr(P, m1, s1), orc.snr(P9, m9, s9), atol=1e-9)
    j = np.arange(P.size)
    kj, kp, ks = orc.snr_filter(j, P, m1, s1, 4.0)
    want = [int(i) for i in range(P.size) if (P[i] - m1) / s1 > 4.0]
    assert kj.tolist() == want and np.allclose(ks, (kp - m1) / s1)
    assert orc.snr_filter(j, P, m1, 0.0, 4.0)[0].size == 0


# ------------------------------------------------------------------------------------------------ H: sifting
def _random_cands(rng, n, nj=4000, nz=21, nw=7, quant=None):
    seen, out = set(), []
    while len(out) < n:
        key = (int(rng.integers(0, nj)), int(rng.integers(0, nz)), int(rng.integers(0, nw)))
        if key in seen:
            continue
        seen.add(key)
        p = float(rng.uniform(20, 90))
        out.append(key + ((round(p / quant) * quant) if quant else p,))
    return out


def test_sift_hand_worked_cases():
    # one cluster: the strongest wins; an isolated weak candidate survives; windows are inclusive
    c = [(100, 5, 3, 50.0), (101, 5, 3, 40.0), (100, 6, 3, 45.0), (100, 5, 4, 30.0), (500, 5, 3, 21.0)]
    assert orc.sift(c, 2, 1, 1) == [(100, 5, 3, 50.0), (500, 5, 3, 21.0)]
    assert orc.sift(c, 0, 0, 0) == sorted(c, key=lambda x: (x[2], x[1], x[0]))
    assert orc.sift([(10, 0, 0, 5.0), (13, 0, 0, 6.0)], 3, 0, 0) == [(13, 0, 0, 6.0)]
    assert orc.sift([(10, 0, 0, 5.0), (14, 0, 0, 6.0)], 3, 0, 0) == [(10, 0, 0, 5.0), (14, 0, 0, 6.0)]
    # suppression is not transitive clustering: b kills a, c kills b, a is not within reach of c but stays dead
    chain = [(0, 0, 0, 1.0), (2, 0, 0, 2.0), (4, 0, 0, 3.0)]
    assert orc.sift(chain, 2, 0, 0) == [(4, 0, 0, 3.0)]
    # equal powers: the smaller (iw, iz, j) wins
    assert orc.sift([(7, 2, 1, 9.0), (7, 2, 0, 9.0)], 0, 0, 1) == [(7, 2, 0, 9.0)]
    assert orc.sift([], 1, 1, 1) == []


def test_sift_invariants():
    rng = np.random.default_rng(2024)
    for quant in (None, 5.0):                      # continuous powers, and heavily tied ones
        c = _random_cands(rng, 400, quant=quant)
        kept = orc.sift(c, 6, 2, 1)
        assert 0 < len(kept) < len(c)
        # order independence
        perm = [c[i] for i in rng.permutation(len(c))]
        assert orc.sift(perm, 6, 2, 1) == kept
        # fixed point
        assert orc.sift(kept, 6, 2, 1) == kept
        # the global best (with the tie rule) survives; every dropped candidate has a surviving-or-not better neighbour
        best = min(c, key=lambda x: (-x[3], x[2], x[1], x[0]))
        assert best in kept
        # no two survivors are within one window of each other
        for i, a in enumerate(kept):
            for b in kept[i + 1:]:
                assert not (abs(a[0] - b[0]) <= 6 and abs(a[1] - b[1]) <= 2 and abs(a[2] - b[2]) <= 1)
        # larger windows never keep more
        assert len(orc.sift(c, 12, 4, 2)) <= len(kept)


# --------------------------------------------------------------------------- section I: numbetween = 1
def test_numbetween1_pins():
    """power_row_nb1 (phase-0 taps on integer bins) against what fixes it independently:
    (i) z = w = 0: R_{0,0}(m) = delta_{m0} (the closed-form sinc of pin P1 at integer q), so P[b] = |X[b]|^2 exactly;
    (ii) library correlation with the phase-0 taps; (iii) P6-style brute force: the de-chirped DFT of a time series at
    integer r equals the spectral correlation with the discrete full-width response (exact at odd N)."""
    rng = np.random.default_rng(12)
    X = (rng.standard_normal(300) + 1j * rng.standard_normal(300)).astype(np.complex128)
    P = orc.power_row_nb1(X, 0.0, 0.0)
    assert np.abs(P - np.abs(X) ** 2).max() < 1e-12
    for (z, w) in [(6.0, -40.0), (-20.0, 60.0)]:
        c, hw, lat = orc.template(z, w)
        m, taps = orc.phase_taps(c, hw, lat, 0)
        full = np.correlate(np.concatenate((np.zeros(600), X, np.zeros(600))), taps, mode="valid")    # sum_k Xp[i+k] conj(taps[k])
        want = np.abs(full[600 + m[0]: 600 + m[0] + 300]) ** 2
        got = orc.power_row_nb1(X, z, w)
        assert np.abs(got - want).max() < 1e-10 * max(1.0, want.max())
        sub = orc.power_row_nb1(X, z, w, 37, 11)
        assert np.array_equal(sub, got[37:48])
    # brute force in the time domain, N odd so that the discrete response has no aliasing ambiguity
    N, z, w = 255, 3.0, 10.0
    x = rng.standard_normal(N) + 1j * rng.standard_normal(N)
    u = np.arange(N) / N
    Xf = np.array([np.sum(x * np.exp(-2j * np.pi * k * u)) for k in range(N)])
    r = 100
    direct = np.sum(x * np.exp(-2j * np.pi * (r * u + z * u * u / 2 + w * u ** 3 / 6)))
    hw = N // 2
    q = np.arange(-hw, hw + 1)
    D = np.array([np.mean(np.exp(2j * np.pi * (z * u * u / 2 + w * u ** 3 / 6 - qq * u))) for qq in q])
    lattice = np.zeros(4 * hw + 1, dtype=np.complex128)
    lattice[0::2] = D                                   # phase-0 lattice points q = -hw..hw; the half-bin points are unused
    Xext = np.concatenate((Xf, Xf, Xf))                 # periodic extension: the routine itself zero-pads
    got = orc.power_row_nb1(Xext, z, w, N + r, 1, tmpl=(0, hw, lattice))[0]
    assert abs(got - abs(direct) ** 2) < 1e-9 * abs(direct) ** 2
