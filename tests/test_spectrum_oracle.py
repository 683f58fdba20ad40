"""Pins of oracle/spectrum_oracle.py (time series -> normalised spectrum), CPU only."""
import numpy as np
import pytest

from oracle import spectrum_oracle as so
import workloads as synth


def test_rfft_equals_the_written_out_sum():
    rng = np.random.default_rng(3)
    for n in (8, 64, 250):
        x = rng.standard_normal(n)
        assert np.allclose(so.real_dft(x), so.real_dft_direct(x), atol=1e-11)


def test_cosine_on_an_integer_bin():
    """a cos(2 pi k0 n / N + phi) -> X[k0] = N a/2 e^{i phi}, every other kept bin 0 (textbook closed form)."""
    n, k0, a, phi = 1024, 37, 0.6, 0.4
    x = a * np.cos(2 * np.pi * k0 * np.arange(n) / n + phi)
    X = so.real_dft(x)
    assert abs(X[k0] - n * a / 2 * np.exp(1j * phi)) < 1e-9
    X[k0] = 0
    assert np.abs(X).max() < 1e-9


def test_dc_kept_nyquist_dropped_and_parseval():
    rng = np.random.default_rng(4)
    n = 512
    x = rng.standard_normal(n) + 0.3
    X = so.real_dft(x)
    assert X.size == n // 2
    assert abs(X[0] - x.sum()) < 1e-10
    nyq = np.sum(x * (-1.0) ** np.arange(n))
    lhs = np.sum(x * x)
    rhs = (abs(X[0]) ** 2 + 2 * np.sum(np.abs(X[1:]) ** 2) + nyq ** 2) / n
    assert abs(lhs - rhs) < 1e-9 * lhs


def test_time_shift_is_a_linear_phase():
    rng = np.random.default_rng(5)
    n, s = 256, 5
    x = rng.standard_normal(n)
    k = np.arange(n // 2)
    assert np.allclose(so.real_dft(np.roll(x, s)), so.real_dft(x) * np.exp(-2j * np.pi * k * s / n), atol=1e-10)


@pytest.mark.parametrize("nbins,block", [(32768, 1000), (2500, 1000), (999, 1000), (7, 3)])
def test_blocks_have_unit_mean_power(nbins, block):
    rng = np.random.default_rng(6)
    X = (rng.standard_normal(nbins) + 1j * rng.standard_normal(nbins)) * np.linspace(0.5, 30.0, nbins)
    Y = so.normalise_blocks(X, block)
    m = so.block_powers(Y, block)
    assert np.allclose(m, 1.0, atol=1e-12)
    # phases untouched, one real positive factor per block
    f = Y / X
    assert np.allclose(f.imag, 0, atol=1e-15) and (f.real > 0).all()
    for b in range(m.size):
        assert np.ptp(f.real[b * block:(b + 1) * block]) < 1e-15 * f.real[b * block]


def test_zero_block_is_left_alone_and_scale_invariance():
    X = np.zeros(2000, dtype=np.complex128)
    X[1000:] = 3.0 + 4.0j
    Y = so.normalise_blocks(X, 1000)
    assert (Y[:1000] == 0).all() and np.allclose(np.abs(Y[1000:]), 1.0)
    rng = np.random.default_rng(7)
    x = rng.standard_normal(4096)
    assert np.allclose(so.prepare_spectrum(x), so.prepare_spectrum(17.5 * x), atol=1e-12)


def test_matches_the_input_generator_recipe():
    """synth.make_spectrum (the seeded input generator of the search tests) follows the same recipe: an independent
    implementation of A + B must reproduce it from the same time series."""
    cfg = synth.config(1)
    rng = np.random.Generator(np.random.PCG64(synth.SEED_BASE + cfg.index))
    x = rng.standard_normal(cfg.n, dtype=np.float32).astype(np.float64)
    sig = synth._draw_signals(cfg, rng)
    for (r0, z0, w0, p) in sig:
        x += synth.chirp_series(cfg.n, r0, z0, w0, np.sqrt(4.0 * p / cfg.n))
    x = x.astype(np.float32).astype(np.float64)
    want = synth.make_spectrum(synth.config(1))
    got = so.prepare_spectrum(x).astype(np.complex64)
    assert np.abs(got - want).max() < 1e-6


# --------------------------------------------------------------------------- normalisation variants (median, red noise)
def _select_kth(values, k):
    """k-th smallest by plain counting (no sort): brute force for tiny inputs."""
    for v in values:
        below = sum(1 for u in values if u < v)
        equal = sum(1 for u in values if u == v)
        if below <= k < below + equal:
            return v
    raise AssertionError


def test_median_against_brute_force_selection():
    rng = np.random.default_rng(9)
    for n in (1, 2, 5, 6, 33, 100):
        v = list(rng.exponential(size=n))
        want = _select_kth(v, n // 2) if n % 2 else 0.5 * (_select_kth(v, n // 2 - 1) + _select_kth(v, n // 2))
        assert so.median_plain(v) == want
    assert so.median_plain([3.0, 1.0, 2.0]) == 2.0 and so.median_plain([4.0, 1.0, 3.0, 2.0]) == 2.5


def test_median_of_exponential_noise_is_ln2_times_the_mean():
    """For complex Gaussian bins |X|^2 is exponential: median = ln 2 * mean.  So on pure noise B-median agrees with B
    (unit mean power per block) to the sampling error of a 1000-bin block (~ 1/sqrt(1000) * few)."""
    rng = np.random.default_rng(10)
    X = (rng.standard_normal(200_000) + 1j * rng.standard_normal(200_000)) * 3.7
    Y = so.normalise_median_blocks(X, so.uniform_bounds(X.size, 1000))
    m = so.block_powers(Y, 1000)
    assert abs(m.mean() - 1.0) < 0.01 and np.abs(m - 1.0).max() < 0.25
    # exact on a constructed block: powers 1..5 -> median 3 -> scale 1/sqrt(3/ln 2)
    Z = np.sqrt(np.arange(1.0, 6.0)).astype(np.complex128)
    out = so.normalise_median_blocks(Z, [0, 5])
    assert np.allclose(np.abs(out) ** 2, np.arange(1.0, 6.0) * np.log(2.0) / 3.0, rtol=1e-14)


def test_median_is_robust_to_a_strong_tone_and_scale_invariant():
    """One strong bin inflates the block MEAN (the noise of that block is pushed down by ~P/1000, reading S15) but leaves
    the MEDIAN-normalised noise level where it was; both variants are invariant under X -> a X."""
    rng = np.random.default_rng(11)
    X = (rng.standard_normal(4000) + 1j * rng.standard_normal(4000)) / np.sqrt(2.0)
    T = X.copy()
    T[1500] += 60.0                                          # power 3600 in block 1
    b = so.uniform_bounds(4000, 1000)
    base, tone = so.normalise_median_blocks(X, b), so.normalise_median_blocks(T, b)
    others = np.ones(4000, bool)
    others[1500] = False
    assert np.abs(tone[others] / base[others] - 1.0).max() < 5e-3          # one of 1000 order statistics moved: < 0.5 %
    mean_tone = so.normalise_blocks(T, 1000)
    mean_base = so.normalise_blocks(X, 1000)
    ratio = np.abs(mean_tone[1000:2000][np.arange(1000) != 500] / mean_base[1000:2000][np.arange(1000) != 500])
    assert ratio.max() < 0.6                                                 # the mean variant loses > 40 % of the noise amplitude there
    assert np.allclose(so.normalise_median_blocks(7.5 * X, b), base, rtol=1e-13)
    assert np.allclose(so.normalise_median_blocks(7.5 * X, so.rednoise_bounds(4000, 1000)), so.normalise_median_blocks(X, so.rednoise_bounds(4000, 1000)), rtol=1e-13)
    zero = np.zeros(10, dtype=np.complex128)
    assert np.array_equal(so.normalise_median_blocks(zero, [0, 10]), zero)   # zero median: left as it is


def test_rednoise_bounds_hand_worked_schedule():
    """len_0 = 6, len_{i+1} = min(block, len_i + max(1, len_i // 8)), worked by hand."""
    lens = [6, 7, 8, 9, 10, 11, 12, 13, 14, 15, 16, 18, 20, 22, 24, 27, 30, 33, 37, 41, 46, 51, 57, 64, 72, 81, 91, 102, 114, 128, 144,
            162, 182, 204, 229, 257, 289, 325, 365, 410, 461, 518, 582, 654, 735, 826, 929, 1000, 1000]
    n = sum(lens) + 17
    b = so.rednoise_bounds(n, 1000)
    assert [y - x for x, y in zip(b[:-1], b[1:])] == lens + [17]
    for nb, blk in ((1, 8), (5, 8), (6, 8), (7, 8), (100, 8), (32768, 1000), (12345, 64)):
        b = so.rednoise_bounds(nb, blk)
        assert b[0] == 0 and b[-1] == nb and all(y > x for x, y in zip(b[:-1], b[1:])) and max(y - x for x, y in zip(b[:-1], b[1:])) <= max(blk, 6)
    with pytest.raises(ValueError):
        so.rednoise_bounds(100, 4)


def test_rednoise_variant_flattens_a_red_spectrum():
    """Noise with a steep low-frequency slope: after B-rednoise every 200-bin stretch has unit mean power within sampling
    error, including the first ones, where one 1000-bin block of the mean variant leaves a slope of a factor > 3."""
    rng = np.random.default_rng(12)
    nb = 20000
    k = np.arange(nb) + 1.0
    shape = np.sqrt(1.0 + (300.0 / k) ** 2)                  # amplitude envelope: power ~ 1 + (300/k)^2
    X = (rng.standard_normal(nb) + 1j * rng.standard_normal(nb)) / np.sqrt(2.0) * shape
    red = so.normalise_median_blocks(X, so.rednoise_bounds(nb, 1000))
    flat = so.normalise_blocks(X, 1000)
    p_red = [np.mean(np.abs(red[a:a + 200]) ** 2) for a in range(200, 2000, 200)]
    p_flat = [np.mean(np.abs(flat[a:a + 200]) ** 2) for a in (0, 800)]
    assert max(p_red) < 1.35 and min(p_red) > 0.7
    assert p_flat[0] / p_flat[1] > 3.0
    # time series -> spectrum through the mode switch
    x = rng.standard_normal(4096)
    assert np.array_equal(so.prepare_spectrum_mode(x, 1000, "mean"), so.prepare_spectrum(x, 1000))
    assert np.array_equal(so.prepare_spectrum_mode(x, 100, "median"), so.normalise_median_blocks(so.real_dft(x), so.uniform_bounds(2048, 100)))
    assert np.array_equal(so.prepare_spectrum_mode(x, 100, "rednoise"), so.normalise_median_blocks(so.real_dft(x), so.rednoise_bounds(2048, 100)))
