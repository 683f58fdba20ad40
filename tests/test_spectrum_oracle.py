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
