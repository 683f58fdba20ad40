"""CPU oracle for the spectrum-preparation stage upstream of the jerk search.

TEST INFRASTRUCTURE ONLY (same rules as jerk_oracle.py): only ``tests/``, ``__graft_entry__.smoke()`` and
``bench.py``'s oracle legs may import it; it shares no code with the CUDA path or with ``workloads.py``.

What it computes (BASELINE.json configs[0]: "The real FFT gives 32768 complex bins, normalised to unit mean power
per 1000-bin block"; PAPER.md:15 the search works on the Fourier transform of the de-dispersed time series;
DESIGN.md reading S15):

  A  X[k] = sum_{n=0}^{N-1} x[n] exp(-2 pi i k n / N),  k = 0 .. N/2 - 1      (DC kept, Nyquist bin dropped)
  B  for every consecutive block of `block` bins (the last one may be shorter):  X[k] /= sqrt(mean_{k in block} |X[k]|^2)
     (a block whose mean power is 0 is left as it is)

A is the plain definition; `real_dft` evaluates it with numpy's rfft in float64 (a library primitive used as a
step) and `real_dft_direct` writes the sum out for tiny N, which pins the former (tests/test_spectrum_oracle.py).

Normalisation variants (SURVEY.md 8(f) N1 "median-based and red-noise variants"; the spectrum of a real
de-dispersed series, whose noise floor is neither white nor free of strong narrow signals; the paper gives no recipe,
so both are readings, listed in DESIGN.md):

  B-median    per block: X[k] /= sqrt(median_{k in block} |X[k]|^2 / ln 2).  For noise powers that are exponentially
              distributed (complex Gaussian bins) the median is ln 2 times the mean, so this equals B on pure noise
              but is not inflated by a few strong bins (an even count takes the mean of the two middle values;
              a block whose median is 0 is left as it is).
  B-rednoise  the same with blocks whose length grows with frequency, so that a steep low-frequency (red) noise
              slope is followed: block i covers [k_i, k_i + len_i), k_0 = 0, len_0 = 6,
              len_{i+1} = min(block, len_i + max(1, len_i // 8)); the last block ends at the last bin.
"""
from __future__ import annotations

import numpy as np


def real_dft_direct(x) -> np.ndarray:
    """Definition A by direct summation, O(N^2), float64: for pins on tiny inputs only."""
    x = np.asarray(x, dtype=np.float64)
    n = x.size
    out = np.zeros(n // 2, dtype=np.complex128)
    for k in range(n // 2):
        acc = 0.0 + 0.0j
        for i in range(n):
            ang = -2.0 * np.pi * ((k * i) % n) / n
            acc += x[i] * complex(np.cos(ang), np.sin(ang))
        out[k] = acc
    return out


def real_dft(x) -> np.ndarray:
    """Definition A: bins 0 .. N/2-1 of the DFT of the real series x (float64 arithmetic)."""
    x = np.asarray(x, dtype=np.float64)
    if x.ndim != 1 or x.size < 2 or x.size % 2:
        raise ValueError("real_dft: x must be 1-D with an even number of samples")
    return np.fft.rfft(x)[: x.size // 2]


def block_powers(X, block: int = 1000) -> np.ndarray:
    """Mean |X|^2 of every consecutive `block`-bin block (last block may be shorter)."""
    X = np.asarray(X, dtype=np.complex128)
    nblk = (X.size + block - 1) // block
    out = np.zeros(nblk, dtype=np.float64)
    for b in range(nblk):
        seg = X[b * block:(b + 1) * block]
        total = 0.0
        for v in seg:
            total += v.real * v.real + v.imag * v.imag
        out[b] = total / seg.size
    return out


def normalise_blocks(X, block: int = 1000) -> np.ndarray:
    """Step B."""
    X = np.array(X, dtype=np.complex128)
    m = block_powers(X, block)
    for b in range(m.size):
        if m[b] > 0.0:
            X[b * block:(b + 1) * block] = X[b * block:(b + 1) * block] / np.sqrt(m[b])
    return X


def prepare_spectrum(x, block: int = 1000) -> np.ndarray:
    """A then B: the normalised complex spectrum (complex128, N/2 bins) handed to the jerk search."""
    return normalise_blocks(real_dft(x), block)


# --------------------------------------------------------------------------- normalisation variants (median, red noise)
def median_plain(values) -> float:
    """Median by sorting (a library sort as the step): middle element, or the mean of the two middle ones."""
    v = np.sort(np.asarray(values, dtype=np.float64))
    n = v.size
    if n == 0:
        raise ValueError("median of nothing")
    return float(v[n // 2]) if n % 2 else float(0.5 * (v[n // 2 - 1] + v[n // 2]))


def uniform_bounds(nbins: int, block: int) -> list:
    """Block starts 0, block, 2 block, ... and the end nbins."""
    return list(range(0, nbins, block)) + [nbins]


def rednoise_bounds(nbins: int, block: int) -> list:
    """Block starts of B-rednoise and the end nbins: lengths 6, 7, 8, ... growing by len // 8 (at least 1) up to `block`."""
    if block < 8:
        raise ValueError("rednoise_bounds: block must be >= 8")
    bounds, k, ln = [0], 0, 6
    while k + ln < nbins:
        k += ln
        bounds.append(k)
        ln = min(block, ln + max(1, ln // 8))
    bounds.append(nbins)
    return bounds


def normalise_median_blocks(X, bounds) -> np.ndarray:
    """Every block [bounds[i], bounds[i+1]) divided by sqrt(median |X|^2 / ln 2) of that block."""
    X = np.array(X, dtype=np.complex128)
    ln2 = float(np.log(2.0))
    for a, b in zip(bounds[:-1], bounds[1:]):
        seg = X[a:b]
        med = median_plain(seg.real * seg.real + seg.imag * seg.imag)
        if med > 0.0:
            X[a:b] = seg / np.sqrt(med / ln2)
    return X


def prepare_spectrum_mode(x, block: int = 1000, mode: str = "mean") -> np.ndarray:
    """A then the chosen normalisation: "mean" (B), "median" (B-median), "rednoise" (B-rednoise)."""
    X = real_dft(x)
    if mode == "mean":
        return normalise_blocks(X, block)
    if mode == "median":
        return normalise_median_blocks(X, uniform_bounds(X.size, block))
    if mode == "rednoise":
        return normalise_median_blocks(X, rednoise_bounds(X.size, block))
    raise ValueError("mode must be mean, median or rednoise")

