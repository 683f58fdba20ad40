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
