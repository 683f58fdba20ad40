"""Seeded synthetic workloads for the jerk-search hot path.

This module holds NONE of the method's arithmetic (no response, no template, no
correlation): it only makes the *input* both the CUDA path and the oracle are fed —
a block-normalised complex64 spectrum of white noise plus injected chirped
sinusoids — and names the five BASELINE.json configs.  The paper names no data
set ("a 10 minute observation"); these inputs stand in for it.

Recipe: rng = Generator(PCG64(1911013530 + config)); noise =
standard_normal(N, float32); each signal a*cos(2 pi (r u + z u^2/2 + w u^3/6)),
u = n/N, a = sqrt(4 P / N), evaluated in float64; X = rfft, bins 0..N/2-1; every
1000-bin block divided by sqrt(mean |X|^2) of that block; cast to complex64.
Signal parameters are drawn from the same rng after the noise, in order.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 1911013530


@dataclass
class Config:
    name: str
    index: int               # 1..5 (BASELINE.json configs[index-1])
    log2n: int
    zmax: float
    dz: float
    wmax: float
    dw: float
    seg_len: int
    threshold: float
    n_signals: int
    harmonics: int = 1
    numbetween: int = 2
    signals: list = field(default_factory=list)   # filled by make_spectrum: (r0, z0, w0, P)

    @property
    def n(self) -> int:
        return 1 << self.log2n

    @property
    def nbins(self) -> int:
        return self.n // 2

    @property
    def nz(self) -> int:
        return int(round(2 * self.zmax / self.dz)) + 1

    @property
    def nw(self) -> int:
        return int(round(2 * self.wmax / self.dw)) + 1

    @property
    def points(self) -> int:
        return self.numbetween * self.nbins * self.nz * self.nw


def config(index: int) -> Config:
    if index == 1:
        return Config("tiny", 1, 16, 20, 2, 60, 20, 1024, 20.0, 1)
    if index == 2:
        return Config("small", 2, 21, 100, 2, 300, 20, 2048, 25.0, 3)
    if index == 3:
        return Config("full", 3, 23, 200, 2, 600, 20, 4096, 25.0, 5)
    if index == 4:
        return Config("long", 4, 25, 200, 2, 600, 20, 8192, 25.0, 8)
    if index == 5:
        return Config("harmonic", 5, 23, 200, 2, 600, 20, 4096, 25.0, 4, harmonics=8)
    raise ValueError("config index must be 1..5")


def _draw_signals(cfg: Config, rng: np.random.Generator) -> list:
    nb = cfg.nbins
    sig = []
    if cfg.index == 1:
        return [(5000.25, 10.0, 40.0, 50.0)]
    if cfg.index == 2:
        for _ in range(3):
            r0 = round(2 * rng.uniform(1e4, 1e6)) / 2
            z0 = 2.0 * rng.integers(-50, 51)
            w0 = 20.0 * rng.integers(-15, 16)
            sig.append((r0, z0, w0, float(rng.uniform(30, 80))))
        return sig
    if cfg.index in (3, 4):
        for i in range(cfg.n_signals):
            r0 = round(2 * rng.uniform(1e4, nb - 1e4)) / 2
            z0 = 2.0 * rng.integers(-100, 101)
            w0 = 20.0 * rng.integers(-30, 31)
            p = float(rng.uniform(30, 80))
            if cfg.index == 4 and i >= cfg.n_signals - 2:
                p = 28.0
            sig.append((r0, z0, w0, p))
        return sig
    for _ in range(cfg.n_signals):          # config 5: fundamentals; harmonic k at k*(r0,z0,w0), amplitude a/k
        r0 = round(2 * rng.uniform(1e4, nb / 8 - 1e3)) / 2
        z0 = 2.0 * rng.integers(-12, 13)
        w0 = 20.0 * rng.integers(-3, 4)
        sig.append((r0, z0, w0, float(rng.uniform(60, 100))))
    return sig


def block_normalise(X: np.ndarray, block: int = 1000) -> np.ndarray:
    """Divide each consecutive `block`-bin block by sqrt(mean |X|^2) of that block (reading S15)."""
    out = np.array(X, dtype=np.complex128)
    for a in range(0, out.size, block):
        seg = out[a:a + block]
        m = np.mean(seg.real ** 2 + seg.imag ** 2)
        if m > 0:
            seg /= np.sqrt(m)
    return out


def chirp_series(n: int, r0: float, z0: float, w0: float, amp: float) -> np.ndarray:
    """amp * cos(2 pi (r0 u + z0 u^2/2 + w0 u^3/6)), u = i/n, float64 (the injected signal model)."""
    u = np.arange(n, dtype=np.float64) / n
    ph = r0 * u + z0 * u * u / 2.0 + w0 * u * u * u / 6.0
    ph -= np.floor(ph)
    return amp * np.cos(2.0 * np.pi * ph)


def make_series(cfg: Config, noise: bool = True, trial: int = 0) -> np.ndarray:
    """float32 time series of config `cfg` (noise + injected signals); fills cfg.signals.  The input of the
    spectrum-preparation stage and the first half of make_spectrum."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + cfg.index + 1000 * trial))
    n = cfg.n
    x = rng.standard_normal(n, dtype=np.float32).astype(np.float64)
    if not noise:
        x[:] = 0.0
    cfg.signals = _draw_signals(cfg, rng)
    for (r0, z0, w0, p) in cfg.signals:
        a = np.sqrt(4.0 * p / n)
        for k in range(1, cfg.harmonics + 1):
            x += chirp_series(n, k * r0, k * z0, k * w0, a / k)
    return x.astype(np.float32)


def make_spectrum(cfg: Config, noise: bool = True, trial: int = 0) -> np.ndarray:
    """complex64 spectrum X[0..nbins) of config `cfg`; fills cfg.signals.

    `trial` > 0 gives an independent realisation of the same workload (another "DM trial": bench.py uses one per
    rank); trial 0 is the configuration the parity tests pin."""
    n = cfg.n
    x = make_series(cfg, noise, trial).astype(np.float64)
    X = np.fft.rfft(x)[: n // 2]
    if noise:
        X = block_normalise(X)
    else:
        X = X * (2.0 / n)         # unit-amplitude signal -> unit coherent amplitude
    return X.astype(np.complex64)


def random_spectrum(nbins: int, seed: int) -> np.ndarray:
    """Unit-variance complex Gaussian spectrum (for invariance / statistics tests)."""
    rng = np.random.Generator(np.random.PCG64(seed))
    re = rng.standard_normal(nbins)
    im = rng.standard_normal(nbins)
    return ((re + 1j * im) / np.sqrt(2.0)).astype(np.complex64)
