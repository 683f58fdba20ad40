"""CPU oracle for the Fourier-domain jerk-search hot path (arXiv 1911.01353).

TEST INFRASTRUCTURE ONLY.  Nothing in the product path may import this module:
only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may call it.  It shares no code with the CUDA path.

What it is: the *plain definition* of what the hot path computes, in float64,
with no segmentation, no FFT and no blocking.  The paper's method (overlap-and-save
FFT convolution with a bank of (z, w) matched filters) reaches,
up to rounding, exactly the direct correlation sum written here, so the oracle is
that sum written out (BASELINE.json north_star: "direct time-domain correlation
with templates from its own numerical integration").

Notation follows PAPER.md:39 (z = fdot*T^2, w = fddot*T^3) and SURVEY.md section 8(c):

  B  response   R_{z,w}(q) = int_0^1 exp(2*pi*i*(z u^2/2 + w u^3/6 - q u)) du
  C  template   centre c(z,w), half-width hw(z,w), taps on the half-bin lattice
  D  plane      A[j; z,w] = sum_m X[b+m] * conj(R_{z,w}(m - p/2)),  j = 2b+p ;  P = |A|^2
  E  candidates P > thr, P > P[j-1], P >= P[j+1] within one (z,w) row
  F  harmonic   S_h(j,iz',iw') = sum_{k=1..h} P[rnd(j k/h); rnd(iz' k/h), rnd(iw' k/h)]
  G  row S/N    mean and (population) standard deviation of P over the 2*nbins points of one (z,w) row;
                snr = (P - mean) / std; a candidate is kept iff snr > snr_threshold
  H  sifting    a candidate is kept iff no other candidate within |dj|<=wj, |diz|<=wz, |diw|<=ww beats it
                (larger power; ties -> smaller (iw, iz, j))

Pins (tests/test_oracle_pins.py): closed-form sinc (z=w=0), Fresnel closed form (w=0),
conjugate symmetry, Parseval unit energy, quadrature refinement, exact-grid recovery of a
noise-free injection, brute-force de-chirped DFT on a tiny input, noise statistics,
shift invariance, brute-force harmonic sum on a toy volume.  No function here is
"parity unpinned"; the *rules* of E (tie handling) and F (rounding) are readings of
BASELINE.json (readings S10/S13) and are pinned only by brute force.
"""
from __future__ import annotations

import math

import numpy as np
from numpy.polynomial.legendre import leggauss

_GL_ORDER = 16


# --------------------------------------------------------------------------- B: response
def response(z: float, w: float, q, panels: int | None = None, order: int = _GL_ORDER) -> np.ndarray:
    """R_{z,w}(q) for an array of offsets q (BASELINE.json north_star item (1)).

    Composite Gauss-Legendre on [0,1].  The integrand's phase rate is
    |g(u) - q| cycles per unit u, g(u) = z u + w u^2/2; with one cycle per panel at
    most and 16 nodes per panel the rule is converged to rounding (pinned by the
    refinement test).
    """
    q = np.atleast_1d(np.asarray(q, dtype=np.float64))
    if panels is None:
        # d/du of the phase (in cycles) is g(u) - q with g(u) = z u + w u^2/2 in [g_lo, g_hi]
        g_lo, g_hi = excursion(z, w)
        rate = max(abs(float(q.max()) - g_lo), abs(float(q.min()) - g_lo),
                   abs(float(q.max()) - g_hi), abs(float(q.min()) - g_hi)) if q.size else 0.0
        panels = int(math.ceil(rate)) + 8
    x, wt = leggauss(order)
    h = 1.0 / panels
    left = np.arange(panels, dtype=np.float64) * h
    u = (left[:, None] + (x[None, :] + 1.0) * (0.5 * h)).ravel()          # nodes in (0,1)
    wu = np.tile(wt * (0.5 * h), panels)                                   # weights
    chirp = z * u * u / 2.0 + w * u * u * u / 6.0
    out = np.empty(q.shape, dtype=np.complex128)
    # chunk over q to bound memory; plain sum of weight * exp(i*phase)
    chunk = max(1, int(4_000_000 // max(1, u.size)))
    for a in range(0, q.size, chunk):
        qq = q[a:a + chunk]
        phase = 2.0 * np.pi * (chirp[None, :] - qq[:, None] * u[None, :])
        out[a:a + chunk] = (np.exp(1j * phase) * wu[None, :]).sum(axis=1)
    return out


# --------------------------------------------------------------------------- C: template
def _round_half_away(v: float) -> int:
    return int(math.copysign(math.floor(abs(v) + 0.5), v)) if v != 0 else 0


def excursion(z: float, w: float) -> tuple[float, float]:
    """min and max over u in [0,1] of the frequency excursion g(u) = z u + w u^2/2."""
    vals = [0.0, z + w / 2.0]
    if w != 0.0:
        us = -z / w
        if 0.0 < us < 1.0:
            vals.append(-z * z / (2.0 * w))
    return min(vals), max(vals)


def centre(z: float, w: float) -> int:
    """c(z,w): midpoint of the excursion, rounded half away from zero (reading S3/S4)."""
    lo, hi = excursion(z, w)
    return _round_half_away((lo + hi) / 2.0)


def halfwidth(z: float, w: float) -> int:
    """hw(z,w) = ceil(|z|/2 + |w|/4) + 8 bins (BASELINE.json configs[0])."""
    return int(math.ceil(abs(z) / 2.0 + abs(w) / 4.0)) + 8


def template(z: float, w: float) -> tuple[int, int, np.ndarray]:
    """(c, hw, lattice) with lattice[i] = R_{z,w}(c - hw + i/2), i = 0..4hw.

    Even i are the phase-0 taps (q integer, m = c-hw..c+hw), odd i the phase-1
    taps (q = m - 1/2, m = c-hw+1..c+hw).  No window, no renormalisation (S6).
    """
    c = centre(z, w)
    hw = halfwidth(z, w)
    q = c - hw + 0.5 * np.arange(4 * hw + 1)
    return c, hw, response(z, w, q)


def phase_taps(c: int, hw: int, lattice: np.ndarray, p: int) -> tuple[np.ndarray, np.ndarray]:
    """(m, R(m - p/2)) for the phase-p taps of a template."""
    if p == 0:
        m = np.arange(c - hw, c + hw + 1)
        return m, lattice[0::2]
    m = np.arange(c - hw + 1, c + hw + 1)
    return m, lattice[1::2]


# --------------------------------------------------------------------------- grid
def grid_values(vmax: float, dv: float) -> np.ndarray:
    """-vmax, -vmax+dv, ..., +vmax  (nz = 2*zmax/dz + 1)."""
    n = int(round(2.0 * vmax / dv)) + 1 if dv > 0 else 1
    return -vmax + dv * np.arange(n, dtype=np.float64)


# --------------------------------------------------------------------------- D: plane
def amplitude_row(X: np.ndarray, z: float, w: float, b_lo: int = 0, b_cnt: int | None = None,
                  tmpl=None) -> np.ndarray:
    """A[j; z,w] for j in [2*b_lo, 2*(b_lo+b_cnt)), by direct summation over the taps.

    X is the complex spectrum, X[k] = 0 outside [0, nbins) (reading S9).
    """
    X = np.asarray(X, dtype=np.complex128)
    nbins = X.size
    if b_cnt is None:
        b_cnt = nbins - b_lo
    c, hw, lattice = tmpl if tmpl is not None else template(z, w)
    pad = abs(c) + hw + 1
    Xp = np.zeros(b_cnt + 2 * pad, dtype=np.complex128)
    # Xp[i] = X[b_lo - pad + i]
    src_lo = max(0, b_lo - pad)
    src_hi = min(nbins, b_lo + b_cnt + pad)
    if src_hi > src_lo:
        Xp[src_lo - (b_lo - pad): src_hi - (b_lo - pad)] = X[src_lo:src_hi]
    A = np.zeros(2 * b_cnt, dtype=np.complex128)
    for p in (0, 1):
        ms, taps = phase_taps(c, hw, lattice, p)
        acc = np.zeros(b_cnt, dtype=np.complex128)
        for m, r in zip(ms, taps):
            acc += Xp[pad + m: pad + m + b_cnt] * np.conj(r)
        A[p::2] = acc
    return A


def power_row(X, z, w, b_lo=0, b_cnt=None, tmpl=None) -> np.ndarray:
    A = amplitude_row(X, z, w, b_lo, b_cnt, tmpl)
    return A.real * A.real + A.imag * A.imag


def plane(X, zmax, dz, wmax, dw, b_lo=0, b_cnt=None) -> np.ndarray:
    """P[iw][iz][j] (float64) over the whole (z,w) grid for the bin range given."""
    zs, ws = grid_values(zmax, dz), grid_values(wmax, dw)
    nb = (np.asarray(X).size - b_lo) if b_cnt is None else b_cnt
    out = np.empty((ws.size, zs.size, 2 * nb), dtype=np.float64)
    for iw, w in enumerate(ws):
        for iz, z in enumerate(zs):
            out[iw, iz] = power_row(X, float(z), float(w), b_lo, b_cnt)
    return out


# --------------------------------------------------------------------------- E: candidates
def row_candidates(P_row: np.ndarray, threshold: float, j_offset: int = 0,
                   left: float = -np.inf, right: float = -np.inf):
    """Local-max candidates of one (z,w) row.

    (j, P, margin): P > threshold, P > P[j-1], P >= P[j+1]; the row's outer neighbours
    are `left` / `right` (-inf at the spectrum ends, S10).  margin = min(P-P[j-1], P-P[j+1])
    is reported so that near-ties can be recognised by the harness (S11).
    """
    P = np.asarray(P_row, dtype=np.float64)
    prev = np.concatenate(([left], P[:-1]))
    nxt = np.concatenate((P[1:], [right]))
    sel = (P > threshold) & (P > prev) & (P >= nxt)
    idx = np.nonzero(sel)[0]
    margin = np.minimum(P[idx] - prev[idx], P[idx] - nxt[idx])
    return idx + j_offset, P[idx], margin


# --------------------------------------------------------------------------- F: harmonic sum
def rnd_frac(a: int, k: int, h: int) -> int:
    """round-half-away-from-zero of a*k/h in integer arithmetic (reading S13)."""
    s = -1 if a < 0 else 1
    return s * ((2 * abs(a) * k + h) // (2 * h))


def harmonic_sum_point(P_lookup, j: int, izs: int, iws: int, h: int) -> float:
    """S_h at the top-harmonic position (j, iz', iw') (signed grid indices).

    P_lookup(j, iz', iw') returns the plane power at a grid point.
    """
    s = 0.0
    for k in range(1, h + 1):
        s += P_lookup(rnd_frac(j, k, h), rnd_frac(izs, k, h), rnd_frac(iws, k, h))
    return s


def harmonic_sum_volume(P: np.ndarray, h: int) -> np.ndarray:
    """S_h over a whole volume P[iw][iz][j] (small inputs only: pure loops over k).

    Signed indices iz' = iz - (nz-1)/2, iw' = iw - (nw-1)/2; j is the absolute half-bin index.
    """
    nw, nz, nj = P.shape
    cz, cw = (nz - 1) // 2, (nw - 1) // 2
    S = np.zeros_like(P, dtype=np.float64)
    jj = np.arange(nj)
    for k in range(1, h + 1):
        js = (2 * jj * k + h) // (2 * h)
        for iw in range(nw):
            iwk = rnd_frac(iw - cw, k, h) + cw
            for iz in range(nz):
                izk = rnd_frac(iz - cz, k, h) + cz
                S[iw, iz] += P[iwk, izk, js]
    return S


# --------------------------------------------------------------------------- G: row statistics and S/N
def row_stats(P) -> tuple[float, float]:
    """(sum of P, sum of P^2) over every point of one (z,w) row, float64 (what the fused kernel accumulates)."""
    P = np.asarray(P, dtype=np.float64)
    return float(np.sum(P)), float(np.sum(P * P))


def row_mean_std(P) -> tuple[float, float]:
    """Mean and population standard deviation of the row: the paper's "mean and standard deviation" of the output
    (PAPER.md:45), taken per (z,w) row over all 2*nbins points."""
    P = np.asarray(P, dtype=np.float64)
    s1, s2 = row_stats(P)
    mean = s1 / P.size
    var = s2 / P.size - mean * mean
    return mean, math.sqrt(var) if var > 0.0 else 0.0


def snr(power, mean: float, std: float):
    """(P - mean) / std."""
    return (np.asarray(power, dtype=np.float64) - mean) / std


def snr_filter(j, power, mean: float, std: float, snr_threshold: float):
    """Candidates of one row (arrays j, power) with snr > snr_threshold: (j, power, snr).  A row with std = 0 keeps nothing."""
    j = np.asarray(j)
    power = np.asarray(power, dtype=np.float64)
    if not std > 0.0:
        return j[:0], power[:0], power[:0]
    s = snr(power, mean, std)
    keep = s > snr_threshold
    return j[keep], power[keep], s[keep]


# --------------------------------------------------------------------------- H: cross-row sifting
def sift(cands, wj: int, wz: int, ww: int) -> list:
    """Non-maximum suppression over a list of (j, iz, iw, power) tuples, written as the plain double loop.

    A candidate survives iff no OTHER candidate with |dj| <= wj, |diz| <= wz, |diw| <= ww beats it: larger power, or
    equal power and smaller (iw, iz, j).  Returns the survivors sorted by (iw, iz, j)."""
    cands = [(int(j), int(iz), int(iw), float(p)) for (j, iz, iw, p) in cands]
    out = []
    for a_i, a in enumerate(cands):
        alive = True
        for b_i, b in enumerate(cands):
            if b_i == a_i:
                continue
            if abs(b[0] - a[0]) <= wj and abs(b[1] - a[1]) <= wz and abs(b[2] - a[2]) <= ww:
                if b[3] > a[3] or (b[3] == a[3] and (b[2], b[1], b[0]) < (a[2], a[1], a[0])):
                    alive = False
                    break
        if alive:
            out.append(a)
    return sorted(out, key=lambda c: (c[2], c[1], c[0]))


# --------------------------------------------------------------------------- I: numbetween = 1
def power_row_nb1(X: np.ndarray, z: float, w: float, b_lo: int = 0, b_cnt: int | None = None, tmpl=None) -> np.ndarray:
    """P[b; z,w] = |sum_m X[b+m] conj(R_{z,w}(m))|^2 on the integer bins b in [b_lo, b_lo+b_cnt) only: the
    numbetween = 1 search keeps the phase-0 tap set of section C (m = c-hw..c+hw, q = m) and drops the half-bin
    phase (the FDAS-style option; SURVEY.md 8(f) N4 "numbetween options").  X[k] = 0 outside [0, nbins)."""
    X = np.asarray(X, dtype=np.complex128)
    nbins = X.size
    if b_cnt is None:
        b_cnt = nbins - b_lo
    c, hw, lattice = tmpl if tmpl is not None else template(z, w)
    out = np.zeros(b_cnt, dtype=np.float64)
    for i in range(b_cnt):
        b = b_lo + i
        acc = 0.0 + 0.0j
        for m in range(c - hw, c + hw + 1):
            k = b + m
            if 0 <= k < nbins:
                acc += X[k] * np.conj(lattice[2 * (m - (c - hw))])
        out[i] = acc.real * acc.real + acc.imag * acc.imag
    return out

