"""Shared helpers for the parity tests (tests/ only)."""
from __future__ import annotations

import os
from concurrent.futures import ProcessPoolExecutor

import numpy as np

from oracle import jerk_oracle as orc

# |P_gpu - P_ref| <= 1e-3 * max(1, P_ref)   (BASELINE.json north_star)
POWER_TOL = 1e-3


def _row_job(args):
    X, z, w, b_lo, b_cnt = args
    return orc.power_row(X, z, w, b_lo, b_cnt)


def oracle_rows(X, zw_list, b_lo, b_cnt, workers=None):
    """Oracle power rows for a list of (z, w), in parallel processes (the oracle itself is single-threaded)."""
    workers = workers or min(8, os.cpu_count() or 1)
    X = np.asarray(X)
    # hand each worker only the bins its taps can reach (|c| + hw <= 508 on the largest grid); a slice that starts
    # at 0 / ends at nbins keeps the true zero-padded spectrum edge
    pad = 700
    lo, hi = max(0, int(b_lo) - pad), min(X.size, int(b_lo) + int(b_cnt) + pad)
    Xs = X[lo:hi]
    jobs = [(Xs, float(z), float(w), int(b_lo) - lo, int(b_cnt)) for z, w in zw_list]
    if workers <= 1 or len(jobs) <= 2:
        return [_row_job(j) for j in jobs]
    import multiprocessing as mp
    with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        return list(ex.map(_row_job, jobs))


def _point_job(args):
    z, w, pieces = args
    tmpl = orc.template(z, w)
    return [orc.power_row(Xs, z, w, b_rel, cnt, tmpl=tmpl) for (Xs, b_rel, cnt) in pieces]


def oracle_point_rows(jobs, cnt=5, workers=None):
    """jobs: [(X, z, w, [b_lo, ...])] -> per job {b_lo: oracle powers of bins b_lo .. b_lo+cnt-1 (2*cnt half-bin values)}.
    One template quadrature per job; the workers get only the few hundred bins each piece can reach."""
    workers = workers or min(8, os.cpu_count() or 1)
    pad = 700
    packed = []
    for X, z, w, b_list in jobs:
        pieces = []
        for b_lo in b_list:
            n = min(cnt, X.size - b_lo)
            lo, hi = max(0, b_lo - pad), min(X.size, b_lo + n + pad)
            pieces.append((np.array(X[lo:hi]), b_lo - lo, n))
        packed.append((float(z), float(w), pieces))
    if workers <= 1 or len(packed) <= 2:
        res = [_point_job(j) for j in packed]
    else:
        import multiprocessing as mp
        with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
            res = list(ex.map(_point_job, packed, chunksize=4))
    return [dict(zip(job[3], r)) for job, r in zip(jobs, res)]


def assert_power_close(p_gpu, p_ref, what=""):
    p_gpu = np.asarray(p_gpu, dtype=np.float64)
    p_ref = np.asarray(p_ref, dtype=np.float64)
    err = np.abs(p_gpu - p_ref) / np.maximum(1.0, p_ref)
    worst = int(np.argmax(err))
    assert err.max() <= POWER_TOL, f"{what}: max |dP|/max(1,P) = {err.max():.3e} at {worst} (gpu {p_gpu.flat[worst]}, ref {p_ref.flat[worst]})"
    return float(err.max())


def oracle_candidates_for_row(X, z, w, thr, b_lo, b_cnt, nbins):
    """Oracle candidates of one row restricted to b in [b_lo, b_lo+b_cnt); neighbours outside the range are real powers."""
    lo = max(0, b_lo - 1)
    hi = min(nbins, b_lo + b_cnt + 1)
    P = orc.power_row(X, z, w, lo, hi - lo)
    left = -np.inf
    right = -np.inf
    j, pw, margin = orc.row_candidates(P, thr, j_offset=2 * lo, left=left, right=right)
    keep = (j >= 2 * b_lo) & (j < 2 * (b_lo + b_cnt))
    # a "candidate" at the artificial range edge is only real if the range edge is the spectrum edge
    if lo > 0:
        keep &= j > 2 * lo
    if hi < nbins:
        keep &= j < 2 * hi - 1
    return j[keep], pw[keep], margin[keep], P, 2 * lo


def _cand_job(args):
    Xs, off, z, w, thr, b_lo, b_cnt, nbins = args
    lo = max(0, b_lo - 1)
    hi = min(nbins, b_lo + b_cnt + 1)
    P = orc.power_row(Xs, z, w, lo - off, hi - lo)       # Xs = X[off : ...] reaches every tap of the range (or the true spectrum edge)
    j, pw, margin = orc.row_candidates(P, thr, j_offset=2 * lo)
    keep = (j >= 2 * b_lo) & (j < 2 * (b_lo + b_cnt))
    if lo > 0:
        keep &= j > 2 * lo
    if hi < nbins:
        keep &= j < 2 * hi - 1
    return j[keep], pw[keep], margin[keep], P, 2 * lo


def oracle_candidates_for_rows(X, jobs, thr, workers=None):
    """oracle_candidates_for_row for many (z, w, b_lo, b_cnt) jobs in parallel processes; each worker gets only the bins
    its taps can reach (a slice that starts at 0 / ends at nbins keeps the true zero-padded spectrum edge)."""
    workers = workers or min(8, os.cpu_count() or 1)
    X = np.asarray(X)
    pad = 700
    packed = []
    for z, w, b_lo, b_cnt in jobs:
        off = max(0, int(b_lo) - 1 - pad)
        end = min(X.size, int(b_lo) + int(b_cnt) + 1 + pad)
        packed.append((X[off:end], off, float(z), float(w), float(thr), int(b_lo), int(b_cnt), int(X.size)))
    if workers <= 1 or len(packed) <= 2:
        return [_cand_job(a) for a in packed]
    import multiprocessing as mp
    with ProcessPoolExecutor(max_workers=workers, mp_context=mp.get_context("spawn")) as ex:
        return list(ex.map(_cand_job, packed))


def compare_row_candidates(gpu_j, gpu_p, ref_j, ref_p, ref_margin, P_ref, j0, thr):
    """Candidate parity for one (z,w) row (BASELINE.json north_star + reading S11).

    - every oracle candidate with P_ref > 1.05*thr must be on the GPU list at the same j, unless its local-max
      margin is a near-tie (< 2e-3 * P), in which case the tied neighbour is accepted;
    - every GPU candidate must be an oracle candidate, or sit where the oracle power is within tolerance of the
      threshold / a near-tie.
    Returns (#matched strong, #strong).
    """
    gset = {int(j): float(p) for j, p in zip(gpu_j, gpu_p)}
    rset = {int(j): (float(p), float(m)) for j, p, m in zip(ref_j, ref_p, ref_margin)}
    strong = matched = 0
    for j, (p, m) in rset.items():
        if p > 1.05 * thr:
            strong += 1
            if j in gset:
                matched += 1
                assert abs(gset[j] - p) <= POWER_TOL * max(1.0, p)
            else:
                assert m < 2e-3 * p and ((j - 1) in gset or (j + 1) in gset), f"oracle candidate j={j} P={p} missing on GPU"
                matched += 1
    for j, p in gset.items():
        if j in rset:
            continue
        pr = P_ref[j - j0]
        tol = POWER_TOL * max(1.0, pr)
        near_thr = abs(pr - thr) <= 2 * tol
        l = P_ref[j - j0 - 1] if j - j0 - 1 >= 0 else -np.inf
        r = P_ref[j - j0 + 1] if j - j0 + 1 < P_ref.size else -np.inf
        near_tie = (pr - l) < 2e-3 * pr or (pr - r) < 2e-3 * pr
        assert abs(p - pr) <= tol, f"GPU candidate j={j} power {p} vs oracle {pr}"
        assert near_thr or near_tie, f"GPU candidate j={j} P={p} is not an oracle candidate (P_ref={pr}, l={l}, r={r})"
    return matched, strong
