"""Host-side sharding of the jerk search over ranks; one process per GPU, torch.distributed plumbing.

The path shards with NO data-path collective: every (segment, template) unit is independent ("processed
independently"; PAPER.md:39 one filter per (z,w)) and the candidate rule is one-dimensional along r inside a (z,w)
row (reading S10).  Two partitions are offered:

  * by trial  (weak scaling, what bench.py --gpus N times): rank r searches spectra r, r+W, r+2W, ... (other DM
    trials) against its own copy of the bank;
  * by template (strong scaling of one spectrum): rank r builds, holds and searches a contiguous range of the flat
    template index ti = iw*nz + iz (jerk_templates_range + jerk_search_candidates_templates); the spectrum is
    broadcast once, candidate lists are concatenated at the end.

The only collectives are the ones around the search: broadcast of the spectrum, gather of the (small) candidate
lists, max-over-ranks of device times.  The harmonic stage shards by r-range of the top harmonic (harmonic_sum_sharded):
whole bank and whole spectrum on every rank, the four stage records gathered and folded at the end.  This module holds no
arithmetic of the method."""
from __future__ import annotations

import numpy as np

CAND_FIELDS = [("j", "<i4"), ("iz", "<i2"), ("iw", "<i2"), ("power", "<f4"), ("flags", "<u4")]


def block_range(n: int, world: int, rank: int) -> tuple[int, int]:
    """Contiguous block partition of range(n): (lo, cnt) of `rank`; the first n % world ranks get one more."""
    if world < 1 or not 0 <= rank < world or n < 0:
        raise ValueError("block_range: bad arguments")
    base, rem = divmod(n, world)
    lo = rank * base + min(rank, rem)
    return lo, base + (1 if rank < rem else 0)


def template_box(nz: int, nw: int, world: int, rank: int) -> tuple[int, int, int, int]:
    """(iz_lo, iz_cnt, iw_lo, iw_cnt) of `rank`: w-rows are split first; when there are more ranks than w-rows the
    ranks that share a w-row block split the z axis."""
    if world <= nw:
        iw_lo, iw_cnt = block_range(nw, world, rank)
        return 0, nz, iw_lo, iw_cnt
    per, extra = divmod(world, nw)          # ranks per w-row; the first `extra` rows get one more
    row, first = 0, 0
    while True:
        k = per + (1 if row < extra else 0)
        if rank < first + k:
            break
        first += k
        row += 1
    iz_lo, iz_cnt = block_range(nz, k, rank - first)
    return iz_lo, iz_cnt, row, 1


def trial_indices(ntrials: int, world: int, rank: int) -> list[int]:
    """Round-robin assignment of independent spectra (DM trials) to ranks."""
    return list(range(rank, ntrials, world))


def broadcast_spectrum(X, src: int = 0, group=None):
    """Broadcast a complex64 spectrum tensor (viewed as float32 pairs) from `src` to every rank, in place."""
    import torch
    import torch.distributed as dist
    buf = torch.view_as_real(X) if X.is_complex() else X
    dist.broadcast(buf, src=src, group=group)
    return X


def gather_candidates(local: np.ndarray, group=None) -> np.ndarray:
    """Concatenate every rank's candidate records (numpy structured array of jerk_cand) on every rank, sorted by
    (iw, iz, j).  Uses all_gather of a padded byte tensor: sizes first, then payload."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    n = torch.tensor([local.shape[0]], dtype=torch.int64, device=dev)
    sizes = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(sizes, n, group=group)
    counts = [int(s.item()) for s in sizes]
    nmax = max(counts) if counts else 0
    itemsize = local.dtype.itemsize
    pad = np.zeros(nmax * itemsize, dtype=np.uint8)
    pad[: local.shape[0] * itemsize] = np.frombuffer(local.tobytes(), dtype=np.uint8)
    mine = torch.from_numpy(pad).to(dev)
    bufs = [torch.empty_like(mine) for _ in range(world)]
    if nmax:
        dist.all_gather(bufs, mine, group=group)
    parts = [np.frombuffer(b.cpu().numpy().tobytes()[: c * itemsize], dtype=local.dtype) for b, c in zip(bufs, counts)]
    out = np.concatenate(parts) if parts else local[:0]
    return np.sort(out, order=["iw", "iz", "j"])


def max_over_ranks(value: float, group=None) -> float:
    """Device-timed milliseconds -> max over ranks (the bench contract's timing rule)."""
    import torch
    import torch.distributed as dist
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    t = torch.tensor([value], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def template_range(ntemplates: int, world: int, rank: int, units=None) -> tuple[int, int]:
    """(ti_lo, ti_cnt) of `rank`: a contiguous split of the flat template index ti = iw*nz + iz.
    Without `units`: equal template COUNTS (at most one template of imbalance).  With `units` (int64[ntemplates] from
    Plan.template_units(): the (segment, template-phase) units a search executes per template -- wide templates run on
    shorter steps and cost more) the cuts are placed at equal WORK: rank r starts at the first template whose cumulative
    units reach r/world of the total, so every rank's share is within one template's units of the mean.  The slowest
    rank sets the step time; on the zmax 200 / wmax 600 grid an equal-count split leaves 6 % between ranks on 8 GPUs."""
    if units is None:
        return block_range(ntemplates, world, rank)
    units = np.asarray(units, dtype=np.int64)
    if units.shape != (ntemplates,) or world < 1 or not 0 <= rank < world:
        raise ValueError("template_range: bad arguments")
    cum = np.concatenate(([0], np.cumsum(units)))                 # cum[t] = units of templates [0, t)
    total = int(cum[-1])
    # cut r = the t whose cum[t] is nearest to r * total / world (integer arithmetic; ties to the smaller t)
    def cut(r):
        if r <= 0:
            return 0
        if r >= world:
            return ntemplates
        target = r * total
        t = int(np.searchsorted(cum * world, target, side="left"))    # first t with cum[t] * world >= target
        if t > 0 and target - int(cum[t - 1]) * world <= int(cum[min(t, ntemplates)]) * world - target:
            t -= 1
        return min(max(t, 0), ntemplates)
    lo, hi = cut(rank), cut(rank + 1)
    return lo, max(hi - lo, 0)


def _units_of(plan):
    """Per-template work of `plan` (Plan.template_units), or None for a plan object that does not report it."""
    f = getattr(plan, "template_units", None)
    return f() if callable(f) else None


def build_bank_shard(plan, group=None):
    """jerk_templates_range for this rank's share: every rank builds and holds only 1/world of the bank."""
    import torch.distributed as dist
    sharded = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    world = dist.get_world_size(group) if sharded else 1
    rank = dist.get_rank(group) if sharded else 0
    ti_lo, ti_cnt = template_range(plan.info.ntemplates, world, rank, _units_of(plan))
    err = None
    try:
        plan.templates_range(ti_lo, ti_cnt)       # ti_cnt == 0 (more ranks than templates) builds the tables only
    except Exception as exc:                      # noqa: BLE001 -- reported below, on every rank
        err = exc
    # a rank must not raise alone: the others would wait for it in the next collective
    if (agree_on_failure(err is not None, group) if sharded else err is not None):
        raise RuntimeError(f"building the bank shard failed on at least one rank (rank {rank}: {err})") from err
    return ti_lo, ti_cnt


def agree_on_failure(flag: bool, group=None) -> bool:
    """True on every rank iff `flag` is set on any rank (all_reduce MAX): a rank must never raise before a collective
    the others are about to enter."""
    import torch
    import torch.distributed as dist
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    t = torch.tensor([1 if flag else 0], dtype=torch.int32, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return bool(t.item())


def search_candidates_sharded(plan, d_spec, threshold, max_cands: int = 1 << 20, group=None, src: int = 0) -> np.ndarray:
    """Strong-scaling search of ONE spectrum over the ranks of `group` (partition by template):
    the spectrum is broadcast from `src`, every rank searches its flat template range
    (jerk_search_candidates_templates) against the part of the bank it holds (build_bank_shard, or the whole bank), and
    the candidate lists are concatenated on every rank (sorted by (iw, iz, j)).  Without an initialised process group
    it is the whole-grid search on this rank.  No collective touches the search itself: the candidate rule is
    one-dimensional along r inside a (z,w) row (reading S10).  A candidate- or seam-buffer overflow on any
    rank raises on EVERY rank (the flag is max-reduced before the gather)."""
    import torch.distributed as dist
    from . import binding
    sharded = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    world = dist.get_world_size(group) if sharded else 1
    rank = dist.get_rank(group) if sharded else 0
    if sharded:
        broadcast_spectrum(d_spec, src=src, group=group)
    ti_lo, ti_cnt = template_range(plan.info.ntemplates, world, rank, _units_of(plan))
    d_c, d_n = plan.search_candidates_templates(d_spec, threshold, ti_lo, ti_cnt, max_cands)
    n = int(d_n.item()) & binding.SEAM_OVERFLOW
    overflow = n > max_cands          # includes the seam-overflow sentinel
    if (agree_on_failure(overflow, group) if sharded else overflow):
        raise RuntimeError(f"candidate or seam buffer overflow (rank {rank}: count {n}, max_cands {max_cands})")
    local, _ = binding.candidates_to_numpy(d_c, d_n)
    if sharded:
        return gather_candidates(local, group=group)
    return np.sort(local, order=["iw", "iz", "j"])


def fold_stage_records(records: np.ndarray) -> np.ndarray:
    """records: structured array [nranks][nstages] of jerk_cand stage tops (j = -1: nothing above the threshold in that
    rank's range).  Per stage the record with the largest power wins; equal powers go to the smallest (iw, iz, j) -- the
    tie rule of jerk_harmonic_sum (include/jerk.h), so the fold of disjoint ranges equals the single call."""
    records = np.asarray(records)
    out = records[0].copy()
    for s in range(records.shape[1]):
        best = None
        for r in range(records.shape[0]):
            c = records[r, s]
            if int(c["j"]) < 0:
                continue
            key = (-float(c["power"]), int(c["iw"]), int(c["iz"]), int(c["j"]))
            if best is None or key < best[0]:
                best = (key, c)
        if best is None:
            out[s] = records[0, s]
            out[s]["j"], out[s]["iz"], out[s]["iw"], out[s]["power"], out[s]["flags"] = -1, 0, 0, 0.0, 0
        else:
            out[s] = best[1]
    return out


def harmonic_sum_sharded(plan, d_spec, harms=(1, 2, 4, 8), thresholds=(25.0, 35.0, 50.0, 75.0), group=None, src: int = 0,
                         scratch_bytes=None) -> np.ndarray:
    """The harmonic-sum stage of ONE spectrum over the ranks of `group` (r-range partition): the spectrum is
    broadcast from `src`, rank r runs jerk_harmonic_sum_range on the contiguous block r of the top-harmonic bins (the
    sub-harmonic sources of a range lie below it, so every rank needs the whole spectrum and the whole bank; work per
    top-harmonic bin is uniform, so equal blocks are balanced), the per-rank stage records (4 x 16 bytes) are all-gathered and
    folded with the tie rule.  Returns the same array on every rank, equal to plan.harmonic_sum on one GPU.  A failure
    on any rank raises on every rank."""
    import torch
    import torch.distributed as dist
    sharded = dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1
    world = dist.get_world_size(group) if sharded else 1
    rank = dist.get_rank(group) if sharded else 0
    if sharded:
        broadcast_spectrum(d_spec, src=src, group=group)
    r_lo, r_cnt = block_range(int(plan.info.nbins), world, rank)
    err, mine = None, None
    try:
        mine = plan.harmonic_sum(d_spec, harms, thresholds, scratch_bytes=scratch_bytes, r_lo=r_lo, r_cnt=r_cnt)
    except Exception as exc:                      # noqa: BLE001 -- agreed below
        err = exc
    if (agree_on_failure(err is not None, group) if sharded else err is not None):
        raise RuntimeError(f"harmonic stage failed on at least one rank (rank {rank}: {err})") from err
    if not sharded:
        return fold_stage_records(mine[None, :])
    dev = torch.device("cuda", torch.cuda.current_device()) if dist.get_backend(group) == "nccl" else torch.device("cpu")
    buf = torch.from_numpy(np.frombuffer(mine.tobytes(), dtype=np.uint8).copy()).to(dev)
    bufs = [torch.empty_like(buf) for _ in range(world)]
    dist.all_gather(bufs, buf, group=group)
    recs = np.stack([np.frombuffer(b.cpu().numpy().tobytes(), dtype=mine.dtype) for b in bufs])
    return fold_stage_records(recs)
