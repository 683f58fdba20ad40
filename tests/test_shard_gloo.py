"""Host-side multi-rank logic on CPU: world_size-2 (and 3) gloo process groups.  No GPU, no kernels:
the per-rank "search" is replaced by slicing a fixed synthetic candidate list by template range, which is exactly what
jerk_search_candidates_templates guarantees (tests/test_gpu_parity.py::test_candidates_range_union checks that on the GPU)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1911_01353_b200 import shard


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _fake_candidates(nz, nw, n=500, seed=5):
    rng = np.random.default_rng(seed)
    c = np.zeros(n, dtype=shard.CAND_FIELDS)
    c["j"] = rng.integers(0, 1 << 20, n)
    c["iz"] = rng.integers(0, nz, n)
    c["iw"] = rng.integers(0, nw, n)
    c["power"] = rng.uniform(25, 90, n).astype(np.float32)
    return np.unique(c)


def _worker(rank, world, port, nz, nw, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        full = _fake_candidates(nz, nw)
        iz_lo, iz_cnt, iw_lo, iw_cnt = shard.template_box(nz, nw, world, rank)
        m = (full["iz"] >= iz_lo) & (full["iz"] < iz_lo + iz_cnt) & (full["iw"] >= iw_lo) & (full["iw"] < iw_lo + iw_cnt)
        merged = shard.gather_candidates(full[m])
        ok_merge = np.array_equal(merged, np.sort(full, order=["iw", "iz", "j"]))
        # spectrum broadcast: rank 0 holds the data, the others zeros
        X = torch.zeros(1000, dtype=torch.complex64)
        if rank == 0:
            X = torch.view_as_complex(torch.arange(2000, dtype=torch.float32).reshape(1000, 2).contiguous())
        shard.broadcast_spectrum(X, src=0)
        ok_bcast = bool(torch.view_as_real(X)[-1, 1] == 1999.0)
        # the whole strong-scaling entry point against a stand-in plan whose "search" slices the fixed list by box
        class _Info:
            pass

        class _FakePlan:
            info = _Info()
            overflow_rank = -1

            build_fail_rank = -1

            def templates_range(self, ti_lo, ti_cnt):
                if rank == self.build_fail_rank:
                    raise ValueError("stand-in build failure")
                self.bank_range = (ti_lo, ti_cnt)

            def search_candidates_templates(self, d_spec, thr, ti_lo, ti_cnt, max_cands):
                assert (ti_lo, ti_cnt) == self.bank_range      # a rank searches exactly the part of the bank it built
                ti = full["iw"].astype(np.int64) * nz + full["iz"]
                sel = full[(ti >= ti_lo) & (ti < ti_lo + ti_cnt) & (full["power"] > thr)]
                buf = np.zeros(max_cands * 16, dtype=np.uint8)
                buf[: sel.size * 16] = np.frombuffer(sel.tobytes(), dtype=np.uint8)
                count = sel.size if rank != self.overflow_rank else max_cands + 1
                return torch.from_numpy(buf), torch.tensor([count], dtype=torch.int64)

        _FakePlan.info.nz, _FakePlan.info.nw, _FakePlan.info.ntemplates = nz, nw, nz * nw
        plan = _FakePlan()
        lo, cnt = shard.build_bank_shard(plan)
        assert (lo, cnt) == shard.template_range(nz * nw, world, rank)
        merged2 = shard.search_candidates_sharded(plan, X, 40.0, max_cands=4096)
        want2 = np.sort(full[full["power"] > 40.0], order=["iw", "iz", "j"])
        ok_merge = ok_merge and np.array_equal(merged2, want2) and bool(torch.view_as_real(X)[-1, 1] == 1999.0)
        # an overflow on ONE rank raises on EVERY rank (agreed collectively before the gather: nobody hangs)
        plan.overflow_rank = world - 1
        try:
            shard.search_candidates_sharded(plan, X, 40.0, max_cands=4096)
            ok_merge = False
        except RuntimeError:
            pass
        plan.overflow_rank = -1
        # a bank build that fails on ONE rank raises on EVERY rank before anybody enters the next collective
        plan.build_fail_rank = 0
        try:
            shard.build_bank_shard(plan)
            ok_merge = False
        except RuntimeError:
            pass
        plan.build_fail_rank = -1
        # more ranks than templates: the surplus ranks build and search an empty range and the merge is still complete
        _FakePlan.info.ntemplates = world - 1
        lo0, cnt0 = shard.build_bank_shard(plan)
        ok_merge = ok_merge and (cnt0 == (1 if rank < world - 1 else 0))
        merged3 = shard.search_candidates_sharded(plan, X, 40.0, max_cands=4096)
        ti_all = full["iw"].astype(np.int64) * nz + full["iz"]
        want3 = np.sort(full[(ti_all < world - 1) & (full["power"] > 40.0)], order=["iw", "iz", "j"])
        ok_merge = ok_merge and np.array_equal(merged3, want3)
        _FakePlan.info.ntemplates = nz * nw
        # harmonic stage by r-range: every rank reports the top of its block, the fold is the global top with the tie rule
        class _HarmPlan:
            info = _Info()
            fail_rank = -1

            def harmonic_sum(self, d_spec, harms, thresholds, scratch_bytes=None, r_lo=0, r_cnt=None):
                if rank == self.fail_rank:
                    raise ValueError("stand-in harmonic failure")
                out = np.zeros(len(harms), dtype=shard.CAND_FIELDS)
                for s_i, h in enumerate(harms):
                    # stand-in volume: power(j) of stage h peaks at j = 1000 h (value 90) and at j = 5000 (value 90 too: a tie
                    # that must go to the smaller j), plus a 50 everywhere; stage 8 has nothing above its threshold
                    peaks = [(1000 * h, 90.0), (5000, 90.0), (2 * r_lo, 50.0)] if h != 8 else []
                    inside = [(j, p) for j, p in peaks if 2 * r_lo <= j < 2 * (r_lo + r_cnt) and p > thresholds[s_i]]
                    if inside:
                        j, pw = min(inside, key=lambda t: (-t[1], t[0]))
                        out[s_i] = (j, 3, 1, pw, 0)
                    else:
                        out[s_i] = (-1, 0, 0, 0.0, 0)
                return out

        _HarmPlan.info.nbins = 6000
        hp = _HarmPlan()
        tops = shard.harmonic_sum_sharded(hp, X, (1, 2, 4, 8), (25.0, 25.0, 25.0, 25.0))
        ok_merge = ok_merge and [int(t["j"]) for t in tops] == [1000, 2000, 4000, -1] and float(tops[0]["power"]) == 90.0
        hp.fail_rank = world - 1
        try:
            shard.harmonic_sum_sharded(hp, X, (1, 2), (25.0, 25.0))
            ok_merge = False
        except RuntimeError:
            pass
        tmax = shard.max_over_ranks(10.0 + rank)
        q.put((rank, ok_merge, ok_bcast, tmax, shard.trial_indices(7, world, rank)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,nz,nw", [(2, 201, 61), (3, 21, 2)])
def test_template_sharding_gloo(world, nz, nw):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, nz, nw, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    trials = []
    for rank, ok_merge, ok_bcast, tmax, tr in res:
        assert ok_merge and ok_bcast
        assert tmax == 10.0 + world - 1
        trials += tr
    assert sorted(trials) == list(range(7))


@pytest.mark.parametrize("nz,nw,world", [(201, 61, 1), (201, 61, 2), (201, 61, 8), (21, 7, 8), (21, 2, 3), (5, 1, 4), (3, 2, 16)])
def test_template_boxes_partition_the_grid(nz, nw, world):
    seen = np.zeros((nw, nz), dtype=np.int32)
    for r in range(world):
        iz_lo, iz_cnt, iw_lo, iw_cnt = shard.template_box(nz, nw, world, r)
        assert 0 <= iz_lo and iz_lo + iz_cnt <= nz and 0 <= iw_lo and iw_lo + iw_cnt <= nw
        seen[iw_lo:iw_lo + iw_cnt, iz_lo:iz_lo + iz_cnt] += 1
    assert (seen == 1).all()


def test_block_range_balanced():
    for n in (0, 1, 7, 61, 201):
        for w in (1, 2, 3, 8):
            parts = [shard.block_range(n, w, r) for r in range(w)]
            assert sum(c for _, c in parts) == n
            assert max(c for _, c in parts) - min(c for _, c in parts) <= 1
            assert all(parts[i][0] + parts[i][1] == parts[i + 1][0] for i in range(w - 1))


def test_fold_stage_records_tie_rule():
    rec = np.zeros((3, 2), dtype=shard.CAND_FIELDS)
    rec[0] = [(-1, 0, 0, 0.0, 0), (10, 5, 2, 40.0, 0)]
    rec[1] = [(7, 1, 1, 30.0, 0), (4, 5, 1, 40.0, 0)]            # stage 1: same power, smaller iw wins
    rec[2] = [(9, 0, 0, 30.0, 0), (-1, 0, 0, 0.0, 0)]            # stage 0: same power, smaller (iw, iz) wins
    out = shard.fold_stage_records(rec)
    assert (int(out[0]["j"]), int(out[0]["iz"]), int(out[0]["iw"])) == (9, 0, 0)
    assert (int(out[1]["j"]), int(out[1]["iz"]), int(out[1]["iw"])) == (4, 5, 1)
    none = np.zeros((2, 1), dtype=shard.CAND_FIELDS)
    none["j"] = -1
    assert int(shard.fold_stage_records(none)[0]["j"]) == -1
