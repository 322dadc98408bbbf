"""Host-side planners behind the C ABI (no GPU): the slice cache of the out-of-core / RI-direct runs
 and the triplet sharding (NEXT-3)."""
import numpy as np
import pytest

import paper_1609_08094_b200 as tb

STREAMED, RI = 1, 2


@pytest.mark.parametrize("o,v,prec,mode,nslots,win", [
    (8, 40, tb.FP64, STREAMED, 0, 0), (8, 40, tb.MIXED, RI, 0, 1), (16, 120, tb.FP64, STREAMED, 12, 2),
    (24, 240, tb.FP64, RI, 0, 0), (24, 240, tb.MIXED, STREAMED, 0, 1), (24, 240, tb.FP64, STREAMED, 9, 1),
    (40, 480, tb.FP64, STREAMED, 0, 0), (5, 9, tb.FP64, RI, 2, 3), (81, 323, tb.FP64, STREAMED, 30, 0),
])
def test_slice_cache_plan_is_consistent(o, v, prec, mode, nslots, win):
    """Replay the load list: every job finds X_r and XT_q in the slots its table names; a streamed load never
    overwrites a slice the running or the previous batch uses (the copy runs while the previous batch computes)."""
    loads, jobs, info = tb.triples_plan_slices(o, v, prec, mode, nslots, win)
    used, nb = info["nslots"], info["batches"]
    assert 1 <= info["win"] <= 4 and (win <= 0 or info["win"] <= win)
    assert min(o, (6 if mode == STREAMED else 3) * info["win"]) <= used <= o
    need = [set() for _ in range(nb)]
    for (b, q, r, xq, xr) in jobs:
        need[b].update((int(q), int(r)))
    slot_has = {}
    li = ji = 0
    for b in range(nb):
        while li < len(loads) and loads[li][0] == b:
            _, r, s = (int(x) for x in loads[li])
            assert 0 <= s < used and r not in slot_has.values()
            old = slot_has.get(s)
            if old is not None:
                assert old not in need[b]
                if mode == STREAMED and b > 0:
                    assert old not in need[b - 1], "prefetch would overwrite a slice the previous batch reads"
            slot_has[s] = r
            li += 1
        while ji < len(jobs) and jobs[ji][0] == b:
            _, q, r, xq, xr = (int(x) for x in jobs[ji])
            assert slot_has.get(xr) == r and slot_has.get(xq) == q
            ji += 1
    assert li == len(loads) and ji == len(jobs)


def test_slice_cache_with_all_slots_loads_every_slice_once():
    o, v = 24, 240
    loads, _, info = tb.triples_plan_slices(o, v, tb.FP64, STREAMED, o, 0)
    assert info["nslots"] == o and len(loads) == o and sorted(int(x[1]) for x in loads) == list(range(o))
    few, _, small = tb.triples_plan_slices(o, v, tb.FP64, STREAMED, 0, 1)
    assert small["nslots"] == 6 and small["win"] == 1 and len(few) > o          # a small cache re-loads slices
    more, _, _ = tb.triples_plan_slices(o, v, tb.FP64, STREAMED, 12, 1)
    assert o <= len(more) < len(few)                                            # more slots, fewer re-loads


def test_streamed_workspace_fits_a_small_budget():
    for (o, v) in [(24, 240), (40, 480), (81, 323)]:
        full = tb.triples_workspace_bytes(o, v, tb.FP64)
        vvvo = 8 * v ** 3 * o
        w1 = tb.triples_workspace_bytes_streamed(o, v, tb.FP64, 0, 1)
        assert 0 < w1 < min(full, vvvo), "window 1 with 6 cache slots needs less than the vvvo tensor itself"
        assert tb.triples_cache_slots(o, v, 0, tb.FP64, STREAMED, w1) == (6, 1)
        assert tb.triples_cache_slots(o, v, 0, tb.FP64, STREAMED, w1 - 4096) == (0, 0)
        w1b = tb.triples_workspace_bytes_streamed(o, v, tb.FP64, 9, 1)
        n, win = tb.triples_cache_slots(o, v, 0, tb.FP64, STREAMED, w1b)
        assert win == 1 and n == 9
        n, win = tb.triples_cache_slots(o, v, 0, tb.FP64, STREAMED, full)
        assert win >= 2 and n >= 6 * win or n == o
    # the paper's largest system (119, 475): resident repacks exceed 180 GB, the streamed cache fits
    assert tb.triples_workspace_bytes(119, 475, tb.FP64) > 180e9
    assert tb.triples_workspace_bytes_streamed(119, 475, tb.FP64, 0, 0) < 90e9       # 25.6 GB of it the t2 repack
    assert tb.triples_workspace_bytes_ri(119, 475, 1425, tb.FP64, 0, 0) < 100e9


@pytest.mark.parametrize("o,v,nshards", [(8, 40, 2), (16, 120, 3), (24, 240, 8), (40, 480, 8), (3, 5, 4)])
def test_shards_partition_the_restricted_loop(o, v, nshards):
    nb, sot, jps = tb.triples_plan_shards(o, v, tb.FP64, nshards)
    trip = tb.triples_triplet_list(o)
    for n, (i, j, k) in enumerate(trip):
        assert (sot[n] == -1) == (i == j == k)            # every non-diagonal triplet in exactly one shard
        assert -1 <= sot[n] < nshards
    _, bot, jobs = tb.triples_plan_batches(o, v, tb.FP64)
    assert jps.sum() == len(jobs)
    # contiguous ranges of the launch order, whole batches
    shard_of_batch = {}
    for n in range(len(trip)):
        if bot[n] >= 0:
            assert shard_of_batch.setdefault(int(bot[n]), int(sot[n])) == int(sot[n])
    seq = [shard_of_batch[b] for b in sorted(shard_of_batch)]
    assert seq == sorted(seq)
    if nb >= 4 * nshards:                                 # balanced by job count (equal task weight, L198)
        assert jps.max() <= 1.5 * jps.mean() + 200


@pytest.mark.parametrize("prec", [tb.FP64, tb.MIXED, tb.EMU64], ids=["fp64", "mixed", "emu64"])
@pytest.mark.parametrize("o,v,mode,naux", [(32, 400, STREAMED, 0), (24, 240, RI, 720), (16, 120, STREAMED, 0), (9, 40, RI, 50)])
def test_cache_slots_uses_the_whole_budget(o, v, mode, naux, prec):
    """triples_cache_slots(bytes) is the LARGEST cache that fits: n slots fit, n + 1 do not (or n == nocc).  The slot
    size is counted in operand words (4 bytes on both packed paths); counting the emulated-FP64 path's 8-byte U
    elements instead left about half of the extra slots unused."""
    wsb = (lambda n, w: tb.triples_workspace_bytes_streamed(o, v, prec, n, w)) if mode == STREAMED else \
          (lambda n, w: tb.triples_workspace_bytes_ri(o, v, naux, prec, n, w))
    lo, hi = wsb(0, 0), wsb(o, 0)
    for frac in (0.0, 0.23, 0.5, 0.77, 1.0):
        budget = int(lo + frac * (hi - lo))
        n, win = tb.triples_cache_slots(o, v, naux, prec, mode, budget)
        assert n >= 1 and win >= 1
        assert wsb(n, win) <= budget
        assert n == o or wsb(n + 1, win) > budget, (n, win, budget)
