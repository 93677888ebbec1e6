"""Segment-based allocator: oracle pins, then product (C++) vs oracle on random alloc/free traces (CPU)."""
import itertools

import numpy as np
import pytest

from oracle.allocator_oracle import OracleAllocator
from paper_2504_03775_b200 import flowkv as F


def _runs(ids):
    ids = list(ids)
    return 0 if not ids else 1 + sum(1 for a, b in zip(ids, ids[1:]) if b != a + 1)


def _free_map_segments(num_blocks, allocated):
    """Maximal-run decomposition of the free set, recomputed from a boolean map (independent of the oracle)."""
    free = np.ones(num_blocks, bool)
    free[list(allocated)] = False
    segs, i = [], 0
    while i < num_blocks:
        if free[i]:
            j = i
            while j < num_blocks and free[j]:
                j += 1
            segs.append((i, j - i))
            i = j
        else:
            i += 1
    return segs


def _min_segments_brute_force(free_segs, n):
    """Fewest free segments whose total length reaches n (any subset; the last one may be used partially)."""
    lens = [l for _, l in free_segs]
    for k in range(1, len(lens) + 1):
        if any(sum(c) >= n for c in itertools.combinations(lens, k)):
            return k
    return None


# ---- oracle pins ------------------------------------------------------------------------------------------
def test_oracle_fresh_pool_and_full_release():
    o = OracleAllocator(32)
    assert o.free == [(0, 32)]
    a, sa = o.allocate(10)
    b, sb = o.allocate(22)
    assert (a, sa, b, sb) == (list(range(10)), 1, list(range(10, 32)), 1)      # contiguous => 1 segment each
    with pytest.raises(MemoryError):
        o.allocate(1)
    o.release(b)
    o.release(a)
    assert o.free == [(0, 32)]                                                 # adjacent segments merged


def test_oracle_best_fit_and_fewest_segments_against_brute_force():
    """Catches: first-fit instead of best-fit, smallest-first instead of largest-first when splitting."""
    rng = np.random.default_rng(3)
    for trial in range(300):
        NB = int(rng.integers(8, 20))
        o = OracleAllocator(NB)
        held = []
        for step in range(30):
            if held and rng.random() < 0.45:
                o.release(held.pop(int(rng.integers(len(held)))))
            else:
                n = int(rng.integers(1, 6))
                before = list(o.free)
                if n > o.free_blocks():
                    with pytest.raises(MemoryError):
                        o.allocate(n)
                    assert o.free == before                                     # failure changes nothing
                    continue
                ids, segs = o.allocate(n)
                assert len(ids) == n and segs == _runs(ids) <= len(before)
                assert segs == _min_segments_brute_force(before, n)             # "one or a few segments"
                if segs == 1:                                                   # "minimize waste": best fit
                    host = [(s, l) for s, l in before if s <= ids[0] < s + l][0]
                    assert host[1] - n == min(l - n for _, l in before if l >= n)
                    assert ids[0] == host[0]                                    # taken from the segment's start
                held.append(ids)
            allocated = set(itertools.chain.from_iterable(held))
            assert len(allocated) == sum(len(h) for h in held)                  # no id handed out twice
            assert o.free == _free_map_segments(NB, allocated)                  # maximal runs, merged, conserved


def test_oracle_rejects_double_free():
    o = OracleAllocator(8)
    ids, _ = o.allocate(3)
    o.release(ids)
    with pytest.raises(ValueError):
        o.release(ids)


# ---- product vs oracle ------------------------------------------------------------------------------------
def test_product_equals_oracle_on_random_traces():
    rng = np.random.default_rng(11)
    for trial in range(60):
        NB = int(rng.integers(16, 400))
        o, p = OracleAllocator(NB), F.Allocator(NB)
        held = []
        for step in range(200):
            if held and rng.random() < 0.5:
                ids = held.pop(int(rng.integers(len(held))))
                if rng.random() < 0.3:
                    ids = list(rng.permutation(ids))                            # any order may be released
                o.release(ids)
                p.free(ids)
            else:
                n = int(rng.integers(0, max(2, NB // 5)))
                if n > o.free_blocks():
                    with pytest.raises(F.FlowKVError) as ei:
                        p.allocate(n)
                    assert ei.value.status == F.FLOWKV_ERR_NOMEM
                    continue
                eids, esegs = o.allocate(n)
                gids, gsegs = p.allocate(n)
                assert list(gids) == eids and gsegs == esegs
                if n:
                    held.append(eids)
            st = p.stats()
            assert st["free_blocks"] == o.free_blocks() and st["free_segments"] == len(o.free)
            assert st["largest_segment"] == max([l for _, l in o.free], default=0)


def test_product_error_paths_change_nothing():
    p = F.Allocator(10)
    ids, _ = p.allocate(4)
    before = p.stats()
    for bad, status in (([0, 1, 1], F.FLOWKV_ERR_INVALID_ARG), ([0, 99], F.FLOWKV_ERR_BLOCK_OOB),
                        ([0, 7], F.FLOWKV_ERR_INVALID_ARG), ([-1], F.FLOWKV_ERR_BLOCK_OOB)):
        with pytest.raises(F.FlowKVError) as ei:
            p.free(bad)
        assert ei.value.status == status
        assert p.stats() == before
    p.free(ids)
    assert p.stats() == {"free_blocks": 10, "free_segments": 1, "largest_segment": 10}
    with pytest.raises(F.FlowKVError):
        p.free(ids)                                                             # double free


def test_allocator_keeps_runs_long_under_churn_vs_free_list():
    """What the allocator is for: block tables with long runs => few transfer segments.  An alloc/free
    churn like configs[2]'s trace, compared with a LIFO free list (the usual paged-attention allocator)."""
    rng = np.random.default_rng(5)
    NB = 4096
    p = F.Allocator(NB)
    lifo = list(range(NB - 1, -1, -1))
    held_p, held_l, runs_p, runs_l, blocks = [], [], 0, 0, 0
    for step in range(3000):
        if held_p and (rng.random() < 0.5 or p.stats()["free_blocks"] < 600):
            k = int(rng.integers(len(held_p)))
            p.free(held_p.pop(k))
            lifo.extend(held_l.pop(k))
        else:
            n = int(np.clip(rng.lognormal(np.log(128), 0.5), 16, 512))
            ids, _ = p.allocate(n)
            lids = [lifo.pop() for _ in range(n)]
            held_p.append(ids)
            held_l.append(lids)
            if step > 1000:
                runs_p += _runs(ids); runs_l += _runs(lids); blocks += n
    assert blocks / runs_p > 20 * (blocks / runs_l) or blocks / runs_p > 64, (blocks / runs_p, blocks / runs_l)
