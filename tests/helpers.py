"""Test-side restatements used to PIN the oracle — independent of oracle/ and of the CUDA path.

Pools are viewed with numpy reshape/transpose only (no stride arithmetic): the logical index
order of every view is [layer, K|V, block, token, head, dim].
"""
from __future__ import annotations

import itertools

import numpy as np


ELEM_DTYPE = {1: np.uint8, 2: np.uint16, 4: np.uint32, 8: np.uint64}


def logical_view(buf_u8: np.ndarray, layout: str, L: int, NB: int, BS: int, H: int, D: int, e: int = 2) -> np.ndarray:
    """Unsigned-integer view (one item per `e`-byte element) of a flat pool buffer, indexed
    [l, c, block, token, head, dim].

    lkbthd = Eq. 5 left side  (L,2,B,H) with H=[token][head][dim]
    blkhtd = Eq. 5 right side (B,L,2,H) with H=[head][token][dim]
    blkthd = Eq. 5 right side (B,L,2,H) with H=[token][head][dim] (H as on the left side)
    """
    w = buf_u8.view(ELEM_DTYPE[e])
    if layout == "lkbthd":
        return w.reshape(L, 2, NB, BS, H, D)
    if layout == "blkhtd":
        return w.reshape(NB, L, 2, H, BS, D).transpose(1, 2, 0, 4, 3, 5)
    if layout == "blkthd":
        return w.reshape(NB, L, 2, BS, H, D).transpose(1, 2, 0, 3, 4, 5)
    raise ValueError(layout)


def token_slots(table, bs: int, T: int) -> np.ndarray:
    """Pool-wide token slot index of each request token: table[t // bs] * bs + t % bs."""
    t = np.arange(T, dtype=np.int64)
    return np.asarray(table, dtype=np.int64)[t // bs] * bs + t % bs


def cuts_by_definition(src_tab, bs_s, dst_tab, bs_d, T):
    """Token positions where a new transfer MUST start: either side's slot index does not step by +1.
    (a transfer is possible exactly over ids that are 'memory-contiguous' on both sides.)"""
    if T == 0:
        return []
    brk = np.zeros(T - 1, dtype=bool)
    if src_tab is not None:
        brk |= np.diff(token_slots(src_tab, bs_s, T)) != 1
    if dst_tab is not None:
        brk |= np.diff(token_slots(dst_tab, bs_d, T)) != 1
    return [0] + [int(i) + 1 for i in np.nonzero(brk)[0]]


def segments_from_cuts(cuts, T):
    ends = list(cuts[1:]) + [T]
    return [(c, e - c) for c, e in zip(cuts, ends)]


def brute_force_min_partition(src_tab, bs_s, dst_tab, bs_d, T):
    """Exhaustive search over all 2^(T-1) ways to cut [0,T) into pieces; a piece is legal iff its token
    slots are consecutive on both sides.  Returns (min #pieces, list of all minimal partitions)."""
    ss = token_slots(src_tab, bs_s, T) if src_tab is not None else np.arange(T)
    ds = token_slots(dst_tab, bs_d, T) if dst_tab is not None else np.arange(T)

    def legal(a, b):
        return np.all(np.diff(ss[a:b]) == 1) and np.all(np.diff(ds[a:b]) == 1)

    best, best_parts = None, []
    for mask in range(1 << (T - 1)):
        cuts = [0] + [i + 1 for i in range(T - 1) if (mask >> i) & 1]
        parts = segments_from_cuts(cuts, T)
        if best is not None and len(parts) > best:
            continue
        if all(legal(a, a + n) for a, n in parts):
            if best is None or len(parts) < best:
                best, best_parts = len(parts), [parts]
            else:
                best_parts.append(parts)
    return best, best_parts


def injective_tables(n_blocks_pool: int, n: int):
    """All injective block tables of length n over a pool of n_blocks_pool blocks."""
    return itertools.permutations(range(n_blocks_pool), n)


def check_segment_invariants(segs, src_tab, bs_s, dst_tab, bs_d, T):
    """Segments tile [0,T) in order, each is +1-contiguous on both sides, neighbours are not mergeable."""
    pos = 0
    ss = token_slots(src_tab, bs_s, T) if src_tab is not None else np.arange(T)
    ds = token_slots(dst_tab, bs_d, T) if dst_tab is not None else np.arange(T)
    for a, n in segs:
        assert a == pos and n > 0
        assert np.all(np.diff(ss[a:a + n]) == 1) and np.all(np.diff(ds[a:a + n]) == 1)
        pos += n
    assert pos == T
    for (a, n), (b, m) in zip(segs, segs[1:]):
        assert not (ss[b] == ss[b - 1] + 1 and ds[b] == ds[b - 1] + 1), "neighbouring segments are mergeable"
