"""Oracle of the segment-based block allocator — TEST INFRASTRUCTURE ONLY (never imported by the product).

Paper, §3.3: "FlowKV uses segment management techniques from operating systems ... It tries to
allocate new requests within one or a few contiguous segments.  ... manages free memory blocks with
segment-based minimum heaps.  It chooses the right segments during allocation to minimize waste and
merges adjacent free segments during deallocation."

The paper gives no pseudo-code; reading A19 fixes the policy, restated here step by step with a
plain sorted list and linear scans (no heaps, no index structures, no code shared with csrc/allocator.cpp):

  allocate(n)
    1. if fewer than n blocks are free: fail, change nothing.
    2. among free segments of length >= (blocks still needed), pick the SHORTEST; ties -> lowest start.
       Take its first blocks.  Done.                                  ("minimize waste": best fit)
    3. if no segment is long enough: take the LONGEST segment whole; ties -> lowest start; go to 2.
                                                                      ("one or a few contiguous segments")
  free(ids)
    every id returns to the free set; the free list is re-formed as maximal runs (adjacent segments merge).

Pins (tests/test_allocator.py): the number of segments an allocation uses equals the brute-force minimum
over all subsets of free segments; when one segment suffices its waste equals the brute-force minimum;
conservation (free + allocated = pool, no id handed out twice); the free list is always the maximal-run
decomposition of the free set (recomputed from a boolean map); a fresh pool is one segment; freeing
everything restores one segment.  Unpinned by the paper: the tie-breaks (lowest start) — the paper is
silent; they are this repo's choice.
"""
from __future__ import annotations

from typing import List, Tuple


class OracleAllocator:
    def __init__(self, num_blocks: int):
        self.num_blocks = num_blocks
        self.free: List[Tuple[int, int]] = [(0, num_blocks)]      # (start, length), sorted by start
        self.allocated = set()

    # -- helpers -----------------------------------------------------------------------------------
    def free_blocks(self) -> int:
        return sum(l for _, l in self.free)

    def _rebuild(self, free_ids) -> None:
        ids = sorted(free_ids)
        segs, i = [], 0
        while i < len(ids):
            j = i
            while j + 1 < len(ids) and ids[j + 1] == ids[j] + 1:
                j += 1
            segs.append((ids[i], j - i + 1))
            i = j + 1
        self.free = segs

    def _free_ids(self):
        return [s + k for s, l in self.free for k in range(l)]

    # -- operations --------------------------------------------------------------------------------
    def allocate(self, n: int):
        """-> (ids in allocation order, number of segments used); raises MemoryError if n > free."""
        if n > self.free_blocks():
            raise MemoryError
        out, segs, left = [], 0, n
        while left > 0:
            fitting = [(l, s) for s, l in self.free if l >= left]
            if fitting:
                l, s = min(fitting)                 # shortest, then lowest start
                take = left
            else:
                longest = max(l for _, l in self.free)
                s = min(s for s, l in self.free if l == longest)
                l = longest
                take = l
            out += list(range(s, s + take))
            self.free.remove((s, l))
            if take < l:
                self.free.append((s + take, l - take))
                self.free.sort()
            left -= take
            segs += 1
        self.allocated.update(out)
        return out, segs

    def release(self, ids) -> None:
        ids = list(ids)
        if len(set(ids)) != len(ids) or any(i not in self.allocated for i in ids):
            raise ValueError("not allocated")
        self.allocated.difference_update(ids)
        self._rebuild(self._free_ids() + ids)
