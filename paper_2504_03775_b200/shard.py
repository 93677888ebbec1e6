"""Sharding a transfer batch over ranks (one process per GPU) — no data-path collective.

Requests are independent units (a segment never spans two requests, A10), so a batch splits
across GPUs by assigning whole requests; each rank plans and moves its own shard between its own pools.
`torch.distributed` is used only for the barrier and for taking the max time over ranks.
"""
from __future__ import annotations

from typing import List, Sequence


def shard_requests(num_tokens: Sequence[int], world: int) -> List[List[int]]:
    """Longest-processing-time-first assignment of request indices to `world` ranks (deterministic):
    requests sorted by length (ties by index), each given to the rank with the fewest tokens so far."""
    loads = [0] * world
    out: List[List[int]] = [[] for _ in range(world)]
    for i in sorted(range(len(num_tokens)), key=lambda i: (-int(num_tokens[i]), i)):
        r = min(range(world), key=lambda k: (loads[k], k))
        out[r].append(i)
        loads[r] += int(num_tokens[i])
    for lst in out:
        lst.sort()
    return out


def max_over_ranks(value: float, device=None) -> float:
    """MAX all-reduce of one float (the timing rule for every multi-GPU number)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([value], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
