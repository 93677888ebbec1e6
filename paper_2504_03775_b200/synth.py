"""Seeded synthetic inputs: request lengths and block tables for the BASELINE.json configs.

This module serves BOTH the tests' oracle leg and the CUDA path with the *same arrays*.
It holds none of the method's arithmetic: no addressing, no alignment, no copying —
only numpy draws of lengths and block-id lists, and the names/sizes of the pools.
It imports neither ``oracle`` nor the CUDA binding.

The inputs stand in for the paper's LongBench-derived and simulated requests
(§4.1; 13k-token request of Fig. 1; 0.5k-12k inputs of Table 3,
P:L276-289): only request *lengths* and block-id *run structure* matter to a KV move.
Recipes are stated in DESIGN.md §4 and follow SURVEY.md §8(d).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import List, Optional, Sequence, Tuple

import numpy as np

SEED_BASE = 250403775  # + 1000*config + point


ELEM_BYTES = {"fp8": 1, "fp16": 2, "bf16": 2, "fp32": 4}


@dataclass(frozen=True)
class Shape:
    num_layers: int
    num_kv_heads: int
    head_dim: int
    dtype: str  # "fp16" | "bf16" (2-byte elements), "fp8" (1 byte), "fp32" (4 bytes)

    @property
    def elem_bytes(self) -> int:
        return ELEM_BYTES[self.dtype]

    @property
    def bytes_per_token(self) -> int:
        return 2 * self.num_layers * self.num_kv_heads * self.head_dim * self.elem_bytes


TINY = Shape(2, 2, 64, "fp16")
LLAMA3_8B = Shape(32, 8, 128, "bf16")
LLAMA3_70B = Shape(80, 8, 128, "bf16")
LLAMA3_8B_FP8 = Shape(32, 8, 128, "fp8")      # fp8 KV cache: rows of 128 B


@dataclass(frozen=True)
class PoolSpec:
    layout: str        # "lkbthd" | "blkhtd" | "blkthd"
    block_size: int    # tokens per block
    num_blocks: int

    def bytes(self, shape: Shape) -> int:
        return self.num_blocks * self.block_size * shape.bytes_per_token


@dataclass
class Request:
    num_tokens: int
    src_blocks: np.ndarray  # int32
    dst_blocks: np.ndarray  # int32


@dataclass
class Workload:
    name: str
    seed: int
    shape: Shape
    src: PoolSpec
    dst: PoolSpec
    requests: List[Request]
    value_dist: str = "normal"        # "normal" N(0,1) | "uniform" U[-1,1]
    notes: dict = field(default_factory=dict)

    @property
    def total_tokens(self) -> int:
        return int(sum(r.num_tokens for r in self.requests))

    @property
    def payload_bytes(self) -> int:
        return self.total_tokens * self.shape.bytes_per_token


def _nblk(tokens: int, bs: int) -> int:
    return (tokens + bs - 1) // bs


# ----------------------------------------------------------------------------------------
# run-length draws and placement
# ----------------------------------------------------------------------------------------
def runs_geometric(rng: np.random.Generator, n_blocks: int, mean: float) -> List[int]:
    """Run lengths ~ Geometric(p=1/mean) on {1,2,...} until they cover n_blocks (last truncated)."""
    out, tot = [], 0
    while tot < n_blocks:
        r = int(rng.geometric(1.0 / mean))
        r = min(r, n_blocks - tot)
        out.append(r)
        tot += r
    return out


def runs_fixed(n_blocks: int, run: int) -> List[int]:
    out, tot = [], 0
    while tot < n_blocks:
        r = min(run, n_blocks - tot)
        out.append(r)
        tot += r
    return out


def place_runs(rng: np.random.Generator, runs: Sequence[int], num_blocks: int,
               touch_top: bool = True) -> List[np.ndarray]:
    """Give every run a start block so that runs do not overlap and memory-neighbouring runs
    have >= 1 free block between them (so two runs never fuse into a longer one).

    Memory order is a seeded permutation of the draw order; the spare blocks are spread over
    the gaps by one multinomial draw.  With ``touch_top`` the last run in memory ends at block
    ``num_blocks-1`` (so byte offsets reach the top of the pool).  Returns one id array per run,
    in draw order."""
    k = len(runs)
    if k == 0:
        return []
    used = int(sum(runs))
    spare = num_blocks - used - (k - 1)
    if spare < 0:
        raise ValueError(f"pool of {num_blocks} blocks cannot hold {used} blocks in {k} separated runs")
    n_slots = k if touch_top else k + 1      # leading gap + (k-1) inner gaps (+ trailing gap)
    extra = rng.multinomial(spare, np.full(n_slots, 1.0 / n_slots))
    order = rng.permutation(k)               # order[j] = which run sits j-th in memory
    starts = np.zeros(k, dtype=np.int64)
    pos = int(extra[0])
    for j, ri in enumerate(order):
        starts[ri] = pos
        pos += int(runs[ri]) + 1 + (int(extra[j + 1]) if j + 1 < k and j + 1 < n_slots else 0)
    ids = [np.arange(starts[i], starts[i] + runs[i], dtype=np.int32) for i in range(k)]
    top = max(int(a[-1]) for a in ids)
    assert top < num_blocks
    if touch_top:
        assert top == num_blocks - 1
    return ids


def _tables_from_trace(rng, req_blocks: Sequence[int], num_blocks: int, mean: float) -> List[np.ndarray]:
    """Block tables left behind by a seeded alloc/free trace on a FIFO free list (the plain block manager of a
    paged-attention server: allocate = pop ids from the head, free = append ids at the tail; no coalescing):
      1. earlier tenants fill the fresh pool one after another, each taking Geometric(mean) consecutive blocks;
      2. a seeded subset of them finishes, in seeded order — their blocks join the free list hole by hole
         (just enough tenants finish to hold this batch plus 10 %, the rest keep their blocks);
      3. the batch's requests are allocated in order from the head of the free list.
    A request's table is then a chain of the holes earlier tenants left: runs of mean ~`mean` blocks at
    scattered addresses (BASELINE.json configs[2]: "50% fragmentation (runs of mean 2) from a seeded alloc/free
    trace").  Input bookkeeping only — none of FlowKV's own allocator or alignment is involved."""
    used = int(sum(req_blocks))
    tenants, pos = [], 0
    while pos < num_blocks:
        n = min(int(rng.geometric(1.0 / mean)), num_blocks - pos)
        tenants.append((pos, n))
        pos += n
    order = rng.permutation(len(tenants))
    free_list, have, want = [], 0, min(num_blocks, int(np.ceil(1.1 * used)))
    for ti in order:
        if have >= want:
            break
        start, n = tenants[ti]
        free_list.append(np.arange(start, start + n, dtype=np.int32))
        have += n
    if have < used:
        raise ValueError(f"pool of {num_blocks} blocks cannot hold {used} blocks")
    flat = np.concatenate(free_list) if free_list else np.zeros(0, dtype=np.int32)
    out, off = [], 0
    for nb in req_blocks:
        out.append(flat[off:off + nb].copy())
        off += nb
    return out


def alloc_free_trace(rng, req_blocks: Sequence[int], num_blocks: int, mean: float) -> List[tuple]:
    """The event list of the alloc/free trace behind ``_tables_from_trace`` — WITHOUT deciding which blocks an
    allocation gets: ("alloc", key, n) for the earlier tenants that fill the pool (Geometric(mean) blocks each),
    ("free", key) for the seeded subset that finishes (in seeded order, until the batch plus 10 % fits), then
    ("request", r, n) for the batch.  Which ids each allocation receives is the block allocator's business
    (P:L105): feed the events to any allocator with ``tables_from_allocator``."""
    used = int(sum(req_blocks))
    events, sizes, pos = [], [], 0
    while pos < num_blocks:
        n = min(int(rng.geometric(1.0 / mean)), num_blocks - pos)
        events.append(("alloc", len(sizes), n))
        sizes.append(n)
        pos += n
    have, want = 0, min(num_blocks, int(np.ceil(1.1 * used)))
    for ti in rng.permutation(len(sizes)):
        if have >= want:
            break
        events.append(("free", int(ti)))
        have += sizes[int(ti)]
    if have < used:
        raise ValueError(f"pool of {num_blocks} blocks cannot hold {used} blocks")
    events += [("request", r, int(nb)) for r, nb in enumerate(req_blocks)]
    return events


def tables_from_allocator(events: Sequence[tuple], allocator) -> List[np.ndarray]:
    """Replay a trace on ``allocator`` (any object with ``allocate(n) -> (ids, n_segments)`` and ``free(ids)``)
    and return the block table each ("request", r, n) event received.  Bookkeeping only."""
    held, out = {}, {}
    for ev in events:
        if ev[0] == "alloc":
            held[ev[1]] = np.asarray(allocator.allocate(ev[2])[0], np.int32)
        elif ev[0] == "free":
            allocator.free(held.pop(ev[1]))
        else:
            out[ev[1]] = np.asarray(allocator.allocate(ev[2])[0], np.int32)
    return [out[r] for r in sorted(out)]


def _tables_from_runs(rng, req_blocks: Sequence[int], num_blocks: int, kind: Tuple) -> List[np.ndarray]:
    """Per-request block tables with the requested run structure, all sharing one pool."""
    if kind[0] == "contiguous":          # request r's blocks follow request r-1's
        out, off = [], 0
        for nb in req_blocks:
            out.append(np.arange(off, off + nb, dtype=np.int32))
            off += nb
        assert off <= num_blocks
        return out
    if kind[0] == "permutation":         # run length exactly 1: no two neighbours differ by +1
        assert len(req_blocks) == 1
        nb = req_blocks[0]
        while True:
            t = rng.permutation(num_blocks)[:nb].astype(np.int32)
            if nb < 2 or not np.any(np.diff(t) == 1):
                return [t]
    if kind[0] == "trace":
        return _tables_from_trace(rng, req_blocks, num_blocks, kind[1])
    if kind[0] == "allocator":           # the same trace, ids chosen by a caller-supplied block allocator
        return tables_from_allocator(alloc_free_trace(rng, req_blocks, num_blocks, kind[1]), kind[2](num_blocks))
    all_runs, owner = [], []
    for r, nb in enumerate(req_blocks):
        runs = runs_geometric(rng, nb, kind[1]) if kind[0] == "geometric" else runs_fixed(nb, kind[1])
        all_runs += runs
        owner += [r] * len(runs)
    ids = place_runs(rng, all_runs, num_blocks)
    out = []
    for r in range(len(req_blocks)):
        parts = [ids[i] for i in range(len(ids)) if owner[i] == r]
        out.append(np.concatenate(parts) if parts else np.zeros(0, dtype=np.int32))
    return out


def n_runs(table: np.ndarray) -> int:
    """Number of maximal +1 runs in a block table (input statistics only, for reporting)."""
    return 0 if len(table) == 0 else 1 + int(np.count_nonzero(np.diff(table.astype(np.int64)) != 1))


def make_workload(name: str, seed: int, shape: Shape, lengths: Sequence[int],
                  src_layout: str, src_bs: int, src_kind: Tuple, src_blocks: Optional[int],
                  dst_layout: str, dst_bs: int, dst_kind: Tuple, dst_blocks: Optional[int],
                  value_dist: str = "normal", src_slack: float = 1.25, dst_slack: float = 1.0625,
                  notes: Optional[dict] = None) -> Workload:
    """Generic builder.  ``*_kind``: ("contiguous",) | ("permutation",) | ("geometric", mean) |
    ("fixed", run) | ("trace", mean) (seeded alloc/free trace on a FIFO free list) | ("allocator", mean, factory)
    (the same trace with the ids chosen by ``factory(num_blocks)``, an object with allocate(n) / free(ids)).  ``*_blocks`` None => pool sized ``ceil(slack * used)`` (never less than
    what separated runs need)."""
    rng = np.random.default_rng(np.random.PCG64(seed))
    lengths = [int(t) for t in lengths]
    sreq = [_nblk(t, src_bs) for t in lengths]
    dreq = [_nblk(t, dst_bs) for t in lengths]

    def size(nb_req, kind, blocks, slack):
        used = sum(nb_req)
        if blocks is not None:
            return blocks
        if kind[0] == "contiguous":
            return max(used, 1)
        # enough for `used` blocks in separated runs: worst case one gap per run
        if kind[0] in ("trace", "allocator"):
            return max(int(np.ceil(slack * used)), 1)
        worst_runs = used if kind[0] != "fixed" else sum(_nblk(n, kind[1]) for n in nb_req)
        return max(int(np.ceil(slack * used)), used + worst_runs, 1)

    snb = size(sreq, src_kind, src_blocks, src_slack)
    dnb = size(dreq, dst_kind, dst_blocks, dst_slack)
    stabs = _tables_from_runs(rng, sreq, snb, src_kind)
    dtabs = _tables_from_runs(rng, dreq, dnb, dst_kind)
    reqs = [Request(t, s, d) for t, s, d in zip(lengths, stabs, dtabs)]
    return Workload(name, seed, shape, PoolSpec(src_layout, src_bs, snb), PoolSpec(dst_layout, dst_bs, dnb),
                    reqs, value_dist, dict(notes or {}))


# ----------------------------------------------------------------------------------------
# the five BASELINE.json configs
# ----------------------------------------------------------------------------------------
def config1_tiny() -> Workload:
    """BASELINE.json configs[0]: Tiny, 1 x 1000 tokens, src = seeded permutation (run length 1)."""
    return make_workload("cfg1_tiny", SEED_BASE + 1000, TINY, [1000],
                         "lkbthd", 16, ("permutation",), 128,
                         "lkbthd", 16, ("contiguous",), 128, value_dist="uniform")


def config2_llama8b_13k(num_layers: Optional[int] = None) -> Workload:
    """BASELINE.json configs[1]: Llama-3-8B shape, 1 x 13,312 tokens, src runs ~ Geometric(mean 4)
    over a 16,384-block (32 GiB) pool, dst contiguous in a 1,024-block pool.
    ``num_layers`` (tests only) shrinks L; tables are unchanged by it."""
    shape = LLAMA3_8B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    return make_workload("cfg2_llama8b_13k", SEED_BASE + 2000, shape, [13312],
                         "lkbthd", 16, ("geometric", 4.0), 16384,
                         "lkbthd", 16, ("contiguous",), 1024)


def config2_blockmajor(layout: str = "blkthd", num_layers: Optional[int] = None, tokens: int = 13312) -> Workload:
    """configs[1]'s request and block tables with BOTH pools in the paper's (B,L,2,H) order (Eq. 5,
    P:L98-103): a block is one 2 MiB range, a run of blocks one span over all layers."""
    shape = LLAMA3_8B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    w = make_workload(f"cfg2_{layout}_13k", SEED_BASE + 2000, shape, [tokens],
                      layout, 16, ("geometric", 4.0), 16384,
                      layout, 16, ("contiguous",), 1024)
    return w


def config3_lengths(n: int = 64) -> List[int]:
    rng = np.random.default_rng(np.random.PCG64(SEED_BASE + 3000 + 999))
    t = np.exp(rng.normal(np.log(8192.0), 0.5, size=64))
    return [int(x) for x in np.clip(np.rint(t), 1024, 32768).astype(np.int64)[:n]]


def config4_lengths(n: int = 16) -> List[int]:
    rng = np.random.default_rng(np.random.PCG64(SEED_BASE + 4000 + 999))
    return [int(x) for x in rng.integers(4096, 32768, size=16, endpoint=True)[:n]]


def fit_prefix(lengths: Sequence[int], shape: Shape, src_bs: int, dst_bs: int, budget_bytes: int,
               src_blocks_of, dst_blocks_of) -> int:
    """Largest n such that pools for the first n requests fit in ``budget_bytes``."""
    best = 0
    for n in range(1, len(lengths) + 1):
        su = sum(_nblk(t, src_bs) for t in lengths[:n])
        du = sum(_nblk(t, dst_bs) for t in lengths[:n])
        need = (src_blocks_of(n, su) * src_bs + dst_blocks_of(n, du) * dst_bs) * shape.bytes_per_token
        if need <= budget_bytes:
            best = n
        else:
            break
    return best


def _cfg3_src_blocks(n: int, used: int) -> int:
    # keeps the 65,536 / 64 ratio; never less than what runs of mean 2 with gaps need (1.6 x used)
    return max(1024 * n, int(np.ceil(1.6 * used)))


def _cfg3_dst_blocks(n: int, used: int) -> int:
    return int(np.ceil(1.125 * used))


def config3_batched(budget_bytes: Optional[int] = None, n_requests: Optional[int] = None,
                    num_layers: Optional[int] = None, allocator=None) -> Workload:
    """BASELINE.json configs[2]: 64 requests, lognormal lengths (median 8k, clip 1k-32k), src tables from a
    seeded alloc/free trace that leaves runs of mean 2 (break probability 1/2), dst runs of mean 16, one batch.  The literal config needs
    ~201 GiB; ``budget_bytes`` keeps the largest seeded prefix of requests that fits (fit rule)."""
    shape = LLAMA3_8B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    lengths = config3_lengths()
    n = len(lengths) if n_requests is None else n_requests
    if budget_bytes is not None:
        n = min(n, fit_prefix(lengths, shape, 16, 16, budget_bytes, _cfg3_src_blocks, _cfg3_dst_blocks))
    lengths = lengths[:n]
    su = sum(_nblk(t, 16) for t in lengths)
    if allocator is not None:
        # the same seeded alloc/free trace, but a block allocator (``allocator(num_blocks)`` ->
        # object with allocate / free; the library's segment allocator) chooses the ids on BOTH sides
        w = make_workload("cfg3_batched_8b_allocator", SEED_BASE + 3000, shape, lengths,
                          "lkbthd", 16, ("allocator", 2.0, allocator), _cfg3_src_blocks(n, su),
                          "lkbthd", 16, ("allocator", 16.0, allocator), _cfg3_dst_blocks(n, su))
        runs = sum(n_runs(r.src_blocks) for r in w.requests)
        w.notes.update(n_requests=n, of_requests=64, mean_src_run=su / max(runs, 1))
        return w
    for attempt in range(8):   # accept iff the generated mean src run is in [1.9, 2.1]
        w = make_workload("cfg3_batched_8b", SEED_BASE + 3000 + attempt, shape, lengths,
                          "lkbthd", 16, ("trace", 2.0), _cfg3_src_blocks(n, su),
                          "lkbthd", 16, ("geometric", 16.0), _cfg3_dst_blocks(n, su))
        runs = sum(n_runs(r.src_blocks) for r in w.requests)
        mean_run = su / max(runs, 1)
        if 1.9 <= mean_run <= 2.1 or n < 8:
            w.notes.update(n_requests=n, of_requests=64, mean_src_run=mean_run, attempt=attempt)
            return w
    raise RuntimeError("cfg3: mean run length outside [1.9, 2.1]")


def _cfg4_src_blocks(n: int, used: int) -> int:
    return int(np.ceil(1.3 * used))


def _cfg4_dst_blocks(n: int, used: int) -> int:
    return used


def config4_hetero(budget_bytes: Optional[int] = None, n_requests: Optional[int] = None,
                   num_layers: Optional[int] = None) -> Workload:
    """BASELINE.json configs[3]: Llama-3-70B shape, 16 requests of 4k-32k tokens; src block 16 LKBTHD,
    fragmented (runs ~ Geometric mean 4); dst block 64 BLKHTD, contiguous."""
    shape = LLAMA3_70B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    lengths = config4_lengths()
    n = len(lengths) if n_requests is None else n_requests
    if budget_bytes is not None:
        n = min(n, fit_prefix(lengths, shape, 16, 64, budget_bytes, _cfg4_src_blocks, _cfg4_dst_blocks))
    lengths = lengths[:n]
    su = sum(_nblk(t, 16) for t in lengths)
    du = sum(_nblk(t, 64) for t in lengths)
    w = make_workload("cfg4_hetero_70b", SEED_BASE + 4000, shape, lengths,
                      "lkbthd", 16, ("geometric", 4.0), _cfg4_src_blocks(n, su),
                      "blkhtd", 64, ("contiguous",), _cfg4_dst_blocks(n, du))
    w.notes.update(n_requests=n, of_requests=16)
    return w


SWEEP_TOKENS = [2 ** k for k in range(7, 18)]          # 128 .. 131,072
SWEEP_RUNS = [1, 2, 8, 64, 0]                          # 0 = fully contiguous


def config5_point(tokens: int, run: int, num_layers: Optional[int] = None) -> Workload:
    """BASELINE.json configs[4]: one request of ``tokens`` tokens, src runs of FIXED length ``run``
    blocks (0 = contiguous), dst contiguous; pool = max(16,384, 2 x blocks) blocks."""
    shape = LLAMA3_8B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    nb = _nblk(tokens, 16)
    point = SWEEP_TOKENS.index(tokens) * len(SWEEP_RUNS) + SWEEP_RUNS.index(run)
    kind = ("contiguous",) if run == 0 or run >= nb else ("fixed", run)
    return make_workload(f"cfg5_sweep_T{tokens}_run{run or 'contig'}", SEED_BASE + 5000 + point, shape,
                         [tokens], "lkbthd", 16, kind, max(16384, 2 * nb),
                         "lkbthd", 16, ("contiguous",), nb)


# The paper's own request sizes: Table 3 reports KV transfer latency for simulated requests of
# 500 .. 12,000 input tokens on Llama-3.1-8B.  Only the lengths come from the paper; the tables are seeded draws.
TABLE3_TOKENS = [500, 1000, 2000, 4000, 8000, 10000, 12000]


def table3_point(tokens: int, num_layers: Optional[int] = None) -> Workload:
    """One request of a Table 3 input length, src runs ~ Geometric(mean 4) over a 16,384-block pool
    and dst contiguous, exactly as configs[1] is built; lengths that are no multiple of 16 end in a partial block."""
    shape = LLAMA3_8B if num_layers is None else Shape(num_layers, 8, 128, "bf16")
    nb = _nblk(tokens, 16)
    return make_workload(f"table3_T{tokens}", SEED_BASE + 6000 + TABLE3_TOKENS.index(tokens), shape, [tokens],
                         "lkbthd", 16, ("geometric", 4.0), 16384,
                         "lkbthd", 16, ("contiguous",), nb)
