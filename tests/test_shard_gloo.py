"""The N>1 path on CPU: world_size-2 gloo processes shard one batch, plan their shards with the host
planner, and agree with the unsharded plan; the max-over-ranks timing helper reduces correctly."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import shard, synth

FAKE = 0x7F0000000000


def _free_port() -> int:
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _plan_stats(w, idx):
    sp = F.make_pool(FAKE, w.shape.num_layers, 8, 128, 2, w.src.num_blocks, 16, "lkbthd")
    dp = F.make_pool(FAKE, w.shape.num_layers, 8, 128, 2, w.dst.num_blocks, 16, "lkbthd")
    reqs = [F.Request(w.requests[i].num_tokens, w.requests[i].src_blocks, w.requests[i].dst_blocks) for i in idx]
    return F.flowkv_plan_host(sp, dp, reqs, F.FLOWKV_CHECK_DST_ALIAS).stats


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = synth.config3_batched(n_requests=9, num_layers=2)
    parts = shard.shard_requests([r.num_tokens for r in w.requests], world)
    st = _plan_stats(w, parts[rank])
    mine = torch.tensor([st["total_tokens"], st["n_segments"], st["payload_bytes"], len(parts[rank])], dtype=torch.int64)
    gathered = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(gathered, mine)
    t = shard.max_over_ranks(10.0 + rank)
    dist.barrier()
    if rank == 0:
        q.put((torch.stack(gathered).sum(0).tolist(), t, parts))
    dist.destroy_process_group()


def test_two_ranks_cover_the_batch_without_overlap():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    sums, tmax, parts = q.get()
    w = synth.config3_batched(n_requests=9, num_layers=2)
    full = _plan_stats(w, range(9))
    assert sums == [full["total_tokens"], full["n_segments"], full["payload_bytes"], 9]
    assert sorted(parts[0] + parts[1]) == list(range(9)) and not set(parts[0]) & set(parts[1])
    assert tmax == 11.0                                   # max over ranks, not rank 0's own value
    loads = [sum(w.requests[i].num_tokens for i in p) for p in parts]
    assert max(loads) - min(loads) <= max(r.num_tokens for r in w.requests)   # LPT balance bound


def test_shard_is_deterministic_and_handles_more_ranks_than_requests():
    assert shard.shard_requests([5, 9, 1], 4) == [[1], [0], [2], []]
    assert shard.shard_requests([], 2) == [[], []]
    assert shard.shard_requests([4, 4, 4, 4], 2) == [[0, 2], [1, 3]]
