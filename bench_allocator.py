#!/usr/bin/env python
"""bench_allocator.py — what the segment-based allocator buys the transfer path.

    python bench_allocator.py [--requests 24] [--out gpurun_out/allocator.json]

A seeded alloc/free churn (lognormal request sizes, 50 % release probability) is run twice on a 16,384-block
Llama-3-8B-shaped src pool: with the library's segment allocator (best fit / largest first / merge on free)
and with a LIFO free list (the usual paged-attention allocator).  After the warm-up churn the next `--requests`
allocations become one transfer batch (dst: the same allocator policy on a fresh pool).  Reported per policy:
mean src run length, aligned segments, the one-kernel transfer time, and the paper's scheme with
cudaMemcpyAsync per (segment, layer, K|V)."""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


class Lifo:
    def __init__(self, n):
        self.free = list(range(n - 1, -1, -1))

    def allocate(self, n):
        return np.asarray([self.free.pop() for _ in range(n)], np.int32), 0

    def release(self, ids):
        self.free.extend(int(i) for i in ids)

    def free_blocks(self):
        return len(self.free)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--requests", type=int, default=24)
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "allocator.json"))
    ap.add_argument("--cfg3-requests", type=int, default=16, help="requests of configs[2]'s trace moved on the GPU")
    args = ap.parse_args()
    import torch
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F, pools as P, synth

    shape, NB = synth.LLAMA3_8B, 16384
    src_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, NB).bytes(shape))
    dst_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, NB).bytes(shape))
    src = F.make_pool(src_buf.data_ptr(), 32, 8, 128, 2, NB, 16, "lkbthd")
    dst = F.make_pool(dst_buf.data_ptr(), 32, 8, 128, 2, NB, 16, "lkbthd")
    s = torch.cuda.current_stream().cuda_stream
    ev = lambda: torch.cuda.Event(enable_timing=True)
    out = {}
    for policy in ("segment_allocator", "lifo_free_list"):
        rng = np.random.default_rng(synth.SEED_BASE + 6000)
        class Seg:
            def __init__(self, n): self.a = F.Allocator(n)
            def allocate(self, n): return self.a.allocate(n)
            def release(self, ids): self.a.free(ids)
            def free_blocks(self): return self.a.stats()["free_blocks"]
        mk = (lambda n: Seg(n)) if policy == "segment_allocator" else (lambda n: Lifo(n))
        A, D = mk(NB), mk(NB)
        held = []
        for step in range(4000):                                    # warm-up churn to a fragmented steady state
            if held and (rng.random() < 0.5 or A.free_blocks() < 2500):
                A.release(held.pop(int(rng.integers(len(held)))))
            else:
                held.append(A.allocate(int(np.clip(rng.lognormal(np.log(128), 0.6), 16, 1024)))[0])
        reqs, blocks, runs = [], 0, 0
        for r in range(args.requests):
            n = int(np.clip(rng.lognormal(np.log(256), 0.5), 64, 1024))
            while A.free_blocks() < n:
                A.release(held.pop(int(rng.integers(len(held)))))
            ids = A.allocate(n)[0]
            dids = D.allocate(n)[0]
            reqs.append(F.Request(n * 16, ids, dids))
            blocks += n
            runs += synth.n_runs(ids)
            if held and rng.random() < 0.5:                         # churn continues between requests
                A.release(held.pop(int(rng.integers(len(held)))))
        plan = F.flowkv_plan(src, dst, reqs, F.FLOWKV_CHECK_DST_ALIAS, None, s)
        st = plan.stats
        for _ in range(3):
            plan.transfer(s)
        ts = []
        for _ in range(10):
            a, b = ev(), ev()
            a.record(); plan.transfer(s); b.record(); torch.cuda.synchronize(); ts.append(a.elapsed_time(b))
        F.flowkv_baseline_segmentwise(plan, s); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); calls = F.flowkv_baseline_segmentwise(plan, s); b.record(); torch.cuda.synchronize()
        out[policy] = {"requests": args.requests, "blocks": blocks, "mean_src_run_blocks": blocks / runs,
                       "aligned_segments": st["n_segments"], "payload_bytes": st["payload_bytes"],
                       "kernel_ms": float(np.median(ts)), "hbm_GBps": 2 * st["payload_bytes"] / np.median(ts) / 1e6,
                       "launches": 1, "segmentwise_memcpy_calls": calls, "segmentwise_memcpy_ms": a.elapsed_time(b)}
        print(policy, json.dumps(out[policy]), flush=True)
        plan.destroy()
    del src_buf, dst_buf
    torch.cuda.empty_cache()

    # ---- BASELINE.json configs[2]'s own alloc/free trace, driven by the allocator ----------------
    # The same seeded trace (earlier tenants fill the pool, a seeded subset finishes, the 64 requests are allocated)
    # with the block ids chosen (i) by the plain FIFO free list of synth.config3_batched (the config as bench.py runs
    # it) and (ii) by flowkv_alloc_* on both pools.  All 64 requests are planned on the host (segments per request);
    # the first `--cfg3-requests` of each are moved on the GPU.
    out["cfg3_trace"] = {}
    for policy, alloc in (("fifo_free_list", None), ("segment_allocator", F.Allocator)):
        w = synth.config3_batched(allocator=alloc)
        n_src = sum(synth.n_runs(r.src_blocks) for r in w.requests)
        n_dst = sum(synth.n_runs(r.dst_blocks) for r in w.requests)
        blocks = sum(len(r.src_blocks) for r in w.requests)
        fake = 0x7F0000000000
        hp = F.flowkv_plan_host(P.describe(w.src, w.shape, fake), P.describe(w.dst, w.shape, fake), P.requests_of(w))
        segs = hp.stats["n_segments"]
        hp.destroy()
        w16 = synth.config3_batched(n_requests=args.cfg3_requests, allocator=alloc)
        dp = P.DevicePools(w16, sentinel_dst=False)
        plan = dp.plan(F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, None, s)
        for _ in range(3):
            plan.transfer(s)
        ts = []
        for _ in range(10):
            a, b = ev(), ev()
            a.record(); plan.transfer(s); b.record(); torch.cuda.synchronize(); ts.append(a.elapsed_time(b))
        F.flowkv_baseline_segmentwise(plan, s); torch.cuda.synchronize()
        a, b = ev(), ev()
        a.record(); calls = F.flowkv_baseline_segmentwise(plan, s); b.record(); torch.cuda.synchronize()
        st16 = plan.stats
        out["cfg3_trace"][policy] = {
            "requests": len(w.requests), "blocks": blocks, "mean_src_run_blocks": blocks / n_src,
            "mean_dst_run_blocks": blocks / n_dst, "aligned_segments": segs, "segments_per_request": segs / len(w.requests),
            "gpu_requests": len(w16.requests), "gpu_segments": st16["n_segments"], "gpu_payload_bytes": st16["payload_bytes"],
            "kernel_ms": float(np.median(ts)), "hbm_GBps": 2 * st16["payload_bytes"] / np.median(ts) / 1e6,
            "segmentwise_memcpy_calls": calls, "segmentwise_memcpy_ms": a.elapsed_time(b)}
        print("cfg3_trace", policy, json.dumps(out["cfg3_trace"][policy]), flush=True)
        plan.destroy()
        del dp
        torch.cuda.empty_cache()
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump(out, open(args.out, "w"), indent=1)


if __name__ == "__main__":
    main()
