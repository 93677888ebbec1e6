#!/usr/bin/env python
"""bench_sweep.py — BASELINE.json configs[4]: Llama-3-8B shape, request length 128..131,072 tokens x src run
length {1, 2, 8, 64, contiguous}, plus the device -> pinned-host pack path at 32,768 tokens.

    python bench_sweep.py [--out gpurun_out/sweep.json] [--reps 20] [--quick]

Per point: payload, kernel time (CUDA events, median and min over reps, L2 flushed between reps when
the payload could stay L2-resident), GB/s, request latency (host call of flowkv_plan -> stream drained),
kernel launches, segments, and the cudaMemcpyAsync baselines (per block/layer/K|V and per segment/layer/K|V).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)


def main(argv=None) -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "sweep.json"))
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--tuning", default=None)
    ap.add_argument("--no-baselines", action="store_true")
    args = ap.parse_args(argv)

    import torch
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F
    from paper_2504_03775_b200 import pools as P
    from paper_2504_03775_b200 import synth

    torch.cuda.set_device(0)
    stream = torch.cuda.current_stream()
    s = stream.cuda_stream
    shape = synth.LLAMA3_8B
    tuning = json.loads(args.tuning) if args.tuning else None
    tokens = synth.SWEEP_TOKENS if not args.quick else [128, 4096, 32768]
    runs = synth.SWEEP_RUNS if not args.quick else [1, 0]
    max_nb = max(tokens) // 16
    src_spec_max = synth.PoolSpec("lkbthd", 16, max(16384, 2 * max_nb))
    src_buf = P.alloc_bytes(src_spec_max.bytes(shape))
    dst_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, max_nb).bytes(shape))
    P.fill_values(src_buf, "normal", "bf16", synth.SEED_BASE + 5000)
    flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")       # > L2 (126 MB)
    ev = lambda: torch.cuda.Event(enable_timing=True)
    rows = []

    def timed(fn, reps, do_flush):
        ts = []
        for _ in range(reps):
            if do_flush:
                flush.zero_()
            a, b = ev(), ev()
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return float(np.median(ts)), float(np.min(ts))

    seen = set()
    for T in tokens:
        for run in runs:
            w = synth.config5_point(T, run)
            r = w.requests[0]
            key = (T, synth.n_runs(r.src_blocks))
            if key in seen:                                   # run >= request size duplicates "contiguous"
                continue
            seen.add(key)
            src = P.describe(w.src, shape, src_buf.data_ptr())
            dst = P.describe(w.dst, shape, dst_buf.data_ptr())
            reqs = [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)]
            payload = w.payload_bytes
            do_flush = 2 * payload < (256 << 20)
            plan = F.flowkv_plan(src, dst, reqs, F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, tuning, s)
            st = plan.stats
            for _ in range(3):
                plan.transfer(s)
            torch.cuda.synchronize()
            n0 = F.flowkv_launch_count()
            med, mn = timed(lambda: plan.transfer(s), args.reps, do_flush)
            launches = (F.flowkv_launch_count() - n0) / args.reps
            # request latency: host-side wall clock from the plan call until the stream drains
            lat = []
            for _ in range(min(args.reps, 10)):
                if do_flush:
                    flush.zero_()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                p2 = F.flowkv_plan(src, dst, reqs, F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, tuning, s)
                p2.transfer(s)
                torch.cuda.synchronize()
                lat.append((time.perf_counter() - t0) * 1e3)
                p2.destroy()
            row = {"tokens": T, "run": run or "contig", "segments": st["n_segments"], "payload_bytes": payload,
                   "kernel_ms_med": med, "kernel_ms_min": mn, "payload_GBps": payload / (med * 1e-3) / 1e9,
                   "hbm_GBps": 2 * payload / (med * 1e-3) / 1e9, "hbm_GBps_best": 2 * payload / (mn * 1e-3) / 1e9,
                   "latency_ms_plan_to_done": float(np.median(lat)), "launches_per_request": launches,
                   "l2_flushed": do_flush, "tile_bytes": st["tile_bytes"], "grid": st["grid"], "threads": st["threads"]}
            if not args.no_baselines:
                a, b = ev(), ev()
                F.flowkv_baseline_segmentwise(plan, s); torch.cuda.synchronize()
                a.record(stream); calls = F.flowkv_baseline_segmentwise(plan, s); b.record(stream); torch.cuda.synchronize()
                row["segmentwise_memcpy"] = {"calls": calls, "ms": a.elapsed_time(b)}
                if T <= 32768 or run in (1, 0):
                    a, b = ev(), ev()
                    a.record(stream); calls = F.flowkv_baseline_blockwise(src, dst, reqs, s); b.record(stream)
                    torch.cuda.synchronize()
                    row["blockwise_memcpy"] = {"calls": calls, "ms": a.elapsed_time(b)}
            plan.destroy()
            rows.append(row)
            print(json.dumps(row), flush=True)

    # ---- device -> pinned host pack at the 32k-token point ------------------------------------------------------
    T = 32768
    if T in tokens:
        nbytes = T * shape.bytes_per_token
        host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
        dev_flat = dst_buf[:nbytes]
        a, b = ev(), ev()
        for _ in range(2):
            a.record(stream); host.copy_(dev_flat, non_blocking=True); b.record(stream); torch.cuda.synchronize()
        link_d2h = nbytes / (a.elapsed_time(b) * 1e-3) / 1e9
        for _ in range(2):
            a.record(stream); dev_flat.copy_(host, non_blocking=True); b.record(stream); torch.cuda.synchronize()
        link_h2d = nbytes / (a.elapsed_time(b) * 1e-3) / 1e9
        for run in runs:
            w = synth.config5_point(T, run)
            r = w.requests[0]
            src = P.describe(w.src, shape, src_buf.data_ptr())
            dst = P.describe(w.dst, shape, dst_buf.data_ptr())
            plan = F.flowkv_plan(src, dst, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)], 0, tuning, s)
            plan.pack(host.data_ptr(), nbytes, s); torch.cuda.synchronize()
            med, mn = timed(lambda: plan.pack(host.data_ptr(), nbytes, s), 3, False)
            umed, umn = timed(lambda: plan.unpack(host.data_ptr(), nbytes, s), 3, False)
            row = {"tokens": T, "run": run or "contig", "op": "pack_to_pinned_host", "payload_bytes": nbytes,
                   "pack_ms_med": med, "pack_GBps": nbytes / (med * 1e-3) / 1e9,
                   "unpack_ms_med": umed, "unpack_GBps": nbytes / (umed * 1e-3) / 1e9,
                   "link_memcpy_d2h_GBps": link_d2h, "link_memcpy_h2d_GBps": link_h2d, "launches": 1}
            plan.destroy()
            rows.append(row)
            print(json.dumps(row), flush=True)
        del host

    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump(rows, open(args.out, "w"), indent=1)


if __name__ == "__main__":
    main()
