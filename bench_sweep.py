#!/usr/bin/env python
"""bench_sweep.py — BASELINE.json configs[4]: Llama-3-8B shape, request length 128..131,072 tokens x src run
length {1, 2, 8, 64, contiguous}, plus the device -> pinned-host pack path at 32,768 tokens.

    python bench_sweep.py [--out gpurun_out/sweep.json] [--reps 20] [--quick] [--tokens 1024,4096] [--runs 1,0]
    python bench_sweep.py --table3          # the paper's own request sizes (Table 3: 500 .. 12,000 tokens)

Per point: payload, kernel time (CUDA events, mean and min over reps, L2 flushed between reps when
the payload could stay L2-resident), GB/s, the SAME-SIZE PLAIN COPY under the same conditions (one contiguous
cudaMemcpyAsync D2D of payload bytes: the honest ceiling at L2-scale sizes) and kernel time as a fraction of it,
the CUDA-graph replay time of flowkv_transfer, request latency (host call of flowkv_plan -> stream drained),
kernel launches, segments, and the cudaMemcpyAsync baselines (per block/layer/K|V and per segment/layer/K|V).

L2 flush = a READ pass over a 512 MiB buffer (leaves clean lines; a write pass would leave ~100 MB of dirty lines
whose write-back the timed kernel then pays for).
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


def main(argv=None, emit=None) -> list:
    """Runs the sweep and returns its rows.  ``emit(row)`` is called per finished row (default: print the row as a
    JSON line on stdout); bench.py passes its own so that its stdout stays ONE JSON line."""
    if emit is None:
        emit = lambda row: print(json.dumps(row), flush=True)
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "sweep.json"))
    ap.add_argument("--reps", type=int, default=20)
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--tuning", default=None)
    ap.add_argument("--no-baselines", action="store_true")
    ap.add_argument("--no-pinned-pack", action="store_true", help="skip the device -> pinned host leg at 32,768 tokens")
    ap.add_argument("--tokens", default=None, help="comma-separated request lengths (default: the whole sweep)")
    ap.add_argument("--runs", default=None, help="comma-separated src run lengths, 0 = contiguous")
    ap.add_argument("--table3", action="store_true",
                    help="the paper's Table 3 request sizes (500 .. 12,000 tokens, src runs ~ Geometric(mean 4)); adds the "
                         "latency of the host route (flowkv_plan + flowkv_transfer_via_host: pool -> pinned host -> pool)")
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
    if args.table3:
        tokens, runs = list(synth.TABLE3_TOKENS), [4]            # one point per length: Geometric(mean 4) runs, as configs[1]
    if args.tokens:
        tokens = [int(x) for x in args.tokens.split(",")]
    if args.runs and not args.table3:
        runs = [int(x) for x in args.runs.split(",")]
    max_nb = (max(tokens) + 15) // 16
    src_spec_max = synth.PoolSpec("lkbthd", 16, max(16384, 2 * max_nb))
    src_buf = P.alloc_bytes(src_spec_max.bytes(shape))
    dst_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, max_nb).bytes(shape))
    P.fill_values(src_buf, "normal", "bf16", synth.SEED_BASE + 5000)
    flush = torch.zeros(512 << 20, dtype=torch.uint8, device="cuda").view(torch.int64)       # > L2 (126 MB)
    flush_out = torch.zeros(1, dtype=torch.int64, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    rows = []

    def timed(fn, reps, do_flush):
        ts = []
        for _ in range(reps):
            if do_flush:
                flush.sum()               # read pass: evicts everything, leaves clean lines
            a, b = ev(), ev()
            a.record(stream); fn(); b.record(stream)
            torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        # CUDA event timestamps tick every ~1 us; the MEAN over reps dithers below one tick (min is kept beside it)
        return float(np.mean(ts)), float(np.min(ts))

    seen = set()
    via_host = None
    for T in tokens:
        for run in runs:
            w = synth.table3_point(T) if args.table3 else synth.config5_point(T, run)
            r = w.requests[0]
            key = (T, synth.n_runs(r.src_blocks))
            if key in seen:                                   # run >= request size duplicates "contiguous"
                continue
            seen.add(key)
            src = P.describe(w.src, shape, src_buf.data_ptr())
            dst = P.describe(w.dst, shape, dst_buf.data_ptr())
            reqs = F.RequestBatch([F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)])    # marshalled once, as a C caller would hold it
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
                    flush.sum()
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                p2 = F.flowkv_plan(src, dst, reqs, F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, tuning, s)
                p2.transfer(s)
                torch.cuda.synchronize()
                lat.append((time.perf_counter() - t0) * 1e3)
                p2.destroy()
            # the same bytes as ONE contiguous cudaMemcpyAsync D2D, timed the same way (same flush, same events)
            flat_s, flat_d = src_buf[:payload], dst_buf[:payload]
            def plain():
                flat_d.copy_(flat_s, non_blocking=True)       # torch issues one cudaMemcpyAsync D2D for this
            plain(); torch.cuda.synchronize()
            pmed, pmn = timed(plain, args.reps, do_flush)
            # CUDA-graph replay of the same flowkv_transfer launch
            gstream = torch.cuda.Stream()
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph, stream=gstream):
                plan.transfer(torch.cuda.current_stream().cuda_stream)
            graph.replay(); torch.cuda.synchronize()
            gmed, gmn = timed(graph.replay, args.reps, do_flush)
            # back to back: 8 launches of the same transfer in a row, per launch (launch ramps can overlap)
            def eight():
                for _ in range(8):
                    plan.transfer(s)
            b2b = timed(eight, max(3, args.reps // 4), do_flush)[0] / 8
            row = {"tokens": T, "run": ("geometric(4)" if args.table3 else run or "contig"), "segments": st["n_segments"], "payload_bytes": payload,
                   "plain_copy_ms_med": pmed, "plain_copy_ms_min": pmn, "frac_of_plain_copy": pmed / med,
                   "graph_replay_ms_med": gmed, "back_to_back_ms_per_launch": b2b,
                   "kernel_ms_med": med, "kernel_ms_min": mn, "payload_GBps": payload / (med * 1e-3) / 1e9,
                   "hbm_GBps": 2 * payload / (med * 1e-3) / 1e9, "hbm_GBps_best": 2 * payload / (mn * 1e-3) / 1e9,
                   "latency_ms_plan_to_done": float(np.median(lat)), "launches_per_request": launches,
                   "l2_flushed": do_flush, "tile_bytes": st["tile_bytes"], "grid": st["grid"], "threads": st["threads"]}
            if args.table3:
                # the host route (the network stand-in): pool -> pinned host -> pool, both PCIe directions inside the
                # timed region; host wall clock from the flowkv_plan call until the stream has drained
                if via_host is None:
                    via_host = torch.empty(max(tokens) * shape.bytes_per_token, dtype=torch.uint8, pin_memory=True)
                pv = F.flowkv_plan(src, dst, reqs, F.FLOWKV_PLAN_NO_TRANSFER, tuning, s)
                sb = F.flowkv_via_host_scratch_bytes(pv, 0)
                pv.destroy()
                scratch = P.alloc_bytes(sb)
                hl = []
                for i in range(min(args.reps, 10) + 1):
                    torch.cuda.synchronize()
                    t0 = time.perf_counter()
                    pv = F.flowkv_plan(src, dst, reqs, F.FLOWKV_PLAN_NO_TRANSFER, tuning, s)
                    F.flowkv_transfer_via_host(pv, via_host.data_ptr(), payload, 0, 0, s, scratch.data_ptr(), sb)
                    torch.cuda.synchronize()
                    if i:                                         # the first call creates the helper streams
                        hl.append((time.perf_counter() - t0) * 1e3)
                    pv.destroy()
                del scratch
                row["via_host_latency_ms_plan_to_done"] = float(np.median(hl))
                row["via_host_GBps_each_way"] = payload / (float(np.median(hl)) * 1e-3) / 1e9
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
            emit(row)

    # ---- device -> pinned host pack at the 32k-token point ------------------------------------------------------
    T = 32768
    if T in tokens and not args.table3 and not args.no_pinned_pack:
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
            emit(row)
        del host

    if args.out:
        os.makedirs(os.path.dirname(args.out), exist_ok=True)
        json.dump(rows, open(args.out, "w"), indent=1)
    return rows


if __name__ == "__main__":
    main()
