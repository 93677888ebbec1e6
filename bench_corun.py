#!/usr/bin/env python
"""bench_corun.py — KV transfer next to a GEMM (transfer kernels "compete for SM resources with
processes like GEMM"; S§8f NEXT-4).

    python bench_corun.py [--out gpurun_out/corun.json]

A bf16 8192^3 cuBLAS GEMM loop (the interferer; library code, not part of the product) runs on one stream, the
configs[1] transfer on another.  Each is timed alone and then together (CUDA events on its own stream, both
loops sized to ~80 ms so they overlap fully), for several SM budgets of the transfer kernel
(`flowkv_tuning.max_sms` x `ctas_per_sm`, ldst and bulk/TMA variants)."""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "corun.json"))
    args = ap.parse_args()
    import torch
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F, pools as P, synth

    w = synth.config2_llama8b_13k()
    dp = P.DevicePools(w, sentinel_dst=False)
    N = 8192
    a = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    b = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    c = torch.empty(N, N, device="cuda", dtype=torch.bfloat16)
    sg, sc = torch.cuda.Stream(), torch.cuda.Stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)
    n_gemm, n_copy = 120, 150

    def gemm_loop():
        e0, e1 = ev(), ev()
        with torch.cuda.stream(sg):
            e0.record(sg)
            for _ in range(n_gemm):
                torch.matmul(a, b, out=c)
            e1.record(sg)
        return e0, e1

    def copy_loop(plan):
        e0, e1 = ev(), ev()
        e0.record(sc)
        for _ in range(n_copy):
            plan.transfer(sc.cuda_stream)
        e1.record(sc)
        return e0, e1

    tf = lambda ms: n_gemm * 2 * N ** 3 / (ms * 1e-3) / 1e12
    gb = lambda ms: n_copy * 2 * w.payload_bytes / (ms * 1e-3) / 1e9
    for _ in range(2):
        e0, e1 = gemm_loop(); torch.cuda.synchronize()
    gemm_alone = tf(e0.elapsed_time(e1))
    rows = []
    settings = [("default (grid <= 256 CTAs/SM)", None),
                ("max_sms 64 x 2 CTAs", {"max_sms": 64, "ctas_per_sm": 2}),
                ("max_sms 32 x 2 CTAs", {"max_sms": 32, "ctas_per_sm": 2}),
                ("max_sms 16 x 2 CTAs", {"max_sms": 16, "ctas_per_sm": 2}),
                ("bulk/TMA, default grid", {"variant": "bulk"}),
                ("bulk/TMA, max_sms 148 x 1 CTA x 1 thread, 6 stages", {"variant": "bulk", "ctas_per_sm": 1, "stages": 6, "tile_bytes": 32768}),
                ("bulk/TMA, max_sms 32 x 1 CTA, 6 stages", {"variant": "bulk", "max_sms": 32, "ctas_per_sm": 1, "stages": 6, "tile_bytes": 32768})]
    for name, t in settings:
        plan = F.flowkv_plan(dp.src, dp.dst, dp.requests, 0, t, sc.cuda_stream)
        sc.synchronize()
        c0, c1 = copy_loop(plan); torch.cuda.synchronize()
        c0, c1 = copy_loop(plan); torch.cuda.synchronize()
        copy_alone = gb(c0.elapsed_time(c1))
        torch.cuda.synchronize()
        g0, g1 = gemm_loop()
        c0, c1 = copy_loop(plan)
        torch.cuda.synchronize()
        row = {"setting": name, "tuning": t, "grid": plan.stats["grid"], "copy_alone_GBps": copy_alone,
               "gemm_alone_TFLOPs": gemm_alone, "copy_corun_GBps": gb(c0.elapsed_time(c1)),
               "gemm_corun_TFLOPs": tf(g0.elapsed_time(g1)),
               "copy_loop_ms": c0.elapsed_time(c1), "gemm_loop_ms": g0.elapsed_time(g1)}
        rows.append(row)
        print(json.dumps(row), flush=True)
        plan.destroy()
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump(rows, open(args.out, "w"), indent=1)


if __name__ == "__main__":
    main()
