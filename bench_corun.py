#!/usr/bin/env python
"""bench_corun.py — KV transfer next to a GEMM (transfer kernels "compete for SM resources with
processes like GEMM"; S§8f NEXT-4).

    python bench_corun.py [--out gpurun_out/corun.json]

A bf16 8192^3 cuBLAS GEMM loop (the interferer; library code, not part of the product) runs on one stream, the
transfer (configs[1], or with --config cfg4 a rows-mode slice of configs[3]) on another.  Each is timed alone and then
next to the other: both loops run for ~0.3 s, every iteration stamps its completion with a CUDA event on its own
stream, and both rates are read over the same window (the middle of the time both streams were busy) — for several
SM budgets of the transfer kernel (`flowkv_tuning.max_sms` x
`ctas_per_sm`, ldst and bulk/TMA variants; in rows mode the bulk variant is the TMA tensor path, fk_rows_tma)."""
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
    ap.add_argument("--config", default="cfg2", choices=["cfg2", "cfg4"],
                    help="cfg2: configs[1] (span mode); cfg4: a 4-request slice of configs[3] (rows mode: src BS16 LKBTHD -> "
                         "dst BS64 BLKHTD; the bulk variant is the TMA tensor path)")
    ap.add_argument("--gemm-priority", action="store_true",
                    help="put the GEMM on a high-priority stream (the transfer stays at default priority): the block "
                         "scheduler then hands freed SM slots to the GEMM first, and the transfer's many short CTAs fill "
                         "what the GEMM leaves")
    args = ap.parse_args()
    import torch
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F, pools as P, synth

    w = synth.config2_llama8b_13k() if args.config == "cfg2" else synth.config4_hetero(n_requests=4)
    dp = P.DevicePools(w, sentinel_dst=False)
    N = 8192
    a = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    b = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    c = torch.empty(N, N, device="cuda", dtype=torch.bfloat16)
    sg, sc = (torch.cuda.Stream(priority=-1) if args.gemm_priority else torch.cuda.Stream()), torch.cuda.Stream()
    ev = lambda: torch.cuda.Event(enable_timing=True)

    def gemm_loop(n, stamps=None):
        with torch.cuda.stream(sg):
            for _ in range(n):
                torch.matmul(a, b, out=c)
                if stamps is not None:
                    e = ev(); e.record(sg); stamps.append(e)

    def copy_loop(plan, n, stamps=None):
        for _ in range(n):
            plan.transfer(sc.cuda_stream)
            if stamps is not None:
                e = ev(); e.record(sc); stamps.append(e)

    def rate_in_window(t0, stamps, lo, hi):
        """Iterations that completed inside [lo, hi] ms (per-iteration completion stamps) per ms."""
        ts = [t0.elapsed_time(e) for e in stamps]
        inside = [t for t in ts if lo <= t <= hi]
        return (len(inside) - 1) / (inside[-1] - inside[0]) if len(inside) > 2 else float("nan")

    tf = lambda per_ms: per_ms * 2 * N ** 3 / 1e-3 / 1e12
    gb = lambda per_ms: per_ms * 2 * w.payload_bytes / 1e-3 / 1e9
    gemm_loop(10); torch.cuda.synchronize()
    t0 = ev(); st_ = []
    t0.record(sg); gemm_loop(20, st_); torch.cuda.synchronize()
    gemm_ms = t0.elapsed_time(st_[-1]) / 20
    # the GEMM alone over the same ~0.3 s and the same window rule (a 1 kW part settles under its power cap: the
    # burst rate of a short loop is not what a co-run of this length should be compared with)
    t0 = ev(); st_ = []
    t0.record(sg); gemm_loop(max(20, int(300.0 / gemm_ms)), st_); torch.cuda.synchronize()
    end = t0.elapsed_time(st_[-1])
    gemm_alone = tf(rate_in_window(t0, st_, 0.15 * end, 0.95 * end))
    rows = []
    settings = [("ldst, default (grid <= 256 CTAs/SM)", None),
                ("ldst, max_sms 64 x 2 CTAs", {"max_sms": 64, "ctas_per_sm": 2}),
                ("ldst, max_sms 32 x 2 CTAs", {"max_sms": 32, "ctas_per_sm": 2}),
                ("ldst, max_sms 16 x 2 CTAs", {"max_sms": 16, "ctas_per_sm": 2}),
                ("ldst, max_sms 16 x 1 CTA", {"max_sms": 16, "ctas_per_sm": 1}),
                ("bulk/TMA, default grid", {"variant": "bulk"}),
                ("bulk/TMA, 148 SMs x 1 CTA x 1 thread, 6 stages", {"variant": "bulk", "ctas_per_sm": 1, "stages": 6, "tile_bytes": 32768}),
                ("bulk/TMA, max_sms 32 x 1 CTA, 6 stages", {"variant": "bulk", "max_sms": 32, "ctas_per_sm": 1, "stages": 6, "tile_bytes": 32768}),
                ("bulk/TMA, max_sms 32 x 2 CTAs, 3 stages", {"variant": "bulk", "max_sms": 32, "ctas_per_sm": 2, "stages": 3, "tile_bytes": 32768}),
                ("bulk/TMA, max_sms 16 x 2 CTAs, 3 stages", {"variant": "bulk", "max_sms": 16, "ctas_per_sm": 2, "stages": 3, "tile_bytes": 32768}),
                ("bulk/TMA, max_sms 16 x 1 CTA, 6 stages", {"variant": "bulk", "max_sms": 16, "ctas_per_sm": 1, "stages": 6, "tile_bytes": 32768})]
    for name, t in settings:
        plan = F.flowkv_plan(dp.src, dp.dst, dp.requests, F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, t, sc.cuda_stream)
        sc.synchronize()
        copy_loop(plan, 2); torch.cuda.synchronize()
        t0 = ev(); cs_ = []
        t0.record(sc); copy_loop(plan, 3, cs_); torch.cuda.synchronize()
        copy_ms = t0.elapsed_time(cs_[-1]) / 3
        n_copy = max(4, int(100.0 / copy_ms))                         # ~100 ms of copying alone
        t0 = ev(); cs_ = []
        t0.record(sc); copy_loop(plan, n_copy, cs_); torch.cuda.synchronize()
        copy_alone = gb(rate_in_window(t0, cs_, 0, 1e9))
        # both loops ~300 ms of their stand-alone time, started together; every iteration stamps its completion on its
        # own stream and both rates are read over the SAME window: the middle of the time both streams were busy
        n_c, n_g = max(6, int(300.0 / copy_ms)), max(20, int(300.0 / gemm_ms))
        t0 = ev(); gs_, cs_ = [], []
        t0.record(sg)
        sc.wait_event(t0)
        gemm_loop(n_g, gs_)
        copy_loop(plan, n_c, cs_)
        torch.cuda.synchronize()
        end = min(t0.elapsed_time(gs_[-1]), t0.elapsed_time(cs_[-1]))
        lo, hi = 0.15 * end, 0.95 * end
        st = plan.stats
        row = {"config": args.config, "gemm_stream": "high priority" if args.gemm_priority else "default priority",
               "setting": name, "tuning": t, "grid": st["grid"], "variant": st["variant"],
               "mode": st["mode_transfer"], "copy_alone_GBps": copy_alone, "gemm_alone_TFLOPs": gemm_alone,
               "copy_corun_GBps": gb(rate_in_window(t0, cs_, lo, hi)), "gemm_corun_TFLOPs": tf(rate_in_window(t0, gs_, lo, hi)),
               "copy_ms_alone": copy_ms, "window_ms": hi - lo}
        rows.append(row)
        print(json.dumps(row), flush=True)
        plan.destroy()
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump(rows, open(args.out, "w"), indent=1)


if __name__ == "__main__":
    main()
