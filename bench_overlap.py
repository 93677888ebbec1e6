#!/usr/bin/env python
"""bench_overlap.py — layer-wise transfer hidden under prefill (S§8f NEXT-2: "layer-range transfers ... overlap
with prefill"; P:L28 Splitwise-style overlap; P:L222-224 the paper's layerwise ablation).

    python bench_overlap.py [--out gpurun_out/overlap.json] [--gemms-per-layer 6]

The paper's "layerwise" scheme was its slow one because it multiplied NCCL calls (one per block per layer).  Here a
layer's KV is ONE window (flowkv_pack_window: one kernel, one contiguous message), so going layer by layer costs
2 launches + 2 copies per layer and lets the link time disappear under the prefill that produces the next layers.

Stand-in for prefill: per layer, a few bf16 8192^3 cuBLAS GEMMs on the compute stream (library code, not the
product; 6 per layer ~ the FLOPs of a 13k-token Llama-3-8B prefill layer).  After layer l's GEMMs an event
releases the transfer of layer l on side streams: pack_window -> D2H -> (host = network stand-in) -> H2D ->
unpack_window.  Reported: prefill alone, prefill followed by the whole transfer (device->device, and through the
host), and prefill with the layer-wise transfer overlapped; "exposed" = time from the end of prefill compute until
the last byte is in the dst pool.  CUDA events; configs[1] payload.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "overlap.json"))
    ap.add_argument("--gemms-per-layer", type=int, default=6)
    ap.add_argument("--reps", type=int, default=3)
    args = ap.parse_args()
    import torch
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F, pools as P, synth

    torch.cuda.set_device(0)
    w = synth.config2_llama8b_13k()
    dp = P.DevicePools(w, sentinel_dst=False)
    L, payload = w.shape.num_layers, w.payload_bytes
    per_layer = payload // L
    N = 8192
    a = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    b = torch.randn(N, N, device="cuda", dtype=torch.bfloat16)
    c = torch.empty(N, N, device="cuda", dtype=torch.bfloat16)
    comp = torch.cuda.current_stream()
    s_out, s_in = torch.cuda.Stream(), torch.cuda.Stream()
    host = torch.empty(payload, dtype=torch.uint8).pin_memory()
    out_slots = [P.alloc_bytes(per_layer) for _ in range(2)]
    in_slots = [P.alloc_bytes(per_layer) for _ in range(2)]
    ev = lambda: torch.cuda.Event(enable_timing=True)
    plan = F.flowkv_plan(dp.src, dp.dst, dp.requests, 0, None, comp.cuda_stream)
    scratch_bytes = F.flowkv_via_host_scratch_bytes(plan, 0)
    scratch = P.alloc_bytes(scratch_bytes)
    # device-resident block tables for the plan-free layer-range launches (flowkv_transfer_tables_layers)
    r0 = w.requests[0]
    d_st = torch.from_numpy(r0.src_blocks[None, :].copy()).cuda()
    d_dt = torch.from_numpy(r0.dst_blocks[None, :].copy()).cuda()
    d_len = torch.tensor([r0.num_tokens], dtype=torch.int32, device="cuda")
    d_flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    torch.cuda.synchronize()

    def prefill_layer():
        for _ in range(args.gemms_per_layer):
            torch.matmul(a, b, out=c)

    def run(mode: str):
        """-> (ms until prefill compute ends, ms until everything has landed)"""
        e0, e_pre, e_all = ev(), ev(), ev()
        e0.record(comp)
        s_out.wait_event(e0)
        s_in.wait_event(e0)
        last_in = None
        for l in range(L):
            prefill_layer()
            if mode == "layerwise_via_host":
                done = torch.cuda.Event()
                done.record(comp)
                s_out.wait_event(done)                                   # layer l's KV exists now
                o, i = out_slots[l & 1], in_slots[l & 1]
                hv = host[l * per_layer:(l + 1) * per_layer]
                F.flowkv_pack_window(plan, o.data_ptr(), per_layer, l, l + 1, s_out.cuda_stream)
                with torch.cuda.stream(s_out):
                    hv.copy_(o, non_blocking=True)
                landed = torch.cuda.Event()
                landed.record(s_out)
                s_in.wait_event(landed)
                with torch.cuda.stream(s_in):
                    i.copy_(hv, non_blocking=True)
                F.flowkv_unpack_window(plan, i.data_ptr(), per_layer, l, l + 1, s_in.cuda_stream)
            elif mode == "layerwise_d2d":
                done = torch.cuda.Event()
                done.record(comp)
                s_out.wait_event(done)
                F.flowkv_transfer_layers(plan, l, l + 1, s_out.cuda_stream)
            elif mode == "layerwise_d2d_tables":                         # no host plan: the kernel reads the tables
                done = torch.cuda.Event()
                done.record(comp)
                s_out.wait_event(done)
                F.flowkv_transfer_tables_layers(dp.src, dp.dst, d_st.data_ptr(), d_dt.data_ptr(), d_len.data_ptr(), 1,
                                                d_st.shape[1], d_dt.shape[1], r0.num_tokens, l, l + 1, d_flag.data_ptr(),
                                                None, s_out.cuda_stream)
        e_pre.record(comp)
        if mode == "serial_d2d":
            F.flowkv_transfer(plan, comp.cuda_stream)
        elif mode == "serial_via_host":
            F.flowkv_transfer_via_host(plan, host.data_ptr(), payload, 0, 0, comp.cuda_stream, scratch.data_ptr(), scratch_bytes)
        for st in (s_out, s_in):
            j = torch.cuda.Event()
            j.record(st)
            comp.wait_event(j)
        e_all.record(comp)
        torch.cuda.synchronize()
        return e0.elapsed_time(e_pre), e0.elapsed_time(e_all)

    rows = []
    for mode in ("prefill_only", "serial_d2d", "layerwise_d2d", "layerwise_d2d_tables", "serial_via_host", "layerwise_via_host"):
        run(mode)
        best = min((run(mode) for _ in range(args.reps)), key=lambda t: t[1])
        row = {"mode": mode, "prefill_ms": best[0], "total_ms": best[1], "exposed_transfer_ms": best[1] - best[0],
               "launches_per_request": {"prefill_only": 0, "serial_d2d": 1, "layerwise_d2d": L, "layerwise_d2d_tables": L, "serial_via_host": 64,
                                        "layerwise_via_host": 2 * L}[mode]}
        rows.append(row)
        print(json.dumps(row), flush=True)
    base = rows[0]["prefill_ms"]
    for r in rows:
        r["prefill_slowdown_pct"] = 100.0 * (r["prefill_ms"] / base - 1.0)
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump({"gemms_per_layer": args.gemms_per_layer, "layers": L, "payload_bytes": payload, "rows": rows},
              open(args.out, "w"), indent=1)
    print(json.dumps({"summary": [(r["mode"], round(r["total_ms"], 2), round(r["exposed_transfer_ms"], 2),
                                   round(r["prefill_slowdown_pct"], 2)) for r in rows]}))


if __name__ == "__main__":
    main()
