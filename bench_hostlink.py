#!/usr/bin/env python
"""bench_hostlink.py — what the host link gives the pinned-host route (S§8f NEXT-3), measured without any of this
library's kernels: the bound that `bench.py`'s `e2e` number is read against.

    python bench_hostlink.py [--bytes 1744830464] [--out gpurun_out/hostlink.json]

Copy engines only (`cudaMemcpyAsync` through torch; library calls, not the product):
  1. one contiguous D2H and one contiguous H2D of the payload, each alone and both at once;
  2. the chunked duplex pipeline the host route has to be: chunk c goes device -> pinned host, and comes back
     host -> device as soon as it has landed, so chunk c+1 outbound overlaps chunk c inbound — for several chunk
     counts, with one queue per direction;
  3. the per-chunk timeline of one such run (start / end of every copy on a common clock), which shows the two
     directions' rates while both are busy and the head / tail where one crosses alone.
"""
from __future__ import annotations

import argparse
import json
import os
import sys

ROOT = os.path.dirname(os.path.abspath(__file__))


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--bytes", type=int, default=13312 * 131072)            # configs[1] payload
    ap.add_argument("--out", default=os.path.join(ROOT, "gpurun_out", "hostlink.json"))
    args = ap.parse_args()
    import torch
    torch.cuda.set_device(0)
    n = args.bytes
    dev_a = torch.empty(n, dtype=torch.uint8, device="cuda")
    dev_b = torch.empty(n, dtype=torch.uint8, device="cuda")
    host = torch.empty(n, dtype=torch.uint8, pin_memory=True)
    host2 = torch.empty(n, dtype=torch.uint8, pin_memory=True)
    main_s = torch.cuda.current_stream()
    qd, qh = torch.cuda.Stream(), torch.cuda.Stream()
    T = lambda: torch.cuda.Event(enable_timing=True)
    E = lambda: torch.cuda.Event()
    gbs = lambda ms: n / (ms * 1e-3) / 1e9
    out = {"bytes": n}

    def best(fn, reps=4):
        ts = []
        for _ in range(reps):
            torch.cuda.synchronize()
            a, b = T(), T()
            a.record(main_s); fn(); b.record(main_s); torch.cuda.synchronize()
            ts.append(a.elapsed_time(b))
        return min(ts)

    out["d2h_alone_GBps"] = gbs(best(lambda: host.copy_(dev_a, non_blocking=True)))
    out["h2d_alone_GBps"] = gbs(best(lambda: dev_b.copy_(host, non_blocking=True)))

    def both():
        qd.wait_stream(main_s)
        with torch.cuda.stream(qd):
            host2.copy_(dev_a, non_blocking=True)
        dev_b.copy_(host, non_blocking=True)
        main_s.wait_stream(qd)
    out["duplex_whole_payload_GBps_each_way"] = gbs(best(both))

    def pipeline(chunks, stamps=None):
        wb = n // chunks
        t0 = E()
        t0.record(main_s)
        qd.wait_event(t0); qh.wait_event(t0)
        for c in range(chunks):
            sl = slice(c * wb, n if c == chunks - 1 else (c + 1) * wb)
            landed = E()
            with torch.cuda.stream(qd):
                if stamps is not None:
                    e = T(); e.record(qd); stamps["d0"].append(e)
                host[sl].copy_(dev_a[sl], non_blocking=True)
                if stamps is not None:
                    e = T(); e.record(qd); stamps["d1"].append(e)
                landed.record(qd)
            qh.wait_event(landed)
            with torch.cuda.stream(qh):
                if stamps is not None:
                    e = T(); e.record(qh); stamps["h0"].append(e)
                dev_b[sl].copy_(host[sl], non_blocking=True)
                if stamps is not None:
                    e = T(); e.record(qh); stamps["h1"].append(e)
        main_s.wait_stream(qd); main_s.wait_stream(qh)

    out["chunked_pipeline"] = []
    for chunks in (8, 16, 32, 64, 128):
        ms = best(lambda: pipeline(chunks))
        out["chunked_pipeline"].append({"chunks": chunks, "ms": ms, "GBps_each_way": gbs(ms)})
        print(json.dumps(out["chunked_pipeline"][-1]), flush=True)

    chunks = 16
    pipeline(chunks); torch.cuda.synchronize()
    st = {"d0": [], "d1": [], "h0": [], "h1": []}
    base = T(); base.record(main_s)
    pipeline(chunks, st)
    torch.cuda.synchronize()
    wb = n // chunks
    rows = []
    for c in range(chunks):
        d0, d1, h0, h1 = (base.elapsed_time(st[k][c]) for k in ("d0", "d1", "h0", "h1"))
        rows.append({"chunk": c, "d2h_start_ms": d0, "d2h_end_ms": d1, "d2h_GBps": wb / (d1 - d0) / 1e6,
                     "h2d_start_ms": h0, "h2d_end_ms": h1, "h2d_GBps": wb / (h1 - h0) / 1e6})
    out["timeline_16_chunks"] = rows
    mid = rows[2:-2]
    out["duplex_rates_mid_pipeline_GBps"] = {"d2h": sum(r["d2h_GBps"] for r in mid) / len(mid),
                                             "h2d": sum(r["h2d_GBps"] for r in mid) / len(mid)}
    print(json.dumps({k: v for k, v in out.items() if k not in ("timeline_16_chunks", "chunked_pipeline")}), flush=True)
    os.makedirs(os.path.dirname(args.out), exist_ok=True)
    json.dump(out, open(args.out, "w"), indent=1)


if __name__ == "__main__":
    main()
