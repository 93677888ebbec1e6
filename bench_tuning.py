#!/usr/bin/env python
"""bench_tuning.py — A/B sweep of flowkv_tuning settings: workloads x tunings -> kernel time and HBM GB/s.

    python bench_tuning.py '[null, {"ctas_per_sm": 16}, {"variant": "bulk"}]'

Workloads: configs[4] points (32,768 tokens x run length 1 / 2 / contiguous, 1,024 tokens, 128 tokens) and a
3-request slice of configs[3] (rows mode, 80 layers).  Kernel-only timing with a pre-built plan (CUDA events,
median of 8 after 2 warm-ups; L2 flushed between reps when the payload could stay L2-resident).  GB/s counts
read + written bytes.  This is how the defaults in csrc/api.cpp:resolve_shape were chosen."""
import json, sys, itertools
import numpy as np, torch
import os
sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
from paper_2504_03775_b200 import flowkv as F, pools as P, synth
st = torch.cuda.current_stream().cuda_stream
flush = torch.empty(512 << 20, dtype=torch.uint8, device="cuda")
def timeit(fn, reps=8, warm=2, do_flush=False):
    for _ in range(warm): fn()
    torch.cuda.synchronize(); ts = []
    for _ in range(reps):
        if do_flush: flush.zero_()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(); fn(); b.record(); torch.cuda.synchronize(); ts.append(a.elapsed_time(b))
    return min(ts), float(np.median(ts))
shape = synth.LLAMA3_8B
src_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, 16384).bytes(shape)); dst_buf = P.alloc_bytes(synth.PoolSpec("lkbthd", 16, 8192).bytes(shape))
tunings = json.loads(sys.argv[1]) if len(sys.argv) > 1 else [None]
points = [(32768, 1), (32768, 2), (32768, 0), (1024, 1), (128, 0)]
out = []
for T, run in points:
    w = synth.config5_point(T, run); r = w.requests[0]
    src = P.describe(w.src, shape, src_buf.data_ptr()); dst = P.describe(w.dst, shape, dst_buf.data_ptr())
    for t in tunings:
        plan = F.flowkv_plan(src, dst, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)], 0, t, st)
        mn, md = timeit(lambda: plan.transfer(st), do_flush=(2 * w.payload_bytes < (256 << 20)))
        s = plan.stats
        rec = dict(T=T, run=run, tuning=t, min_us=round(mn * 1e3, 2), med_us=round(md * 1e3, 2), gbs=round(2 * w.payload_bytes / md / 1e6), grid=s["grid"], thr=s["threads"], grp=s["group_threads"], tile=s["tile_bytes"])
        print(json.dumps(rec), flush=True); out.append(rec); plan.destroy()
# cfg4-like rows mode: 3 requests, full 80 layers
del src_buf, dst_buf; torch.cuda.empty_cache()
w = synth.config4_hetero(n_requests=3)
dp = P.DevicePools(w, sentinel_dst=False)
for t in tunings:
    plan = dp.plan(0, t, st)
    mn, md = timeit(lambda: plan.transfer(st), reps=5)
    s = plan.stats
    rec = dict(T="cfg4x3", tuning=t, min_us=round(mn * 1e3, 2), med_us=round(md * 1e3, 2), gbs=round(2 * w.payload_bytes / md / 1e6), grid=s["grid"], thr=s["threads"], grp=s["group_threads"], tile=s["tile_bytes"])
    print(json.dumps(rec), flush=True); out.append(rec); plan.destroy()
