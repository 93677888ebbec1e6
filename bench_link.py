#!/usr/bin/env python
"""bench_link.py — what the host link sustains with D2H and H2D in flight together: copy engines
(cudaMemcpyAsync) against the library's pack / unpack kernels storing to / loading from pinned host memory,
alone, together and mixed.  This is the measurement behind flowkv_transfer_via_host's copy-engine mode
(profiles/r01_sweep.md).  configs[1] payload (1.625 GiB each way), CUDA events, best of 3-5.

    python bench_link.py        # prints one line per combination, writes gpurun_out/pcie_duplex.json
"""
import os, sys, json
ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import torch
from paper_2504_03775_b200 import flowkv as F, pools as P, synth

torch.cuda.set_device(0)
N = 1744830464
dev_a = torch.empty(N, dtype=torch.uint8, device="cuda"); dev_a.random_(0, 255)
dev_b = torch.empty(N, dtype=torch.uint8, device="cuda")
host_a = torch.empty(N, dtype=torch.uint8).pin_memory()
host_b = torch.empty(N, dtype=torch.uint8).pin_memory(); host_b.fill_(3)
s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()

def timeit(fn, reps=5):
    fn(); torch.cuda.synchronize()
    best = 1e9
    for _ in range(reps):
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        s1.wait_event(e0); s2.wait_event(e0)
        fn()
        ea, eb = torch.cuda.Event(), torch.cuda.Event()
        ea.record(s1); eb.record(s2)
        torch.cuda.current_stream().wait_event(ea); torch.cuda.current_stream().wait_event(eb)
        e1.record(); torch.cuda.synchronize()
        best = min(best, e0.elapsed_time(e1))
    return best

def ce_d2h():
    with torch.cuda.stream(s1): host_a.copy_(dev_a, non_blocking=True)
def ce_h2d():
    with torch.cuda.stream(s2): dev_b.copy_(host_b, non_blocking=True)
def ce_both():
    ce_d2h(); ce_h2d()
def ce_both_chunked(k=16):
    c = N // k
    for i in range(k):
        with torch.cuda.stream(s1): host_a[i*c:(i+1)*c].copy_(dev_a[i*c:(i+1)*c], non_blocking=True)
        with torch.cuda.stream(s2): dev_b[i*c:(i+1)*c].copy_(host_b[i*c:(i+1)*c], non_blocking=True)

out = {}
for name, fn in [("ce_d2h", ce_d2h), ("ce_h2d", ce_h2d), ("ce_both", ce_both), ("ce_both_chunked16", ce_both_chunked)]:
    ms = timeit(fn)
    out[name] = {"ms": ms, "GBps_each": N / ms / 1e6}
    print(name, out[name], flush=True)

# our kernels: pack (D2H stores) on s1 + unpack (H2D loads) on s2 on independent buffers, various grids
w = synth.config2_llama8b_13k()
dp = P.DevicePools(w)
for variant in ("ldst", "bulk"):
    for ctas in (16, 32, 64, 148, 296):
        tun = {"max_sms": min(ctas, 148), "ctas_per_sm": max(1, ctas // 148), "variant": variant}
        try:
            plan = dp.plan(0, tun)
        except Exception as e:
            print("plan fail", tun, e); continue
        def k_pack(): plan.pack(host_a.data_ptr(), N, s1.cuda_stream)
        def k_unpack(): plan.unpack(host_b.data_ptr(), N, s2.cuda_stream)
        def k_both(): k_pack(); k_unpack()
        def pack_ce(): k_pack(); ce_h2d()
        def ce_unpack(): ce_d2h(); k_unpack()
        for name, fn in [("pack", k_pack), ("unpack", k_unpack), ("both", k_both), ("pack+ce_h2d", pack_ce), ("ce_d2h+unpack", ce_unpack)]:
            ms = timeit(fn, reps=3)
            key = f"{variant}_{ctas}_{name}"
            out[key] = {"ms": ms, "GBps_each": N / ms / 1e6}
            print(key, out[key], flush=True)
        plan.destroy()
os.makedirs(os.path.join(ROOT, "gpurun_out"), exist_ok=True)
json.dump(out, open(os.path.join(ROOT, "gpurun_out", "pcie_duplex.json"), "w"), indent=1)
