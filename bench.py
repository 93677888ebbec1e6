#!/usr/bin/env python
"""bench.py — FlowKV KV-cache transfer on B200: device-timed GB/s, % of HBM peak, launches/request.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config cfg2|cfg1|cfg3|cfg4]
    python bench.py --impl reference ...      # the CPU oracle, as it stands, on the host cores
    python bench.py --sweep                   # BASELINE.json configs[4]: length x run-length sweep

One "step" is one pass of the whole hot path over one transfer batch: validate + bidirectional
segment alignment + tile schedule + plan upload (flowkv_plan), ONE persistent kernel (flowkv_transfer),
plan release.  Pools are resident in HBM before the timed region.  Prints ONE JSON line (rank 0).
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "kv_transfer_payload_GBps"      # BASELINE.json metric: KV transfer GB/s (payload bytes moved / device time)
UNIT = "GB/s"


# ---------------------------------------------------------------------------------------------------
# clocks during the timed region
# ---------------------------------------------------------------------------------------------------
class ClockSampler:
    """Samples SM clock and clock-event (throttle) reasons through NVML while the timed region runs."""
    REASONS = {0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
               0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x10: "sync_boost"}

    def __init__(self, device_index: int, period_s: float = 0.001):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        self.period = period_s
        self.h = None
        try:
            import pynvml
            import torch
            pynvml.nvmlInit()
            self.nv = pynvml
            try:
                uuid = str(torch.cuda.get_device_properties(device_index).uuid)
                if not uuid.startswith("GPU-"):
                    uuid = "GPU-" + uuid
                self.h = pynvml.nvmlDeviceGetHandleByUUID(uuid.encode())
            except Exception:
                self.h = pynvml.nvmlDeviceGetHandleByIndex(device_index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception as e:  # pragma: no cover
            self.err = repr(e)
            self.h = None

    def _reasons_now(self) -> int:
        for fn in ("nvmlDeviceGetCurrentClocksEventReasons", "nvmlDeviceGetCurrentClocksThrottleReasons"):
            if hasattr(self.nv, fn):
                try:
                    return int(getattr(self.nv, fn)(self.h))
                except Exception:
                    pass
        return 0

    def sample(self):
        if self.h is None:
            return
        try:
            self.samples.append(int(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM)))
            bits = self._reasons_now()
            for b, name in self.REASONS.items():
                if bits & b:
                    self.reasons.add(name)
        except Exception:
            pass

    def _run(self):
        while not self._stop.is_set():
            self.sample()
            self._stop.wait(self.period)

    def start(self):
        """One sample now (the GPU is already under load: call after the warm-up steps have been queued), then one
        per millisecond until stop(); stop() takes a last one, so even a 10 ms timed region is covered."""
        self.sample()
        if self.h is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self) -> dict:
        self.sample()
        self._stop.set()
        if self._thr:
            self._thr.join()
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "samples": 0}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ---------------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------------
def build_workload(name: str, free_bytes: int):
    from paper_2504_03775_b200 import synth
    budget = int(0.85 * free_bytes)
    if name == "cfg1":
        return synth.config1_tiny(), "configs[0] Tiny: 2 layers, 2 KV heads, head_dim 64, fp16, 1 x 1000 tokens"
    if name == "cfg2":
        return (synth.config2_llama8b_13k(),
                "configs[1] Llama-3-8B KV: 32 layers, 8 KV heads, head_dim 128, bf16, block 16, 1 x 13,312 tokens, "
                "src 16,384-block pool (32 GiB) runs~Geom(mean 4), dst contiguous")
    if name == "cfg2sep":
        return (synth.config2_llama8b_13k(),
                "configs[1] request and tables, src pool as 32 SEPARATE per-layer tensors of 1 GiB (the cache the paper "
                "starts from, P:L98; flowkv_pool.plane_offsets), dst one contiguous pool")
    if name == "cfg2mig":
        w = synth.make_workload("cfg2_mig_13k", synth.SEED_BASE + 2000, synth.LLAMA3_8B, [13312],
                                "lkbthd", 16, ("geometric", 4.0), 16384, "blkthd", 16, ("contiguous",), 1024)
        return w, ("configs[1] request and src tables; src pool = 32 SEPARATE per-layer tensors (the cache the paper starts "
                   "from, P:L98), dst = ONE (B,L,2,H) tensor: Eq. 5's re-layout fused into the move, one launch")
    if name in ("cfg2bm", "cfg2bm_ragged"):
        w = synth.config2_blockmajor("blkthd", tokens=13312 if name == "cfg2bm" else 13307)
        return w, ("configs[1] request and tables, both pools in the paper's (B,L,2,H) order (Eq. 5; BLKTHD): "
                   f"1 x {w.total_tokens} tokens, whole-block runs move as flat 2 MiB-per-block spans")
    if name == "cfg3":
        w = synth.config3_batched(budget_bytes=budget)
        return w, (f"configs[2] batched Llama-3-8B KV: first {w.notes['n_requests']} of 64 requests (fit rule), "
                   "lognormal lengths, src runs mean 2, dst runs mean 16, one batch")
    if name == "cfg4":
        w = synth.config4_hetero(budget_bytes=budget)
        return w, (f"configs[3] hetero Llama-3-70B KV: first {w.notes['n_requests']} of 16 requests (fit rule), "
                   "src block 16 LKBTHD -> dst block 64 BLKHTD")
    raise SystemExit(f"unknown --config {name}")


def workload_config(w, desc: str, n_segments: int) -> dict:
    """`config` of the JSON line: names the workload only, so both arms (ours, --impl reference) print the same dict.
    What an arm DOES with it (step, launch shape, dst placement) goes under the line's `run` key."""
    payload = w.payload_bytes
    return {"workload": desc, "name": w.name, "requests": len(w.requests), "tokens": w.total_tokens,
            "payload_bytes": payload, "segments": int(n_segments),
            "mean_src_run_blocks": run_mean(w, "src"), "mean_dst_run_blocks": run_mean(w, "dst"),
            "l2": "inputs larger than L2 (payload %.0f MiB >> 126 MB), no flush" % (payload / 2 ** 20)
            if payload > 512 * 2 ** 20 else "payload is L2-resident; no flush (latency-bound config)"}


def load_peaks() -> tuple:
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        j = json.load(open(p))
        return float(j["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, plain torch copy, read+write bytes)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


NCU_CAPTURES = {      # workload name -> (committed summary of its `ncu --set full` capture, commit whose kernels it measured)
    "cfg2_llama8b_13k": ("r03_ncu_full_cfg2_fk_span_ldst.csv", "a3a5a7c"),
    "cfg2_mig_13k+po": ("r03_ncu_full_cfg2mig_fk_rows_ldst_po.csv", "a3a5a7c"),
    "cfg2_llama8b_13k+po": ("r02_ncu_full_cfg2sep_fk_span_ldst_po.csv", "32ce955"),
    "cfg2_blkthd_13k": ("r02_ncu_full_cfg2bm_fk_flat_ldst.csv", "8d434be"),
    "cfg2_llama8b_13k+tables": ("r02_ncu_full_cfg2_fk_tables_ldst.csv", "8d434be"),
    "cfg3_batched_8b": ("r02_ncu_full_cfg3_fk_span_ldst.csv", "8d434be"),
    "cfg4_hetero_70b": ("r03_ncu_full_cfg4_fk_rows_ldst.csv", "a3a5a7c"),
    "cfg4_hetero_70b+bulk": ("r02_ncu_full_cfg4_fk_rows_tma.csv", "8d434be"),
}


def traffic_source(workload_key: str):
    """Where `roofline.traffic` comes from: a COMMITTED ncu capture (another box, an earlier commit), not this run —
    the file and the commit whose kernels it measured, so a stale constant is visible in the line itself."""
    ent = NCU_CAPTURES.get(workload_key)
    if not ent:
        return None
    return f"profiles/{ent[0]} @ {ent[1]}; committed ncu --set full capture, not measured by this run"


def load_traffic(workload_key: str):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch (bytes; mean over the captured launches) from the
    committed summary of the ncu --set full capture of this workload's kernel, or None."""
    import csv
    ent = NCU_CAPTURES.get(workload_key)
    if not ent:
        return None
    try:
        rows = list(csv.reader(open(os.path.join(ROOT, "profiles", ent[0]))))
        head, units = rows[0], rows[1]
        scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9, "Tbyte": 1e12}
        tot = []
        for r in rows[2:]:
            v = 0.0
            for col in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
                i = head.index(col)
                v += float(r[i]) * scale[units[i]]
            tot.append(v)
        return sum(tot) / len(tot) if tot else None
    except Exception:
        return None


# ---------------------------------------------------------------------------------------------------
# the CPU oracle as a baseline (bounded sample)
# ---------------------------------------------------------------------------------------------------
def oracle_geoms(w, num_layers=None):
    from oracle import oracle as O
    L = w.shape.num_layers if num_layers is None else num_layers
    mk = lambda spec: getattr(O.PoolGeom, spec.layout)(L, w.shape.num_kv_heads, w.shape.head_dim, w.shape.elem_bytes,
                                                       spec.num_blocks, spec.block_size)
    return mk(w.src), mk(w.dst)


def oracle_sample_setup(w, n_layers: int, src_dev=None):
    """Host copies of the first n_layers of the pools, laid out as n_layers-deep pools of the same kind.
    For LKBTHD the first layers are a prefix of the buffer; for BLKHTD each block keeps its first layers."""
    import dataclasses
    from oracle import oracle as O
    gs_full, gd_full = oracle_geoms(w)
    gs, gd = oracle_geoms(w, n_layers)
    rng = np.random.default_rng(1)

    def host_pool(g, full, dev, layout):
        nbytes = g.span_bytes()
        if dev is not None and layout == "lkbthd":
            return dev[:nbytes].cpu().numpy()
        return rng.integers(0, 256, size=nbytes, dtype=np.uint8)     # values are irrelevant to a copy's speed
    src = host_pool(gs, gs_full, src_dev, w.src.layout)
    dst = np.zeros(gd.span_bytes(), np.uint8)
    dst[:] = 0xA5                                                    # touch every page before timing
    return O, gs, gd, src, dst


def oracle_run(O, gs, gd, src, dst, w, n_tokens_cap=None) -> int:
    """Token-by-token oracle transfer over every request (optionally only the first tokens of each).
    Returns payload bytes moved."""
    moved = 0
    for r in w.requests:
        T = r.num_tokens if n_tokens_cap is None else min(r.num_tokens, n_tokens_cap)
        O.transfer(src, gs, dst, gd, r.src_blocks[: -(-T // w.src.block_size)], r.dst_blocks[: -(-T // w.dst.block_size)], T)
        moved += T * 2 * gs.num_layers * gs.num_kv_heads * gs.head_dim * gs.elem_bytes
    return moved


def cpu_baseline(w, src_dev, target_s: float = 12.0) -> dict:
    n_layers = 1
    O, gs, gd, src, dst = oracle_sample_setup(w, n_layers, src_dev)
    t0 = time.perf_counter()
    moved = oracle_run(O, gs, gd, src, dst, w)
    dt = time.perf_counter() - t0
    reps = 1
    while dt < target_s and reps < 1024:                               # repeat the same sample until ~target_s of CPU work
        t1 = time.perf_counter()
        moved += oracle_run(O, gs, gd, src, dst, w)
        dt += time.perf_counter() - t1
        reps += 1
    return {"value": moved / dt / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": f"layer 0 of {w.shape.num_layers} (all requests, all tokens, both K and V) of the same workload, "
                      f"{reps} passes, {dt:.1f} s of single-threaded oracle/flowkv_oracle.c (gcc -O2)",
            "seconds": dt, "host_cores_available": os.cpu_count()}


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle, as it stands, on the host cores
# ---------------------------------------------------------------------------------------------------
def run_reference(args) -> None:
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, desc = build_workload(args.config, 170 * 2 ** 30)
    O, gs, gd, src, dst = oracle_sample_setup(w, 1, None)
    # calibrate: how many tokens per request keep the whole run within ~2 minutes
    t0 = time.perf_counter()
    moved = oracle_run(O, gs, gd, src, dst, w, n_tokens_cap=512)
    rate = moved / max(time.perf_counter() - t0, 1e-6)               # bytes/s
    budget_per_step = 100.0 / max(args.steps + args.warmup, 1)
    per_tok = 2 * gs.num_kv_heads * gs.head_dim * gs.elem_bytes * len(w.requests)
    cap = int(max(64, min(max(r.num_tokens for r in w.requests), budget_per_step * rate / per_tok)))
    for _ in range(args.warmup):
        oracle_run(O, gs, gd, src, dst, w, cap)
    t0 = time.perf_counter()
    moved = 0
    for _ in range(args.steps):
        moved += oracle_run(O, gs, gd, src, dst, w, cap)
    dt = time.perf_counter() - t0
    val = moved / dt / 1e9
    sample = (f"layer 0 of {w.shape.num_layers}, first {cap} tokens of each request, per step; "
              f"single-threaded oracle/flowkv_oracle.c (gcc -O2), host-resident pools")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": dt / max(args.steps, 1) * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "u16", "data": "synthetic",
            "config": workload_config(w, desc, sum(O.count_segments(r.src_blocks, w.src.block_size, r.dst_blocks,
                                                                     w.dst.block_size, r.num_tokens) for r in w.requests)),
            "run": {"step": "okv_transfer (oracle/flowkv_oracle.c) over a bounded sample of the workload per step; "
                            "host-resident pools, no device"},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# our arm
# ---------------------------------------------------------------------------------------------------
def host_info(device_index: int) -> dict:
    """What SURVEY §8d asks to state beside the numbers: the host CPU model behind `cpu_baseline.cores` and the PCIe
    link the pinned-host route runs over (generation and width as NVML reports them, current / maximum)."""
    info = {"cpu_model": None, "host_cores": os.cpu_count()}
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                info["cpu_model"] = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    try:
        import pynvml
        import torch
        pynvml.nvmlInit()
        uuid = str(torch.cuda.get_device_properties(device_index).uuid)
        h = pynvml.nvmlDeviceGetHandleByUUID(("GPU-" + uuid if not uuid.startswith("GPU-") else uuid).encode())
        info["pcie"] = {"gen_current": int(pynvml.nvmlDeviceGetCurrPcieLinkGeneration(h)),
                        "gen_max": int(pynvml.nvmlDeviceGetMaxPcieLinkGeneration(h)),
                        "width_current": int(pynvml.nvmlDeviceGetCurrPcieLinkWidth(h)),
                        "width_max": int(pynvml.nvmlDeviceGetMaxPcieLinkWidth(h))}
    except Exception as e:  # pragma: no cover
        info["pcie"] = {"error": repr(e)}
    return info


def device_tables_of(w, device):
    """Padded block tables + lengths resident on the device, as flowkv_transfer_tables takes them."""
    import torch
    n_rq = len(w.requests)
    max_t = max((r.num_tokens for r in w.requests), default=0)
    ws_, wd_ = max(1, -(-max_t // w.src.block_size)), max(1, -(-max_t // w.dst.block_size))
    hs_, hd_ = np.full((n_rq, ws_), -1, np.int32), np.full((n_rq, wd_), -1, np.int32)
    for i, r in enumerate(w.requests):
        hs_[i, :len(r.src_blocks)], hd_[i, :len(r.dst_blocks)] = r.src_blocks, r.dst_blocks
    return (torch.from_numpy(hs_).to(device), torch.from_numpy(hd_).to(device),
            torch.tensor([r.num_tokens for r in w.requests], dtype=torch.int32, device=device),
            torch.zeros(1, dtype=torch.int32, device=device), n_rq, ws_, wd_, max_t)


def time_steps(F, w, src, dst, requests, K, W, tuning, stream, barrier, local, dev_tables=None, latency_reps=0):
    """W warm-up steps, then EXACTLY K timed steps of the whole hot path (plan + one kernel + release, or the
    table-driven launch) bracketed by barrier + synchronize; one CUDA-event pair around every kernel launch, on
    the launching stream.  Returns a dict of raw measurements (this rank's)."""
    import torch
    s = stream.cuda_stream
    XFER_ONLY = F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK      # the step moves pool -> pool only

    def step(ev_a=None, ev_b=None):
        if dev_tables is not None:
            st_, dt_, ln_, fl_, n_rq, ws_, wd_, max_t = dev_tables
            if ev_a is not None:
                ev_a.record(stream)
            F.flowkv_transfer_tables(src, dst, st_.data_ptr(), dt_.data_ptr(), ln_.data_ptr(), n_rq, ws_, wd_, max_t,
                                     fl_.data_ptr(), tuning, s)             # ONE launch, nothing else
            if ev_b is not None:
                ev_b.record(stream)
            return
        plan = F.flowkv_plan(src, dst, requests, XFER_ONLY, tuning, s)   # a1-a4 (upload is stream-ordered)
        if ev_a is not None:
            ev_a.record(stream)
        F.flowkv_transfer(plan, s)                                           # a5: ONE launch
        if ev_b is not None:
            ev_b.record(stream)
        plan.destroy()                                                       # stream-ordered free

    for _ in range(max(W, 3)):
        step()
    plan0 = F.flowkv_plan(src, dst, requests, XFER_ONLY, tuning, s)
    stats = plan0.stats
    plan0.destroy()
    ka = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    kb = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    clocks = ClockSampler(local)
    barrier()
    for _ in range(3):                       # the sampler's first sample must see the GPU under this load
        step()
    clocks.start()
    n0 = F.flowkv_launch_count()
    c0 = F.flowkv_api_call_count()
    e0.record(stream)
    for k in range(K):
        step(ka[k], kb[k])
    e1.record(stream)
    barrier()
    launches = F.flowkv_launch_count() - n0
    api_calls = F.flowkv_api_call_count() - c0
    clk = clocks.stop()
    per_kernel = [a.elapsed_time(b) for a, b in zip(ka, kb)]
    out = {"t_ms": e0.elapsed_time(e1), "kern_ms": float(np.mean(per_kernel)), "kern_min_ms": float(np.min(per_kernel)),
           "launches": int(launches), "api_calls": int(api_calls), "clocks": clk, "stats": stats}
    if latency_reps:
        # true request latency: host wall clock from the flowkv_plan call until the stream has drained, one
        # synchronous request at a time (nothing pipelined, nothing queued behind another batch)
        lat = []
        for _ in range(latency_reps):
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            if dev_tables is not None:
                step()
                plan = None
            else:
                plan = F.flowkv_plan(src, dst, requests, XFER_ONLY, tuning, s)
                F.flowkv_transfer(plan, s)
            stream.synchronize()
            lat.append((time.perf_counter() - t0) * 1e3)
            if plan is not None:
                plan.destroy()
        out["latency_ms_call_to_done"] = float(np.median(lat))
        out["latency_ms_call_to_done_min"] = float(np.min(lat))
    return out


def run_mean(w, side: str) -> float:
    """Mean length (blocks) of the maximal +1 runs in the generated block tables (input statistics, S§8d)."""
    from paper_2504_03775_b200 import synth
    tabs = [r.src_blocks if side == "src" else r.dst_blocks for r in w.requests]
    return sum(len(t) for t in tabs) / max(1, sum(synth.n_runs(t) for t in tabs))


def kernel_name(stats, device_tables: bool) -> str:
    if device_tables:
        return "fk_tables_ldst"
    if stats["variant"] == 2:       # FLOWKV_VARIANT_BULK: the TMA kernels (rows mode = the tensor path)
        return {1: "fk_span_bulk", 2: "fk_rows_tma", 3: "fk_flat_bulk"}[stats["mode_transfer"]]
    return {1: "fk_span_ldst", 2: "fk_rows_ldst", 3: "fk_flat_ldst"}[stats["mode_transfer"]]


def roofline_of(m, payload, w_key, stats, K, device_tables, po=False):
    peak, peak_src = load_peaks()
    achieved = 2 * payload / (m["kern_ms"] * 1e-3) / 1e9
    tkey = w_key + "+po" if po else w_key
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            # `frac` is read against a measured PLAIN COPY (the contract's denominator), which a good copy kernel can
            # beat by a few per cent — it says "no slower than a contiguous copy", not "how much headroom is left".
            # The headroom figure is the fraction of the nominal 8 TB/s (always < 1):
            "frac_of": "measured plain device copy (MEASURED_PEAKS.json); may read a little above 1",
            "vs_plain_copy": achieved / peak, "frac_of_nominal_8TBps": achieved / 8000.0,
            "traffic": load_traffic(tkey), "traffic_source": traffic_source(tkey), "peak_source": peak_src,
            # pools with per-plane offsets (cfg2sep) run the *_po instantiation of the same loop body
            "kernel": kernel_name(stats, device_tables) + ("_po" if po else ""),
            "kernel_ms_avg": m["kern_ms"], "kernel_ms_min": m["kern_min_ms"], "algorithmic_bytes_per_launch": 2 * payload,
            "kernel_share_of_step": m["kern_ms"] / (m["t_ms"] / K)}


def run_ours(args) -> None:
    import torch
    import torch.distributed as dist
    from paper_2504_03775_b200 import build as B
    B.build()
    from paper_2504_03775_b200 import flowkv as F
    from paper_2504_03775_b200 import pools as P
    from paper_2504_03775_b200 import shard

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = 0 if args.same_device else int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    assert local < torch.cuda.device_count(), f"rank {rank}: no cuda:{local} on this node (--gpus {args.gpus})"
    torch.cuda.set_device(local)
    backend = "gloo" if args.same_device else "nccl"     # ranks sharing one GPU (tests) cannot form an NCCL group
    reduce_dev = "cpu" if args.same_device else "cuda"
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=torch.device("cuda", local))
        else:
            dist.init_process_group("gloo")
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    tuning = json.loads(args.tuning) if args.tuning else None
    stream = torch.cuda.current_stream()
    K, W = args.steps, args.warmup

    def primary():
        """Everything measured on --config's workload; its pools die with this frame (the batched config that follows
        sizes its own pools from the free HBM)."""
        s = stream.cuda_stream
        free_b, _total = torch.cuda.mem_get_info()
        if args.same_device:
            free_b //= world
        w, desc = build_workload(args.config, free_b)
        dp = P.DevicePools(w, device=f"cuda:{local}", sentinel_dst=False, separate_src_layers=args.config in ("cfg2sep", "cfg2mig"))
        payload = w.payload_bytes
        # --peer: rank r's kernel stores into the dst pool that rank (r+1) % N owns, mapped through CUDA IPC — the paper's
        # single-machine "IPC" mode as a one-sided put; over NVLink when the ranks sit on different GPUs
        dst_desc, peer_keep = dp.dst, None
        if args.peer:
            assert world > 1, "--peer needs at least 2 ranks (torchrun, or bench.py --gpus N)"
            from paper_2504_03775_b200 import peer
            handles = [None] * world
            dist.all_gather_object(handles, peer.export_pool(dp.dst_buf))
            peer_keep = peer.import_pool(handles[(rank + 1) % world])
            dst_desc = P.describe(w.dst, w.shape, peer_keep.data_ptr())
            barrier()

        dev_tables = device_tables_of(w, dp.device) if args.device_tables else None
        m = time_steps(F, w, dp.src, dst_desc, dp.batch, K, W, tuning, stream, barrier, local, dev_tables,
                       latency_reps=max(20, args.latency_reps))
        stats = m["stats"]
        t_ms = shard.max_over_ranks(m["t_ms"], device=reduce_dev)                   # max over ranks, device-timed
        value = world * K * payload / (t_ms * 1e-3) / 1e9
        # one record per rank, so that a rank that moved nothing, fell back or sat on the wrong device shows in the line
        mine = {"rank": rank, "pid": os.getpid(), "device_index": local,
                "device_uuid": str(torch.cuda.get_device_properties(local).uuid), "t_ms": m["t_ms"], "kernel_ms_avg": m["kern_ms"],
                "gpu_launches": m["launches"], "payload_bytes_moved": K * payload,
                "dst": "next rank's pool (CUDA IPC)" if args.peer else "own pool"}
        if args.peer:
            # the importing side's check: a sample of what this rank's kernel stored through the IPC mapping, read back
            # through that mapping, against the same sample computed from this rank's src pool by the definition
            # (token t of layer 0, K plane: src block table -> dst block table); a few tokens, exact bytes
            tokb = w.shape.num_kv_heads * w.shape.head_dim * w.shape.elem_bytes
            r0 = w.requests[0]
            ok = True
            for t in sorted({0, r0.num_tokens // 2, r0.num_tokens - 1}):
                sb, so = int(r0.src_blocks[t // w.src.block_size]), t % w.src.block_size
                db, do = int(r0.dst_blocks[t // w.dst.block_size]), t % w.dst.block_size
                if w.src.layout == "lkbthd" and w.dst.layout == "lkbthd":
                    a0 = (sb * w.src.block_size + so) * tokb
                    b0 = (db * w.dst.block_size + do) * tokb
                    ok = ok and bool(torch.equal(dp.src_buf[a0:a0 + tokb].cpu(), peer_keep[b0:b0 + tokb].cpu()))
            mine["peer_sample_matches_src"] = ok
        per_rank = [None] * world
        if world > 1:
            dist.all_gather_object(per_rank, mine)
        else:
            per_rank = [mine]

        line = None
        if rank == 0:
            m["t_ms"] = t_ms
            wkey = w.name + ("+tables" if args.device_tables else "+bulk" if stats["variant"] == 2 and stats["mode_transfer"] == 2 else "")
            line = {
                "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": max(W, 3),
                "ms_per_step": t_ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "u16", "data": "synthetic",
                "config": workload_config(w, desc, stats["n_segments"]),
                "run": {"step": ("flowkv_transfer_tables per step (device-resident block tables, no plan); pools resident in HBM"
                                 if args.device_tables else
                                 "flowkv_plan (pool->pool schedule only) + flowkv_transfer + flowkv_plan_destroy per step; pools resident in HBM"),
                        "dst": ("the NEXT rank's dst pool, mapped through CUDA IPC (one-sided peer put)" if args.peer
                                else "this rank's own dst pool"),
                        "launch": {k: stats[k] for k in ("grid", "threads", "group_threads", "tile_bytes", "variant",
                                                         "vec_bytes", "cache_hint", "tile_order", "stages")}},
                "clocks": m["clocks"],
                "per_rank": per_rank,
                "gpu_launches": m["launches"],
                "launches_per_batch": m["launches"] / K, "cuda_api_calls_per_batch": m["api_calls"] / K,
                "launches_per_request": m["launches"] / K / max(len(w.requests), 1),
                # throughput view: steps are pipelined (planning batch k+1 overlaps the kernel of batch k)
                "pipelined_step_ms_per_request": t_ms / K / max(len(w.requests), 1),
                # latency view: one synchronous request at a time, host wall clock, flowkv_plan call -> stream drained
                "latency_ms_call_to_done": m["latency_ms_call_to_done"],
                "latency_ms_call_to_done_min": m["latency_ms_call_to_done_min"],
                "latency_ms_call_to_done_per_request": m["latency_ms_call_to_done"] / max(len(w.requests), 1),
                "hbm_GBps": 2 * value, "pct_of_8TBps_nominal": 100 * 2 * value / world / 8000.0,
                "roofline": roofline_of(m, payload, wkey, stats, K, args.device_tables, po=args.config in ("cfg2sep", "cfg2mig")),
                "host": host_info(local),
            }

        # ---- end to end through host memory: pool -> pinned host (flowkv_pack) -> pool (flowkv_unpack) -------------
        if not args.no_e2e and payload > (24 << 30):
            # the route needs a pinned host buffer of the whole payload; beyond 24 GiB that is the host's RAM, not the path
            if rank == 0:
                line["e2e"] = {"skipped": "payload of %.1f GiB: pinned host staging of that size is not attempted" % (payload / 2 ** 30)}
        elif not args.no_e2e:
            nbytes = payload
            host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
            Ke = max(2, min(args.e2e_steps, K))
            scratch, scratch_bytes = None, 0
            if not (args.e2e_serial or args.e2e_direct):
                p0 = F.flowkv_plan(dp.src, dp.dst, dp.requests, F.FLOWKV_PLAN_NO_TRANSFER, tuning, s)
                scratch_bytes = F.flowkv_via_host_scratch_bytes(p0, args.e2e_chunks)
                p0.destroy()
                scratch = P.alloc_bytes(scratch_bytes, device=f"cuda:{local}")

            def e2e_step():
                plan = F.flowkv_plan(dp.src, dp.dst, dp.batch, F.FLOWKV_PLAN_NO_TRANSFER, tuning, s)
                if args.e2e_serial:
                    F.flowkv_pack(plan, host.data_ptr(), nbytes, s)      # device -> pinned host, one kernel
                    F.flowkv_unpack(plan, host.data_ptr(), nbytes, s)    # pinned host -> device, one kernel
                else:                                                    # same result, both PCIe directions overlapped
                    F.flowkv_transfer_via_host(plan, host.data_ptr(), nbytes, args.e2e_chunks, args.e2e_ctas, s,
                                               scratch.data_ptr() if scratch is not None else 0, scratch_bytes)
                plan.destroy()
            e2e_step()
            barrier()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(stream)
            for _ in range(Ke):
                e2e_step()
            b.record(stream)
            barrier()
            te = a.elapsed_time(b)
            te = shard.max_over_ranks(te, device=reduce_dev)
            # latency view of the same route: one synchronous request at a time, host wall clock, plan call -> drained
            e2e_lat = []
            for _ in range(5):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                e2e_step()
                torch.cuda.synchronize()
                e2e_lat.append((time.perf_counter() - t0) * 1e3)
            # link references: one contiguous copy-engine D2H / H2D of the same bytes, alone and both at once
            pb = min(nbytes, 2 << 30)                             # link probes: at most 2 GiB each way
            dev_flat = dp.dst_buf[:pb] if dp.dst_buf.numel() >= pb else P.alloc_bytes(pb)
            dev_flat2 = dp.src_buf[:pb]                           # read-only leg of the duplex probe
            host_p = host[:pb]
            host2 = torch.empty(pb, dtype=torch.uint8, pin_memory=True)
            a.record(stream); host_p.copy_(dev_flat, non_blocking=True); b.record(stream); torch.cuda.synchronize()
            d2h = pb / (a.elapsed_time(b) * 1e-3) / 1e9
            a.record(stream); dev_flat.copy_(host_p, non_blocking=True); b.record(stream); torch.cuda.synchronize()
            h2d = pb / (a.elapsed_time(b) * 1e-3) / 1e9
            side = torch.cuda.Stream()
            best = None
            for _ in range(3):                                    # D2H on the side stream + H2D on this one, together
                torch.cuda.synchronize()
                a.record(stream)
                side.wait_stream(stream)
                with torch.cuda.stream(side):
                    host2.copy_(dev_flat2, non_blocking=True)
                dev_flat.copy_(host_p, non_blocking=True)
                stream.wait_stream(side)
                b.record(stream)
                torch.cuda.synchronize()
                best = a.elapsed_time(b) if best is None else min(best, a.elapsed_time(b))
            duplex = pb / (best * 1e-3) / 1e9
            # ... and what the route must be: a CHUNKED duplex pipeline (chunk c returns once it has landed), copy
            # engines only, same chunk count as the route — the bound e2e.value is read against
            planes_ = 2 * w.shape.num_layers                     # the library's default rule: equal chunks, count nearest sqrt(payload / 400 KB)
            tgt_ = min(64.0, max(4.0, float(np.sqrt(nbytes / 400e3))))
            n_ch = args.e2e_chunks or min((d for d in range(min(planes_, 4), min(planes_, 64) + 1) if planes_ % d == 0),
                                          key=lambda d: abs(np.log(d / tgt_)))
            wbp = pb // n_ch
            side2 = torch.cuda.Stream()
            bestp = None
            for _ in range(3):
                torch.cuda.synchronize()
                a.record(stream)
                side.wait_stream(stream); side2.wait_stream(stream)
                for c in range(n_ch):
                    sl = slice(c * wbp, pb if c == n_ch - 1 else (c + 1) * wbp)
                    landed = torch.cuda.Event()
                    with torch.cuda.stream(side):
                        host_p[sl].copy_(dev_flat2[sl], non_blocking=True)
                        landed.record(side)
                    side2.wait_event(landed)
                    with torch.cuda.stream(side2):
                        dev_flat[sl].copy_(host_p[sl], non_blocking=True)
                stream.wait_stream(side); stream.wait_stream(side2)
                b.record(stream)
                torch.cuda.synchronize()
                bestp = a.elapsed_time(b) if bestp is None else min(bestp, a.elapsed_time(b))
            chunked = pb / (bestp * 1e-3) / 1e9
            if rank == 0:
                e2e_val = world * Ke * payload / (te * 1e-3) / 1e9
                line["e2e"] = {"value": e2e_val, "unit": UNIT,
                               "h2d_bytes_per_step": nbytes + stats["plan_device_bytes"], "d2h_bytes_per_step": nbytes,
                               "steps": Ke, "ms_per_step": te / Ke,
                               "latency_ms_call_to_done": float(np.median(e2e_lat)),
                               "path": ("flowkv_plan (host tables) + flowkv_pack to pinned host + flowkv_unpack from pinned host"
                                        if args.e2e_serial else
                                        "flowkv_plan (host tables) + flowkv_transfer_via_host, direct mode: pack kernels store to "
                                        "pinned host and unpack kernels load from it, pipelined over layer chunks on two streams"
                                        if args.e2e_direct else
                                        "flowkv_plan (host tables) + flowkv_transfer_via_host, copy-engine mode: per layer chunk "
                                        "flowkv_pack_window into device scratch, D2H to pinned host, H2D back, flowkv_unpack_window; "
                                        "four queues (pack kernels, D2H engine, H2D engine, unpack kernels), both PCIe directions busy"),
                               "device_scratch_bytes": scratch_bytes,
                               "link_memcpy_d2h_GBps": d2h, "link_memcpy_h2d_GBps": h2d,
                               "link_memcpy_duplex_GBps_each_way": duplex,
                               "link_chunked_duplex_pipeline_GBps_each_way": chunked,
                               "frac_of_one_way_link": e2e_val / world / min(d2h, h2d),
                               "frac_of_duplex_bound": e2e_val / world / duplex,
                               "frac_of_chunked_pipeline_bound": e2e_val / world / chunked}
            del host, host2, host_p

        # ---- comparison baselines on the same pools (outside the timed region) ---------------------------------
        if rank == 0 and not args.no_baselines and not args.peer:
            extra = {}
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            if stats["mode_transfer"] in (1, 3) and w.src.block_size == w.dst.block_size:
                for name, fn in (("blockwise_memcpy", lambda: F.flowkv_baseline_blockwise(dp.src, dp.dst, dp.requests, s)),):
                    fn(); torch.cuda.synchronize()
                    t0 = time.perf_counter(); a.record(stream); calls = fn(); b.record(stream); torch.cuda.synchronize()
                    extra[name] = {"calls": calls, "device_ms": a.elapsed_time(b), "wall_ms": (time.perf_counter() - t0) * 1e3,
                                   "GBps": payload / (a.elapsed_time(b) * 1e-3) / 1e9}
                plan = F.flowkv_plan(dp.src, dp.dst, dp.requests, 0, tuning, s)
                F.flowkv_baseline_segmentwise(plan, s); torch.cuda.synchronize()
                t0 = time.perf_counter(); a.record(stream); calls = F.flowkv_baseline_segmentwise(plan, s); b.record(stream)
                torch.cuda.synchronize()
                extra["segmentwise_memcpy"] = {"calls": calls, "device_ms": a.elapsed_time(b),
                                               "wall_ms": (time.perf_counter() - t0) * 1e3,
                                               "GBps": payload / (a.elapsed_time(b) * 1e-3) / 1e9}
                plan.destroy()
            flat_a = dp.src_buf[:payload]
            flat_b = dp.dst_buf[:payload] if dp.dst_buf.numel() >= payload else P.alloc_bytes(payload)
            ts = []
            for _ in range(5):
                a.record(stream); flat_b.copy_(flat_a); b.record(stream); torch.cuda.synchronize(); ts.append(a.elapsed_time(b))
            extra["contiguous_copy"] = {"calls": 1, "device_ms": min(ts), "GBps": payload / (min(ts) * 1e-3) / 1e9}
            line["baselines"] = extra

        if rank == 0 and world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(w, dp.src_buf)
        return line

    line = primary()
    import gc
    gc.collect()
    torch.cuda.empty_cache()

    # ---- the batched config (BASELINE.json configs[2]) in the same line: north_star asks for >= 80 % of HBM peak on
    # "the Llama-3-8B 13k-token AND batched configs".  Same step, same timing rules, its own clock record.
    if args.config == "cfg2" and not args.no_secondary and not args.peer and not args.same_device:
        free_b, _ = torch.cuda.mem_get_info()
        w3, desc3 = build_workload("cfg3", free_b)
        dp3 = P.DevicePools(w3, device=f"cuda:{local}", sentinel_dst=False)
        K3 = max(20, min(K, args.secondary_steps))
        m3 = time_steps(F, w3, dp3.src, dp3.dst, dp3.batch, K3, 3, tuning, stream, barrier, local,
                        device_tables_of(w3, dp3.device) if args.device_tables else None, latency_reps=5)
        t3 = shard.max_over_ranks(m3["t_ms"], device=reduce_dev)
        if rank == 0:
            m3["t_ms"] = t3
            p3 = w3.payload_bytes
            line["secondary"] = {
                "workload": desc3, "name": w3.name, "requests": len(w3.requests), "tokens": w3.total_tokens,
                "payload_bytes": p3, "segments": m3["stats"]["n_segments"], "steps": K3,
                "mean_src_run_blocks": run_mean(w3, "src"), "mean_dst_run_blocks": run_mean(w3, "dst"),
                "value": world * K3 * p3 / (t3 * 1e-3) / 1e9, "unit": UNIT, "ms_per_step": t3 / K3,
                "kernel_ms_avg": m3["kern_ms"], "kernel_ms_min": m3["kern_min_ms"],
                "pct_of_8TBps_nominal": 100 * 2 * K3 * p3 / (t3 * 1e-3) / 8e12,
                "pct_of_8TBps_nominal_kernel_only": 100 * 2 * p3 / (m3["kern_ms"] * 1e-3) / 8e12,
                "roofline": roofline_of(m3, p3, w3.name + ("+tables" if args.device_tables else ""), m3["stats"], K3,
                                        args.device_tables),
                "clocks": m3["clocks"], "gpu_launches": m3["launches"], "launches_per_batch": m3["launches"] / K3,
                "cuda_api_calls_per_batch": m3["api_calls"] / K3,
                "latency_ms_call_to_done": m3["latency_ms_call_to_done"],
                "latency_ms_call_to_done_per_request": m3["latency_ms_call_to_done"] / max(len(w3.requests), 1)}
        del dp3

    # ---- every other config and mode, each under its own key with its own roofline, clocks and launch count, so that
    # the driver's line — not only builder-run files under profiles/ — carries them.  One GPU only; a failure in one
    # record is written into that record and never costs the line.
    if args.config == "cfg2" and world == 1 and not args.no_extras and not args.device_tables:
        gc.collect()
        torch.cuda.empty_cache()
        line["configs"] = extra_records(args, F, P, stream, barrier, local, tuning)

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def extra_records(args, F, P, stream, barrier, local, tuning) -> dict:
    """BASELINE.json configs[0], configs[3] (register path and TMA tensor path), configs[4] (a summary of the sweep with
    the same-size plain copy beside every point, plus the 32k-token pack / unpack through pinned host memory), the
    paper's Table 3 request lengths, and the non-default modes on configs[1]'s request: flat mode (both
    pools (B,L,2,H), Eq. 5), the table-driven kernel, per-layer src tensors, the Eq. 5 migration, and
    flowkv_transfer_static.  Same step, same timing rules as the primary record; pools of one record are freed before
    the next is built."""
    import gc
    import torch
    out = {}
    Kx = max(10, min(args.extra_steps, args.steps))

    def record(w, desc, m, K, device_tables=False, po=False, step=None):
        stats, p = m["stats"], w.payload_bytes
        wkey = w.name + ("+tables" if device_tables else "+bulk" if stats["variant"] == 2 and stats["mode_transfer"] == 2
                         else "+bulk (no ncu capture committed)" if stats["variant"] == 2 else "")
        return {"workload": desc, "name": w.name, "requests": len(w.requests), "tokens": w.total_tokens, "payload_bytes": p,
                "segments": stats["n_segments"], "steps": K, "ms_per_step": m["t_ms"] / K,
                "value": K * p / (m["t_ms"] * 1e-3) / 1e9, "unit": UNIT,
                "step": step or ("flowkv_transfer_tables per step" if device_tables else "flowkv_plan + flowkv_transfer + flowkv_plan_destroy per step"),
                "pct_of_8TBps_nominal": 100 * 2 * K * p / (m["t_ms"] * 1e-3) / 8e12,
                "pct_of_8TBps_nominal_kernel_only": 100 * 2 * p / (m["kern_ms"] * 1e-3) / 8e12,
                "roofline": roofline_of(m, p, wkey, stats, K, device_tables, po=po),
                "clocks": m["clocks"], "gpu_launches": m["launches"], "launches_per_batch": m["launches"] / K,
                "cuda_api_calls_per_batch": m["api_calls"] / K,
                "latency_ms_call_to_done": m.get("latency_ms_call_to_done"),
                "launch": {k: stats[k] for k in ("grid", "threads", "group_threads", "tile_bytes", "variant", "vec_bytes", "stages")}}

    def on_pools(cfg, variants, sep=False):
        """variants: (key, tuning, device_tables) measured one after the other on ONE pool set of workload `cfg`."""
        try:
            free_b, _ = torch.cuda.mem_get_info()
            w, desc = build_workload(cfg, free_b)
            dp = P.DevicePools(w, device=f"cuda:{local}", sentinel_dst=False, separate_src_layers=sep)
        except Exception as e:                                   # pragma: no cover
            for key, _, _ in variants:
                out[key] = {"error": repr(e)}
            return
        for key, tn, tables in variants:
            try:
                K = Kx if w.payload_bytes < (8 << 30) else max(5, Kx // 4)
                m = time_steps(F, w, dp.src, dp.dst, dp.batch, K, 3, tn, stream, barrier, local,
                               device_tables_of(w, dp.device) if tables else None, latency_reps=5)
                out[key] = record(w, desc, m, K, device_tables=tables, po=sep)
            except Exception as e:                               # pragma: no cover
                out[key] = {"error": repr(e)}
        if cfg == "cfg3":
            try:                                                 # the allocation-free entry point on the batched config
                out["cfg3_batched_static_no_alloc"] = static_record(w, desc, dp)
            except Exception as e:                               # pragma: no cover
                out["cfg3_batched_static_no_alloc"] = {"error": repr(e)}
        del dp
        gc.collect()
        torch.cuda.empty_cache()

    def static_record(w, desc, dp):
        """flowkv_plan_host + flowkv_transfer_static per step: no device allocation anywhere in the step."""
        s = stream.cuda_stream
        K = 5

        def step(a=None, b=None):
            plan = F.flowkv_plan_host(dp.src, dp.dst, dp.batch, F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, tuning)
            if a is not None:
                a.record(stream)
            F.flowkv_transfer_static(plan, s)
            if b is not None:
                b.record(stream)
            return plan
        stats = step().stats
        for _ in range(2):
            step()
        ka = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        kb = [torch.cuda.Event(enable_timing=True) for _ in range(K)]
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        clocks = ClockSampler(local)
        barrier()
        step()
        clocks.start()
        n0, c0 = F.flowkv_launch_count(), F.flowkv_api_call_count()
        e0.record(stream)
        for k in range(K):
            step(ka[k], kb[k])
        e1.record(stream)
        barrier()
        m = {"t_ms": e0.elapsed_time(e1), "kern_ms": float(np.mean([a.elapsed_time(b) for a, b in zip(ka, kb)])),
             "kern_min_ms": float(np.min([a.elapsed_time(b) for a, b in zip(ka, kb)])),
             "launches": F.flowkv_launch_count() - n0, "api_calls": F.flowkv_api_call_count() - c0,
             "clocks": clocks.stop(), "stats": stats}
        rec = record(w, desc, m, K, step="flowkv_plan_host + flowkv_transfer_static per step (schedule copy + kernel inside "
                                         "the per-kernel events; no device allocation)")
        rec["schedule_entries"] = stats["n_chunks_transfer"]
        return rec

    on_pools("cfg1", [("cfg1_tiny", tuning, False)])
    on_pools("cfg2", [("cfg2_13k_tables", tuning, True), ("cfg2_13k_bulk", dict(tuning or {}, variant="bulk"), False)])
    on_pools("cfg2bm", [("cfg2bm_flat", tuning, False), ("cfg2bm_flat_bulk", dict(tuning or {}, variant="bulk"), False)])
    on_pools("cfg2sep", [("cfg2sep_per_layer_src", tuning, False)], sep=True)
    on_pools("cfg2mig", [("cfg2mig_eq5_migration", tuning, False)], sep=True)
    on_pools("cfg3", [("cfg3_batched_tables", tuning, True)])
    on_pools("cfg4", [("cfg4_hetero_ldst", tuning, False), ("cfg4_hetero_tma", dict(tuning or {}, variant="bulk"), False),
                      ("cfg4_hetero_tables", tuning, True)])

    # configs[4]: sweep summary + pinned pack at 32k tokens; Table 3 lengths.  bench_sweep times the kernel alone (a
    # built plan, L2 flushed between repetitions where the payload could stay resident) and the same-size plain copy.
    import bench_sweep
    log = lambda row: print(json.dumps(row), file=sys.stderr, flush=True)
    for key, argv in (("cfg5_sweep", ["--tokens", "128,256,512,4096,32768,131072", "--runs", "1,0", "--reps", "20", "--no-baselines", "--out", ""]),
                      ("table3_lengths", ["--table3", "--reps", "20", "--no-baselines", "--out", ""])):
        try:
            clocks = ClockSampler(local)
            clocks.start()
            rows = bench_sweep.main(argv, emit=log)
            clk = clocks.stop()
            for r in rows:
                if "hbm_GBps" in r:
                    r["pct_of_8TBps_nominal"] = r["hbm_GBps"] / 80.0
            out[key] = {"rows": rows, "clocks": clk,
                        "timing": "kernel alone on a built plan, CUDA events, mean of 20; L2 flushed by a read pass between "
                                  "repetitions when 2 x payload < 256 MiB; plain_copy = one cudaMemcpyAsync D2D of the same bytes"}
        except Exception as e:                                   # pragma: no cover
            out[key] = {"error": repr(e)}
        gc.collect()
        torch.cuda.empty_cache()
    return out


def spawn_ranks(args) -> None:
    """`python bench.py --gpus N` with N > 1 and no launcher: start the N ranks here, one process per GPU, exactly as
    the driver does (`python -m torch.distributed.run --nnodes=1 --nproc-per-node N ...`), and become that launcher."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    os.execv(sys.executable, cmd)


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=500)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="cfg2", choices=["cfg1", "cfg2", "cfg2sep", "cfg2mig", "cfg2bm", "cfg2bm_ragged", "cfg3", "cfg4"])
    ap.add_argument("--tuning", default=None, help="JSON dict of flowkv_tuning fields")
    ap.add_argument("--device-tables", action="store_true",
                    help="time flowkv_transfer_tables (block tables resident on the device, no plan) instead of plan+transfer")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-serial", action="store_true", help="pack then unpack on one stream instead of the pipeline")
    ap.add_argument("--e2e-direct", action="store_true",
                    help="pipeline with SM loads/stores over PCIe (no device scratch) instead of the copy engines")
    ap.add_argument("--e2e-chunks", type=int, default=0)
    ap.add_argument("--e2e-ctas", type=int, default=0)
    ap.add_argument("--no-baselines", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep", action="store_true", help="run the configs[4] sweep instead (see bench_sweep.py)")
    ap.add_argument("--latency-reps", type=int, default=20, help="synchronous requests behind latency_ms_call_to_done")
    ap.add_argument("--no-secondary", action="store_true", help="skip the configs[2] (batched) measurement that the "
                    "default cfg2 run appends under `secondary`")
    ap.add_argument("--secondary-steps", type=int, default=20)
    ap.add_argument("--no-extras", action="store_true", help="skip the records of the other configs and modes that the "
                    "default cfg2 run appends under `configs`")
    ap.add_argument("--extra-steps", type=int, default=20)
    ap.add_argument("--peer", action="store_true", help="rank r stores into rank (r+1)%%N's dst pool through CUDA IPC "
                    "(one-sided peer put; needs >= 2 ranks)")
    ap.add_argument("--same-device", action="store_true", help="all ranks on cuda:0 with a gloo control plane (a "
                    "functional check of the multi-rank path on a one-GPU box; not a scaling number)")
    args = ap.parse_args()
    if args.config in ("cfg2sep", "cfg2mig"):     # the src pool is 32 separate tensors: no whole-pool probes, link legs or memcpy baselines
        args.no_e2e = args.no_baselines = True
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        spawn_ranks(args)          # does not return
    if args.sweep:
        import bench_sweep
        bench_sweep.main([])
        return
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
