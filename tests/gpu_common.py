"""Shared by the `-m gpu` parity tests: run the CUDA path through the C-ABI binding, run the oracle on
the same seeded inputs, compare the ENTIRE dst pool byte for byte (sentinel-filled, so untouched
bytes are checked too)."""
from __future__ import annotations

import numpy as np
import torch

from oracle import oracle as O
from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import pools as P
from paper_2504_03775_b200 import synth


def geom(spec: synth.PoolSpec, shape: synth.Shape, num_layers=None) -> O.PoolGeom:
    L = shape.num_layers if num_layers is None else num_layers
    return getattr(O.PoolGeom, spec.layout)(L, shape.num_kv_heads, shape.head_dim, shape.elem_bytes,
                                            spec.num_blocks, spec.block_size)


def oracle_transfer(w: synth.Workload, src_np: np.ndarray) -> np.ndarray:
    gs, gd = geom(w.src, w.shape), geom(w.dst, w.shape)
    exp = np.full(w.dst.bytes(w.shape), P.SENTINEL_BYTE, np.uint8)
    for r in w.requests:
        O.transfer(src_np, gs, exp, gd, r.src_blocks, r.dst_blocks, r.num_tokens)
    return exp


def oracle_pack(w: synth.Workload, src_np: np.ndarray) -> np.ndarray:
    gs = geom(w.src, w.shape)
    out = np.full(w.payload_bytes, P.SENTINEL_BYTE, np.uint8)
    off = 0
    for r in w.requests:
        O.pack(src_np, gs, r.src_blocks, r.num_tokens, out, off)
        off += r.num_tokens
    return out


def oracle_unpack(w: synth.Workload, staging_np: np.ndarray) -> np.ndarray:
    gd = geom(w.dst, w.shape)
    exp = np.full(w.dst.bytes(w.shape), P.SENTINEL_BYTE, np.uint8)
    off = 0
    for r in w.requests:
        O.unpack(staging_np, off, exp, gd, r.dst_blocks, r.num_tokens)
        off += r.num_tokens
    return exp


def assert_same(got: np.ndarray, exp: np.ndarray, what: str) -> None:
    if not np.array_equal(got, exp):
        bad = np.nonzero(got != exp)[0]
        raise AssertionError(f"{what}: {bad.size} of {exp.size} bytes differ; first at byte {int(bad[0])} "
                             f"(got {int(got[bad[0]])}, expected {int(exp[bad[0]])})")


def run_transfer_and_check(w: synth.Workload, tuning=None, fill=None, flags=0):
    """GPU transfer vs oracle on the whole dst pool; also checks src is unchanged and launches == 1."""
    dp = P.DevicePools(w, fill=fill)
    src_before = P.to_numpy(dp.src_buf)
    st = torch.cuda.current_stream()
    plan = dp.plan(flags | F.FLOWKV_CHECK_DST_ALIAS, tuning, st.cuda_stream)
    n0 = F.flowkv_launch_count()
    plan.transfer(st.cuda_stream)
    n1 = F.flowkv_launch_count()
    torch.cuda.synchronize()
    assert n1 - n0 == (1 if w.total_tokens else 0), "exactly one kernel launch per transfer batch"
    got = P.to_numpy(dp.dst_buf)
    exp = oracle_transfer(w, src_before)
    assert_same(got, exp, f"{w.name} transfer {tuning}")
    assert_same(P.to_numpy(dp.src_buf), src_before, "src pool must not change")
    return dp, plan, exp


def window_of(full_wire: np.ndarray, w: synth.Workload, l0: int, l1: int) -> np.ndarray:
    """Layer window [l0,l1) of the wire format, by its definition: per request, the slab of planes
    [2*l0, 2*l1) of that request's region ([request][layer][K|V][token][head][dim]), requests concatenated."""
    tokb = w.shape.num_kv_heads * w.shape.head_dim * w.shape.elem_bytes
    bpt = w.shape.bytes_per_token
    parts, off = [], 0
    for r in w.requests:
        base = off * bpt
        parts.append(full_wire[base + 2 * l0 * r.num_tokens * tokb: base + 2 * l1 * r.num_tokens * tokb])
        off += r.num_tokens
    return np.concatenate(parts) if parts else np.zeros(0, np.uint8)


def oracle_pack_window(w: synth.Workload, src_np: np.ndarray, l0: int, l1: int) -> np.ndarray:
    """The oracle's layer window [l0,l1) of the whole batch (oracle/flowkv_oracle.c okv_pack_window)."""
    gs = geom(w.src, w.shape)
    tokb = w.shape.num_kv_heads * w.shape.head_dim * w.shape.elem_bytes
    out = np.full(w.total_tokens * 2 * (l1 - l0) * tokb, P.SENTINEL_BYTE, np.uint8)
    off = 0
    for r in w.requests:
        O.pack_window(src_np, gs, r.src_blocks, r.num_tokens, out, off, l0, l1)
        off += r.num_tokens
    return out


def oracle_pack_planes(w: synth.Workload, src_np: np.ndarray, p0: int, p1: int) -> np.ndarray:
    """The oracle's plane window [p0,p1) of the whole batch (oracle/flowkv_oracle.c okv_pack_planes, reading A21)."""
    gs = geom(w.src, w.shape)
    tokb = w.shape.num_kv_heads * w.shape.head_dim * w.shape.elem_bytes
    out = np.full(w.total_tokens * (p1 - p0) * tokb, P.SENTINEL_BYTE, np.uint8)
    off = 0
    for r in w.requests:
        O.pack_planes(src_np, gs, r.src_blocks, r.num_tokens, out, off, p0, p1)
        off += r.num_tokens
    return out
