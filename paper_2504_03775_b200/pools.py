"""Device memory for synthetic pools: torch is used ONLY to allocate, fill and read back buffers.

Nothing here copies KV data between pools — that is the C/CUDA library's job (flowkv.py).
Shared by the GPU tests and bench.py.  Imports neither ``oracle`` nor any oracle output.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np
import torch

from . import flowkv as F
from . import synth

SENTINEL_BYTE = 0xA5


def describe(spec: synth.PoolSpec, shape: synth.Shape, base_ptr: int) -> F.flowkv_pool:
    return F.make_pool(base_ptr, shape.num_layers, shape.num_kv_heads, shape.head_dim, shape.elem_bytes,
                       spec.num_blocks, spec.block_size, spec.layout)


def alloc_bytes(nbytes: int, device="cuda:0") -> torch.Tensor:
    """Flat uint8 buffer (torch's allocator returns >= 256-byte aligned pointers)."""
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def fill_values(buf: torch.Tensor, dist: str, dtype: str, seed: int, chunk_bytes: int = 1 << 30) -> None:
    """Seeded values with the distribution BASELINE.json names (irrelevant to a copy, kept anyway):
    'normal' N(0,1), 'uniform' U[-1,1], 'bits' uniformly random 16-bit patterns (NaNs, Infs, -0,
    denormals included).  Filled in place, chunk by chunk, so no pool-sized temporary exists."""
    gen = torch.Generator(device=buf.device)
    gen.manual_seed(seed)
    tdt = {"bf16": torch.bfloat16, "fp16": torch.float16, "fp32": torch.float32, "fp8": None}[dtype]
    if tdt is None:                   # fp8: every byte is a valid code; values are irrelevant to a copy
        dist = "bits"
    n = buf.numel()
    for off in range(0, n, chunk_bytes):
        part = buf[off:min(off + chunk_bytes, n)]
        if dist == "bits":
            part.view(torch.int16).random_(-32768, 32768, generator=gen)
        elif dist == "normal":
            part.view(tdt).normal_(0.0, 1.0, generator=gen)
        elif dist == "uniform":
            part.view(tdt).uniform_(-1.0, 1.0, generator=gen)
        else:
            raise ValueError(dist)


def fill_sentinel(buf: torch.Tensor) -> None:
    buf.fill_(SENTINEL_BYTE)


def requests_of(w: synth.Workload, src: bool = True, dst: bool = True) -> Sequence[F.Request]:
    return [F.Request(r.num_tokens, r.src_blocks if src else None, r.dst_blocks if dst else None) for r in w.requests]


class DevicePools:
    """src + dst pools of a workload on one device, described for the library."""

    def __init__(self, w: synth.Workload, device="cuda:0", fill: Optional[str] = None, sentinel_dst: bool = True,
                 separate_src_layers: bool = False):
        """``separate_src_layers``: the src pool (LKBTHD) is allocated as one tensor PER LAYER — the cache the paper
        starts from — and described through ``flowkv_pool.plane_offsets``; ``src_layers`` holds the tensors and
        ``src_buf`` is layer 0's."""
        self.w = w
        self.device = torch.device(device)
        self.dst_buf = alloc_bytes(w.dst.bytes(w.shape), device)
        if separate_src_layers:
            assert w.src.layout == "lkbthd", "separate layer tensors are (2,B,H) each"
            L = w.shape.num_layers
            per = w.src.bytes(w.shape) // L
            self.src_layers = [alloc_bytes(per, device) for _ in range(L)]
            for l, t in enumerate(self.src_layers):
                fill_values(t, fill or w.value_dist, w.shape.dtype, w.seed + l)
            base = min(t.data_ptr() for t in self.src_layers)
            self.src_buf = self.src_layers[0]
            self.src = F.make_pool(base, L, w.shape.num_kv_heads, w.shape.head_dim, w.shape.elem_bytes, w.src.num_blocks,
                                   w.src.block_size, "lkbthd", layer_offsets=[t.data_ptr() - base for t in self.src_layers])
        else:
            self.src_buf = alloc_bytes(w.src.bytes(w.shape), device)
            fill_values(self.src_buf, fill or w.value_dist, w.shape.dtype, w.seed)
            self.src = describe(w.src, w.shape, self.src_buf.data_ptr())
        if sentinel_dst:
            fill_sentinel(self.dst_buf)
        self.dst = describe(w.dst, w.shape, self.dst_buf.data_ptr())
        self.requests = requests_of(w)
        self.batch = F.RequestBatch(self.requests)      # marshalled once; what bench.py's timed step passes

    def plan(self, flags: int = 0, tuning=None, stream: int = 0) -> F.Plan:
        return F.flowkv_plan(self.src, self.dst, self.requests, flags, tuning, stream)


def to_numpy(buf: torch.Tensor) -> np.ndarray:
    return buf.cpu().numpy()


def pool_from_tensors(layers=None, k_layers=None, v_layers=None) -> F.flowkv_pool:
    """Describe a cache that lives in per-layer torch tensors — the layout engines usually have and the one the paper
    starts from — without copying anything.  Either

      ``layers``               one tensor per layer shaped [2, num_blocks, block_size, num_kv_heads, head_dim]  (K|V stacked), or
      ``k_layers, v_layers``   one K and one V tensor per layer, each [num_blocks, block_size, num_kv_heads, head_dim].

    All tensors: same shape, dtype and CUDA device, contiguous.  The descriptor's base is the lowest data pointer and
    ``plane_offsets`` the distances of the 2L planes from it; the caller keeps the tensors alive."""
    if layers is not None:
        assert k_layers is None and v_layers is None
        ts = list(layers)
        assert ts and all(t.dim() == 5 and t.shape[0] == 2 for t in ts), "layers: [2, NB, BS, H, D] each"
        planes = [t[c] for t in ts for c in (0, 1)]
    else:
        assert k_layers is not None and v_layers is not None and len(k_layers) == len(v_layers) > 0
        planes = [t for kv in zip(k_layers, v_layers) for t in kv]
    p0 = planes[0]
    assert all(t.shape == p0.shape and t.dtype == p0.dtype and t.device == p0.device and t.is_contiguous() for t in planes), \
        "every plane: same shape, dtype, device; contiguous"
    nb, bs, h, d = (int(x) for x in p0.shape)
    base = min(t.data_ptr() for t in planes)
    return F.make_pool(base, len(planes) // 2, h, d, p0.element_size(), nb, bs, "lkbthd",
                       plane_offsets=[t.data_ptr() - base for t in planes])
