"""ctypes binding of ``libflowkv.so`` — same names as include/flowkv.h, argument marshalling only.

Every step of the path (planning, scheduling, the copy) runs inside the C/CUDA library; this module
turns Python objects into the structs of the header and raises :class:`FlowKVError` on a non-zero
status.  There is no fallback of any kind: if the library is missing, importing this module fails.

Pointers are plain integers (``tensor.data_ptr()``, ``stream.cuda_stream``); torch is not imported
here.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass
from typing import List, Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libflowkv.so")

# ---- enums / flags of the header -------------------------------------------------------------
FLOWKV_OK = 0
(FLOWKV_ERR_INVALID_ARG, FLOWKV_ERR_BLOCK_OOB, FLOWKV_ERR_TABLE_LEN, FLOWKV_ERR_DST_ALIAS, FLOWKV_ERR_ALIGN,
 FLOWKV_ERR_SHAPE_MISMATCH, FLOWKV_ERR_UNSUPPORTED, FLOWKV_ERR_STAGING_TOO_SMALL, FLOWKV_ERR_NOMEM,
 FLOWKV_ERR_CUDA) = range(1, 11)
FLOWKV_LAYOUT_LKBTHD, FLOWKV_LAYOUT_BLKHTD, FLOWKV_LAYOUT_STRIDED, FLOWKV_LAYOUT_BLKTHD = 0, 1, 2, 3
FLOWKV_CHECK_DST_ALIAS, FLOWKV_PLAN_NO_TRANSFER, FLOWKV_PLAN_NO_PACK, FLOWKV_PLAN_NO_UNPACK = 1, 2, 4, 8
FLOWKV_VARIANT_AUTO, FLOWKV_VARIANT_LDST, FLOWKV_VARIANT_BULK = 0, 1, 2
LAYOUTS = {"lkbthd": FLOWKV_LAYOUT_LKBTHD, "blkhtd": FLOWKV_LAYOUT_BLKHTD, "strided": FLOWKV_LAYOUT_STRIDED,
           "blkthd": FLOWKV_LAYOUT_BLKTHD}

FLOWKV_VERSION = 4          # include/flowkv.h; the struct layouts below are this version's
FLOWKV_STATIC_SCHEDULE_ENTRIES = 32768      # include/flowkv.h: capacity of flowkv_transfer_static's fixed device array

EXPORTS = ["flowkv_version", "flowkv_pool_strides", "flowkv_plan", "flowkv_plan_host", "flowkv_plan_info", "flowkv_transfer",
           "flowkv_pack", "flowkv_unpack", "flowkv_plan_destroy", "flowkv_status_string", "flowkv_last_error",
           "flowkv_launch_count", "flowkv_api_call_count", "flowkv_baseline_blockwise", "flowkv_baseline_segmentwise",
           "flowkv_transfer_layers", "flowkv_pack_layers", "flowkv_unpack_layers", "flowkv_transfer_via_host",
           "flowkv_window_bytes", "flowkv_pack_window", "flowkv_unpack_window", "flowkv_via_host_scratch_bytes",
           "flowkv_transfer_tables", "flowkv_transfer_tables_layers", "flowkv_pack_tables", "flowkv_unpack_tables",
           "flowkv_alloc_create", "flowkv_alloc_allocate", "flowkv_alloc_free", "flowkv_alloc_stats",
           "flowkv_alloc_destroy", "flowkv_transfer_static", "flowkv_trim", "flowkv_cache_counts"]


class flowkv_pool(C.Structure):
    _fields_ = [("base", C.c_void_p), ("num_layers", C.c_uint32), ("num_kv_heads", C.c_uint32),
                ("head_dim", C.c_uint32), ("elem_bytes", C.c_uint32), ("num_blocks", C.c_uint32),
                ("block_size", C.c_uint32), ("layout", C.c_uint32), ("_reserved", C.c_uint32),
                ("stride_bytes", C.c_int64 * 5), ("plane_offsets", C.c_void_p)]


class flowkv_request(C.Structure):
    _fields_ = [("num_tokens", C.c_uint32), ("n_src_blocks", C.c_uint32), ("src_blocks", C.c_void_p),
                ("dst_blocks", C.c_void_p), ("n_dst_blocks", C.c_uint32), ("_reserved", C.c_uint32)]


class flowkv_segment(C.Structure):
    _fields_ = [("request", C.c_uint32), ("first_token", C.c_uint32), ("n_tokens", C.c_uint32),
                ("src_block", C.c_uint32), ("src_tok_off", C.c_uint32), ("dst_block", C.c_uint32),
                ("dst_tok_off", C.c_uint32), ("_reserved", C.c_uint32), ("staging_tok_off", C.c_uint64)]


class flowkv_tuning(C.Structure):
    _fields_ = [("tile_bytes", C.c_uint32), ("ctas_per_sm", C.c_uint32), ("max_sms", C.c_uint32),
                ("threads", C.c_uint32), ("group_threads", C.c_uint32), ("variant", C.c_uint32),
                ("tile_order", C.c_uint32), ("cache_hint", C.c_uint32), ("stages", C.c_uint32),
                ("plan_in_params", C.c_uint32), ("_reserved", C.c_uint32 * 2)]


class flowkv_plan_stats(C.Structure):
    _fields_ = [("n_requests", C.c_uint64), ("n_segments", C.c_uint64), ("total_tokens", C.c_uint64),
                ("payload_bytes", C.c_uint64), ("staging_bytes", C.c_uint64), ("n_chunks_transfer", C.c_uint64),
                ("n_chunks_pack", C.c_uint64), ("n_chunks_unpack", C.c_uint64), ("plan_device_bytes", C.c_uint64),
                ("n_planes", C.c_uint32), ("mode_transfer", C.c_uint32), ("mode_pack", C.c_uint32),
                ("mode_unpack", C.c_uint32), ("grid", C.c_uint32), ("threads", C.c_uint32),
                ("group_threads", C.c_uint32), ("tile_bytes", C.c_uint32), ("variant", C.c_uint32),
                ("vec_bytes", C.c_uint32), ("tile_order", C.c_uint32), ("cache_hint", C.c_uint32),
                ("stages", C.c_uint32), ("smem_bytes", C.c_uint32), ("num_sms", C.c_uint32), ("n_flat_chunks", C.c_uint32)]

    def as_dict(self) -> dict:
        return {n: int(getattr(self, n)) for n, _ in self._fields_ if not n.startswith("_")}


class FlowKVError(RuntimeError):
    def __init__(self, status: int, name: str, text: str):
        super().__init__(f"{name}: {text}")
        self.status = status
        self.name = name


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2504_03775_b200.build` "
                          "(there is no fallback implementation)")
    lib = C.CDLL(LIB_PATH)
    P = C.POINTER
    lib.flowkv_pool_strides.argtypes = [P(flowkv_pool)]
    lib.flowkv_plan.argtypes = [P(flowkv_pool), P(flowkv_pool), P(flowkv_request), C.c_uint32, C.c_uint32,
                                P(flowkv_tuning), C.c_void_p, P(C.c_void_p)]
    lib.flowkv_plan_host.argtypes = [P(flowkv_pool), P(flowkv_pool), P(flowkv_request), C.c_uint32, C.c_uint32,
                                     P(flowkv_tuning), P(C.c_void_p)]
    lib.flowkv_plan_info.argtypes = [C.c_void_p, P(flowkv_plan_stats), P(P(flowkv_segment))]
    lib.flowkv_transfer.argtypes = [C.c_void_p, C.c_void_p]
    lib.flowkv_transfer_static.argtypes = [C.c_void_p, C.c_void_p]
    lib.flowkv_trim.argtypes = []
    lib.flowkv_cache_counts.argtypes = [P(C.c_uint32), P(C.c_uint32)]
    lib.flowkv_pack.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
    lib.flowkv_unpack.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_void_p]
    lib.flowkv_transfer_layers.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, C.c_void_p]
    lib.flowkv_pack_layers.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
    lib.flowkv_unpack_layers.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
    lib.flowkv_transfer_via_host.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p,
                                             C.c_uint64, C.c_void_p]
    lib.flowkv_window_bytes.argtypes = [C.c_void_p, C.c_uint32, C.c_uint32, P(C.c_uint64)]
    lib.flowkv_pack_window.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
    lib.flowkv_unpack_window.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32, C.c_uint32, C.c_void_p]
    lib.flowkv_via_host_scratch_bytes.argtypes = [C.c_void_p, C.c_uint32, P(C.c_uint64)]
    lib.flowkv_transfer_tables.argtypes = [P(flowkv_pool), P(flowkv_pool), C.c_void_p, C.c_void_p, C.c_void_p, C.c_uint32,
                                           C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p, P(flowkv_tuning), C.c_void_p]
    lib.flowkv_transfer_tables_layers.argtypes = [P(flowkv_pool), P(flowkv_pool), C.c_void_p, C.c_void_p, C.c_void_p,
                                                  C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32, C.c_uint32,
                                                  C.c_void_p, P(flowkv_tuning), C.c_void_p]
    for fn in (lib.flowkv_pack_tables, lib.flowkv_unpack_tables):
        fn.argtypes = [P(flowkv_pool), C.c_void_p, C.c_void_p, C.c_uint32, C.c_uint32, C.c_uint32, C.c_void_p, C.c_uint64,
                       C.c_uint32, C.c_uint32, C.c_void_p, P(flowkv_tuning), C.c_void_p]
    lib.flowkv_plan_destroy.argtypes = [C.c_void_p]
    lib.flowkv_plan_destroy.restype = None
    lib.flowkv_status_string.argtypes = [C.c_int]
    lib.flowkv_status_string.restype = C.c_char_p
    try:                                             # a stale libflowkv.so next to a newer binding: fail loudly, never guess
        lib.flowkv_version.argtypes = []
        lib.flowkv_version.restype = C.c_uint32
        have = lib.flowkv_version()
    except AttributeError:
        have = "< 4"
    if have != FLOWKV_VERSION:
        raise ImportError(f"{LIB_PATH} is FLOWKV_VERSION {have}, this binding needs {FLOWKV_VERSION} (struct layouts "
                          "differ): rebuild it with `python -m paper_2504_03775_b200.build --force`")
    lib.flowkv_last_error.argtypes = []
    lib.flowkv_last_error.restype = C.c_char_p
    lib.flowkv_launch_count.argtypes = []
    lib.flowkv_launch_count.restype = C.c_uint64
    lib.flowkv_api_call_count.argtypes = []
    lib.flowkv_api_call_count.restype = C.c_uint64
    lib.flowkv_baseline_blockwise.argtypes = [P(flowkv_pool), P(flowkv_pool), P(flowkv_request), C.c_uint32,
                                              C.c_void_p, P(C.c_uint64)]
    lib.flowkv_baseline_segmentwise.argtypes = [C.c_void_p, C.c_void_p, P(C.c_uint64)]
    lib.flowkv_alloc_create.argtypes = [C.c_uint32, P(C.c_void_p)]
    lib.flowkv_alloc_allocate.argtypes = [C.c_void_p, C.c_uint32, C.c_void_p, P(C.c_uint32)]
    lib.flowkv_alloc_free.argtypes = [C.c_void_p, C.c_void_p, C.c_uint32]
    lib.flowkv_alloc_stats.argtypes = [C.c_void_p, P(C.c_uint32), P(C.c_uint32), P(C.c_uint32)]
    lib.flowkv_alloc_destroy.argtypes = [C.c_void_p]
    lib.flowkv_alloc_destroy.restype = None
    for n in EXPORTS:
        if n not in ("flowkv_version", "flowkv_plan_destroy", "flowkv_status_string", "flowkv_last_error", "flowkv_launch_count",
                     "flowkv_api_call_count",
                     "flowkv_alloc_destroy"):
            getattr(lib, n).restype = C.c_int
    return lib


_lib = _load()


def _check(status: int) -> None:
    if status != FLOWKV_OK:
        raise FlowKVError(status, _lib.flowkv_status_string(status).decode(), _lib.flowkv_last_error().decode())


def flowkv_status_string(status: int) -> str:
    return _lib.flowkv_status_string(status).decode()


def flowkv_last_error() -> str:
    return _lib.flowkv_last_error().decode()


def flowkv_launch_count() -> int:
    return int(_lib.flowkv_launch_count())


def flowkv_api_call_count() -> int:
    return int(_lib.flowkv_api_call_count())


# ---- marshalling helpers ----------------------------------------------------------------------
def make_pool(base: int, num_layers: int, num_kv_heads: int, head_dim: int, elem_bytes: int, num_blocks: int,
              block_size: int, layout="lkbthd", strides: Optional[Sequence[int]] = None,
              layer_offsets: Optional[Sequence[int]] = None, plane_offsets: Optional[Sequence[int]] = None) -> flowkv_pool:
    """Describe a pool.  ``strides`` (layer, kv, block, token, head; bytes) only for layout 'strided'.
    ``plane_offsets``: byte offset of every plane 2*layer + (0 K | 1 V) from ``base`` when the planes are separate
    allocations (reading A22); ``layer_offsets``: the special case of one tensor per layer with K and V stacked s_kv
    apart inside it.  The int64 array is kept alive by the returned object."""
    assert layer_offsets is None or plane_offsets is None
    p = flowkv_pool()
    p.base = base
    p.num_layers, p.num_kv_heads, p.head_dim, p.elem_bytes = num_layers, num_kv_heads, head_dim, elem_bytes
    p.num_blocks, p.block_size = num_blocks, block_size
    p.layout = LAYOUTS[layout] if isinstance(layout, str) else int(layout)
    if strides is not None:
        for i, s in enumerate(strides):
            p.stride_bytes[i] = int(s)
    if plane_offsets is not None:           # set before the stride check: layer / K|V strides are then ignored
        po = np.ascontiguousarray(np.asarray(plane_offsets, dtype=np.int64))
        assert po.shape == (2 * num_layers,), "one offset per plane"
        p._plane_offsets_keep = po
        p.plane_offsets = po.ctypes.data
    if layer_offsets is not None:
        assert len(layer_offsets) == num_layers, "one offset per layer"
        po = np.zeros(2 * num_layers, dtype=np.int64)
        p._plane_offsets_keep = po
        p.plane_offsets = po.ctypes.data
        flowkv_pool_strides(p)              # fills s_kv for the named layouts (the layer stride is already ignored)
        assert p.stride_bytes[1] > 0, "layer_offsets needs the K|V stride inside a layer"
        po[:] = [int(o) + c * p.stride_bytes[1] for o in layer_offsets for c in (0, 1)]
    flowkv_pool_strides(p)
    return p


def flowkv_pool_strides(pool: flowkv_pool) -> flowkv_pool:
    _check(_lib.flowkv_pool_strides(C.byref(pool)))
    return pool


def pool_bytes(pool: flowkv_pool) -> int:
    """Bytes from the base to one past the last addressable element."""
    s = pool.stride_bytes
    if pool.plane_offsets:
        po = getattr(pool, "_plane_offsets_keep")
        return int(po.max()) + ((pool.num_blocks - 1) * s[2] + (pool.block_size - 1) * s[3]
                                + (pool.num_kv_heads - 1) * s[4] + pool.head_dim * pool.elem_bytes)
    return ((pool.num_layers - 1) * s[0] + s[1] + (pool.num_blocks - 1) * s[2] + (pool.block_size - 1) * s[3]
            + (pool.num_kv_heads - 1) * s[4] + pool.head_dim * pool.elem_bytes)


@dataclass
class Request:
    num_tokens: int
    src_blocks: Optional[np.ndarray] = None
    dst_blocks: Optional[np.ndarray] = None


def _table(tab) -> np.ndarray:
    """int32 C-contiguous view/copy of a block table (no copy when it already is one)."""
    if type(tab) is np.ndarray and tab.dtype == np.int32 and tab.flags.c_contiguous:
        return tab
    return np.ascontiguousarray(np.asarray(tab, dtype=np.int32))


def _addr(a: np.ndarray) -> int:
    """Address of an array's first element (the ctypes buffer route is ~3x faster than ``a.ctypes.data``)."""
    try:
        return C.addressof(C.c_char.from_buffer(a))
    except (TypeError, ValueError):          # read-only arrays cannot export a writable buffer
        return a.ctypes.data


def _marshal_requests(requests: Sequence) -> tuple:
    """-> (flowkv_request array, n, arrays kept alive for the duration of the call)."""
    n = len(requests)
    arr = (flowkv_request * max(n, 1))()
    keep: List[np.ndarray] = []
    for i, r in enumerate(requests):
        q = arr[i]
        q.num_tokens = int(r.num_tokens)
        tab = getattr(r, "src_blocks", None)
        if tab is not None:
            a = _table(tab)
            keep.append(a)
            q.n_src_blocks = a.size
            if a.size:
                q.src_blocks = _addr(a)
        tab = getattr(r, "dst_blocks", None)
        if tab is not None:
            a = _table(tab)
            keep.append(a)
            q.n_dst_blocks = a.size
            if a.size:
                q.dst_blocks = _addr(a)
    return arr, n, keep


class RequestBatch:
    """A batch marshalled ONCE into the C array ``flowkv_plan`` takes (plus the int32 tables it points into, kept
    alive here).  Passing the same batch to several ``flowkv_plan*`` calls skips the per-call marshalling of the
    Python objects (~4 us per request) — what a C caller holding a ``flowkv_request[]`` does anyway.  The tables
    must not be modified or resized while the batch is in use."""

    def __init__(self, requests: Sequence):
        self.array, self.n, self._keep = _marshal_requests(requests)

    def __len__(self) -> int:
        return self.n


def _requests_arg(requests) -> tuple:
    if isinstance(requests, RequestBatch):
        return requests.array, requests.n, requests
    return _marshal_requests(requests)


class Plan:
    """Owner of a ``flowkv_plan_t*``; destroyed with the object (or by :meth:`destroy`)."""

    def __init__(self, handle: int):
        self._h = C.c_void_p(handle)

    @property
    def handle(self) -> C.c_void_p:
        if not self._h:
            raise ValueError("plan was destroyed")
        return self._h

    def info(self):
        st = flowkv_plan_stats()
        segp = C.POINTER(flowkv_segment)()
        _check(_lib.flowkv_plan_info(self.handle, C.byref(st), C.byref(segp)))
        return st, segp

    @property
    def stats(self) -> dict:
        return self.info()[0].as_dict()

    @property
    def segments(self) -> List[dict]:
        st, segp = self.info()
        names = [n for n, _ in flowkv_segment._fields_ if not n.startswith("_")]
        return [{k: int(getattr(segp[i], k)) for k in names} for i in range(st.n_segments)]

    def transfer(self, stream: int = 0) -> None:
        flowkv_transfer(self, stream)

    def pack(self, staging: int, nbytes: int, stream: int = 0) -> None:
        flowkv_pack(self, staging, nbytes, stream)

    def unpack(self, staging: int, nbytes: int, stream: int = 0) -> None:
        flowkv_unpack(self, staging, nbytes, stream)

    def destroy(self) -> None:
        if self._h:
            _lib.flowkv_plan_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _tuning(tuning) -> Optional[flowkv_tuning]:
    if tuning is None:
        return None
    if isinstance(tuning, flowkv_tuning):
        return tuning
    t = flowkv_tuning()
    for k, v in dict(tuning).items():
        if isinstance(v, str):
            v = {"ldst": FLOWKV_VARIANT_LDST, "bulk": FLOWKV_VARIANT_BULK, "auto": 0}[v]
        setattr(t, k, int(v))
    return t


def flowkv_plan(src: Optional[flowkv_pool], dst: Optional[flowkv_pool], requests, flags: int = 0,
                tuning=None, stream: int = 0) -> Plan:
    """``requests``: a sequence of :class:`Request`-like objects, or a :class:`RequestBatch` marshalled beforehand."""
    arr, n, keep = _requests_arg(requests)
    out = C.c_void_p()
    t = _tuning(tuning)
    _check(_lib.flowkv_plan(C.byref(src) if src is not None else None, C.byref(dst) if dst is not None else None,
                            arr, n, flags, C.byref(t) if t is not None else None, C.c_void_p(stream), C.byref(out)))
    del keep
    return Plan(out.value)


def flowkv_plan_host(src: Optional[flowkv_pool], dst: Optional[flowkv_pool], requests, flags: int = 0,
                     tuning=None) -> Plan:
    arr, n, keep = _requests_arg(requests)
    out = C.c_void_p()
    t = _tuning(tuning)
    _check(_lib.flowkv_plan_host(C.byref(src) if src is not None else None,
                                 C.byref(dst) if dst is not None else None, arr, n, flags,
                                 C.byref(t) if t is not None else None, C.byref(out)))
    del keep
    return Plan(out.value)


def flowkv_transfer(plan: Plan, stream: int = 0) -> None:
    _check(_lib.flowkv_transfer(plan.handle, C.c_void_p(stream)))


def flowkv_transfer_static(plan: Plan, stream: int = 0) -> None:
    """flowkv_transfer for callers that may not allocate device memory (an engine that owns all of HBM, a loop that
    cannot take an allocator stall): the schedule rides in a fixed 1 MiB array inside the library instead of a
    per-plan device buffer.  ``plan`` may come from :func:`flowkv_plan_host`.  At most
    ``FLOWKV_STATIC_SCHEDULE_ENTRIES`` schedule entries; calls that overlap on the GPU race on the array."""
    _check(_lib.flowkv_transfer_static(plan.handle, C.c_void_p(stream)))


def flowkv_pack(plan: Plan, staging: int, nbytes: int, stream: int = 0) -> None:
    _check(_lib.flowkv_pack(plan.handle, C.c_void_p(staging), nbytes, C.c_void_p(stream)))


def flowkv_unpack(plan: Plan, staging: int, nbytes: int, stream: int = 0) -> None:
    _check(_lib.flowkv_unpack(plan.handle, C.c_void_p(staging), nbytes, C.c_void_p(stream)))


def flowkv_transfer_layers(plan: Plan, layer_begin: int, layer_end: int, stream: int = 0) -> None:
    _check(_lib.flowkv_transfer_layers(plan.handle, layer_begin, layer_end, C.c_void_p(stream)))


def flowkv_pack_layers(plan: Plan, staging: int, nbytes: int, layer_begin: int, layer_end: int, stream: int = 0) -> None:
    _check(_lib.flowkv_pack_layers(plan.handle, C.c_void_p(staging), nbytes, layer_begin, layer_end, C.c_void_p(stream)))


def flowkv_unpack_layers(plan: Plan, staging: int, nbytes: int, layer_begin: int, layer_end: int, stream: int = 0) -> None:
    _check(_lib.flowkv_unpack_layers(plan.handle, C.c_void_p(staging), nbytes, layer_begin, layer_end, C.c_void_p(stream)))


def flowkv_transfer_via_host(plan: Plan, host_staging: int, nbytes: int, n_chunks: int = 0, ctas_per_kernel: int = 0,
                             stream: int = 0, device_scratch: int = 0, scratch_bytes: int = 0) -> None:
    _check(_lib.flowkv_transfer_via_host(plan.handle, C.c_void_p(host_staging), nbytes, n_chunks, ctas_per_kernel,
                                         C.c_void_p(device_scratch) if device_scratch else None, scratch_bytes,
                                         C.c_void_p(stream)))


def flowkv_via_host_scratch_bytes(plan: Plan, n_chunks: int = 0) -> int:
    out = C.c_uint64()
    _check(_lib.flowkv_via_host_scratch_bytes(plan.handle, n_chunks, C.byref(out)))
    return int(out.value)


def flowkv_window_bytes(plan: Plan, layer_begin: int, layer_end: int) -> int:
    out = C.c_uint64()
    _check(_lib.flowkv_window_bytes(plan.handle, layer_begin, layer_end, C.byref(out)))
    return int(out.value)


def flowkv_pack_window(plan: Plan, window: int, nbytes: int, layer_begin: int, layer_end: int, stream: int = 0) -> None:
    _check(_lib.flowkv_pack_window(plan.handle, C.c_void_p(window), nbytes, layer_begin, layer_end, C.c_void_p(stream)))


def flowkv_unpack_window(plan: Plan, window: int, nbytes: int, layer_begin: int, layer_end: int, stream: int = 0) -> None:
    _check(_lib.flowkv_unpack_window(plan.handle, C.c_void_p(window), nbytes, layer_begin, layer_end, C.c_void_p(stream)))


def flowkv_transfer_tables(src: flowkv_pool, dst: flowkv_pool, src_tables: int, dst_tables: int, num_tokens: int,
                           n_reqs: int, max_src_blocks: int, max_dst_blocks: int, max_tokens: int, error_flag: int = 0,
                           tuning=None, stream: int = 0) -> None:
    """Device pointers as integers: int32 tables [n_reqs][max_*_blocks], uint32 lengths [n_reqs], uint32 flag."""
    t = _tuning(tuning)
    _check(_lib.flowkv_transfer_tables(C.byref(src), C.byref(dst), C.c_void_p(src_tables), C.c_void_p(dst_tables),
                                       C.c_void_p(num_tokens), n_reqs, max_src_blocks, max_dst_blocks, max_tokens,
                                       C.c_void_p(error_flag) if error_flag else None,
                                       C.byref(t) if t is not None else None, C.c_void_p(stream)))


def flowkv_transfer_tables_layers(src: flowkv_pool, dst: flowkv_pool, src_tables: int, dst_tables: int, num_tokens: int,
                                  n_reqs: int, max_src_blocks: int, max_dst_blocks: int, max_tokens: int,
                                  layer_begin: int, layer_end: int, error_flag: int = 0, tuning=None, stream: int = 0) -> None:
    """flowkv_transfer_tables restricted to layers [layer_begin, layer_end)."""
    t = _tuning(tuning)
    _check(_lib.flowkv_transfer_tables_layers(C.byref(src), C.byref(dst), C.c_void_p(src_tables), C.c_void_p(dst_tables),
                                              C.c_void_p(num_tokens), n_reqs, max_src_blocks, max_dst_blocks, max_tokens,
                                              layer_begin, layer_end, C.c_void_p(error_flag) if error_flag else None,
                                              C.byref(t) if t is not None else None, C.c_void_p(stream)))


def _tables_window(fn, pool, tables, cu_tokens, n_reqs, max_blocks, max_tokens, window, nbytes, layer_begin, layer_end,
                   error_flag, tuning, stream) -> None:
    t = _tuning(tuning)
    _check(fn(C.byref(pool), C.c_void_p(tables), C.c_void_p(cu_tokens), n_reqs, max_blocks, max_tokens, C.c_void_p(window),
              nbytes, layer_begin, layer_end, C.c_void_p(error_flag) if error_flag else None,
              C.byref(t) if t is not None else None, C.c_void_p(stream)))


def flowkv_pack_tables(src: flowkv_pool, src_tables: int, cu_tokens: int, n_reqs: int, max_src_blocks: int,
                       max_tokens: int, window: int, nbytes: int, layer_begin: int, layer_end: int, error_flag: int = 0,
                       tuning=None, stream: int = 0) -> None:
    """Device pointers as integers: int32 table [n_reqs][max_src_blocks], uint64 cu_tokens [n_reqs+1], uint32 flag."""
    _tables_window(_lib.flowkv_pack_tables, src, src_tables, cu_tokens, n_reqs, max_src_blocks, max_tokens, window, nbytes,
                   layer_begin, layer_end, error_flag, tuning, stream)


def flowkv_unpack_tables(dst: flowkv_pool, dst_tables: int, cu_tokens: int, n_reqs: int, max_dst_blocks: int,
                         max_tokens: int, window: int, nbytes: int, layer_begin: int, layer_end: int, error_flag: int = 0,
                         tuning=None, stream: int = 0) -> None:
    _tables_window(_lib.flowkv_unpack_tables, dst, dst_tables, cu_tokens, n_reqs, max_dst_blocks, max_tokens, window, nbytes,
                   layer_begin, layer_end, error_flag, tuning, stream)


def flowkv_trim() -> None:
    """Give back the library's idle caches (plane-offset tables no plan holds, finished staging buffers, unused helper
    streams).  Synchronises the device when it drops a table."""
    _check(_lib.flowkv_trim())


def flowkv_cache_counts() -> dict:
    a, b = C.c_uint32(), C.c_uint32()
    _check(_lib.flowkv_cache_counts(C.byref(a), C.byref(b)))
    return {"plane_offset_tables": int(a.value), "pinned_buffers": int(b.value)}


def flowkv_plan_destroy(plan: Plan) -> None:
    plan.destroy()


def flowkv_baseline_blockwise(src: flowkv_pool, dst: flowkv_pool, requests, stream: int = 0) -> int:
    arr, n, keep = _requests_arg(requests)
    calls = C.c_uint64()
    _check(_lib.flowkv_baseline_blockwise(C.byref(src), C.byref(dst), arr, n, C.c_void_p(stream), C.byref(calls)))
    del keep
    return int(calls.value)


def flowkv_baseline_segmentwise(plan: Plan, stream: int = 0) -> int:
    calls = C.c_uint64()
    _check(_lib.flowkv_baseline_segmentwise(plan.handle, C.c_void_p(stream), C.byref(calls)))
    return int(calls.value)


class Allocator:
    """Owner of a ``flowkv_allocator_t*`` (segment-based block allocator)."""

    def __init__(self, num_blocks: int):
        h = C.c_void_p()
        _check(_lib.flowkv_alloc_create(num_blocks, C.byref(h)))
        self._h = h

    def allocate(self, n: int):
        """-> (int32 ids in allocation order, number of segments used)"""
        ids = np.empty(max(n, 1), dtype=np.int32)
        segs = C.c_uint32()
        _check(_lib.flowkv_alloc_allocate(self._h, n, ids.ctypes.data, C.byref(segs)))
        return ids[:n].copy(), int(segs.value)

    def free(self, ids) -> None:
        a = np.ascontiguousarray(np.asarray(ids, dtype=np.int32))
        _check(_lib.flowkv_alloc_free(self._h, a.ctypes.data if a.size else None, a.size))

    def stats(self) -> dict:
        fb, fs, lg = C.c_uint32(), C.c_uint32(), C.c_uint32()
        _check(_lib.flowkv_alloc_stats(self._h, C.byref(fb), C.byref(fs), C.byref(lg)))
        return {"free_blocks": fb.value, "free_segments": fs.value, "largest_segment": lg.value}

    def destroy(self) -> None:
        if self._h:
            _lib.flowkv_alloc_destroy(self._h)
            self._h = C.c_void_p(None)

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass
