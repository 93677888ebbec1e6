"""ctypes front end of the CPU oracle (``flowkv_oracle.c``) — TEST INFRASTRUCTURE ONLY.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_2504_03775_b200`` and the product never imports it.

The arithmetic lives in ``flowkv_oracle.c`` (one function per operation, each citing
the passage of /root/reference/PAPER.md it follows).  This file only builds that C
file with gcc, describes pools as stride tuples and marshals numpy arrays.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "flowkv_oracle.c")
_SO = os.path.join(_HERE, "libflowkv_oracle.so")


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain -O2, single-threaded, no tuning flags)."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        tmp = _SO + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-o", tmp, _SRC])
        os.replace(tmp, _SO)
    return _SO


class _Pool(C.Structure):
    _fields_ = [
        ("num_layers", C.c_uint32), ("num_kv_heads", C.c_uint32), ("head_dim", C.c_uint32),
        ("elem_bytes", C.c_uint32), ("num_blocks", C.c_uint32), ("block_size", C.c_uint32),
        ("s_layer", C.c_int64), ("s_kv", C.c_int64), ("s_block", C.c_int64),
        ("s_token", C.c_int64), ("s_head", C.c_int64),
        ("layer0", C.c_uint32), ("_pad", C.c_uint32),
        ("plane_off", C.c_void_p),
    ]


_lib = None


def _load():
    global _lib
    if _lib is None:
        lib = C.CDLL(build())
        u8p, i32p, u32p = C.c_void_p, C.c_void_p, C.c_void_p
        lib.okv_transfer.restype = C.c_int
        lib.okv_transfer.argtypes = [u8p, C.POINTER(_Pool), u8p, C.POINTER(_Pool), i32p, i32p,
                                     C.c_uint32, C.c_uint32, C.c_uint32]
        lib.okv_pack.restype = C.c_int
        lib.okv_pack.argtypes = [u8p, C.POINTER(_Pool), i32p, C.c_uint32, u8p, C.c_uint64,
                                 C.c_uint32, C.c_uint32]
        lib.okv_unpack.restype = C.c_int
        lib.okv_unpack.argtypes = [u8p, C.c_uint64, u8p, C.POINTER(_Pool), i32p, C.c_uint32,
                                   C.c_uint32, C.c_uint32]
        lib.okv_pack_window.restype = C.c_int
        lib.okv_pack_window.argtypes = [u8p, C.POINTER(_Pool), i32p, C.c_uint32, u8p, C.c_uint64,
                                        C.c_uint32, C.c_uint32]
        lib.okv_unpack_window.restype = C.c_int
        lib.okv_unpack_window.argtypes = [u8p, C.c_uint64, u8p, C.POINTER(_Pool), i32p, C.c_uint32,
                                          C.c_uint32, C.c_uint32]
        lib.okv_pack_planes.restype = C.c_int
        lib.okv_pack_planes.argtypes = lib.okv_pack_window.argtypes
        lib.okv_unpack_planes.restype = C.c_int
        lib.okv_unpack_planes.argtypes = lib.okv_unpack_window.argtypes
        lib.okv_align.restype = C.c_uint64
        lib.okv_align.argtypes = [i32p, C.c_uint32, i32p, C.c_uint32, C.c_uint32, u32p, u32p, C.c_uint64]
        lib.okv_blockwise_calls.restype = C.c_uint64
        lib.okv_blockwise_calls.argtypes = [C.c_uint32, C.c_uint32]
        _lib = lib
    return _lib


@dataclass(frozen=True)
class PoolGeom:
    """Geometry of a paged KV pool: shape and byte strides (dim stride = elem_bytes).

    The two named orders of Eq. 5:
      ``lkbthd``  [layer][K|V][block][token][head][dim]   — (L,2,B,H), H=[token][head][dim]
      ``blkhtd``  [block][layer][K|V][head][token][dim]   — (B,L,2,H), H=[head][token][dim]
      ``blkthd``  [block][layer][K|V][token][head][dim]   — (B,L,2,H), H=[token][head][dim]
    """
    num_layers: int
    num_kv_heads: int
    head_dim: int
    elem_bytes: int
    num_blocks: int
    block_size: int
    s_layer: int
    s_kv: int
    s_block: int
    s_token: int
    s_head: int
    plane_off: tuple | None = None      # readings A22 / A3: byte offset of every plane 2*l + c (separate allocations)

    def with_plane_offsets(self, plane_off) -> "PoolGeom":
        """The same pool with every plane (layer, K|V) at its own byte offset from the buffer start; s_layer and s_kv
        are then unused (the cache the paper starts from keeps 'separate tensor structures across all layer
        dimensions'; A3: K and V may be separate tensors as well)."""
        off = tuple(int(x) for x in plane_off)
        assert len(off) == 2 * self.num_layers
        return PoolGeom(self.num_layers, self.num_kv_heads, self.head_dim, self.elem_bytes, self.num_blocks,
                        self.block_size, self.s_layer, self.s_kv, self.s_block, self.s_token, self.s_head, off)

    def with_layer_offsets(self, layer_off) -> "PoolGeom":
        """One tensor per layer with K and V stacked inside it: plane (l, c) at layer_off[l] + c * s_kv."""
        assert len(layer_off) == self.num_layers
        return self.with_plane_offsets([int(o) + c * self.s_kv for o in layer_off for c in (0, 1)])

    def plane_bytes(self) -> int:
        """Bytes from the first to one past the last addressable element of ONE plane."""
        return ((self.num_blocks - 1) * self.s_block + (self.block_size - 1) * self.s_token
                + (self.num_kv_heads - 1) * self.s_head + self.head_dim * self.elem_bytes)

    def layer_bytes(self) -> int:
        """The same for ONE layer with K and V stacked (s_kv apart)."""
        return self.s_kv + self.plane_bytes()

    @staticmethod
    def lkbthd(L, Hkv, Dh, e, NB, BS) -> "PoolGeom":
        s_head = Dh * e
        s_token = Hkv * s_head
        s_block = BS * s_token
        s_kv = NB * s_block
        s_layer = 2 * s_kv
        return PoolGeom(L, Hkv, Dh, e, NB, BS, s_layer, s_kv, s_block, s_token, s_head)

    @staticmethod
    def blkhtd(L, Hkv, Dh, e, NB, BS) -> "PoolGeom":
        s_token = Dh * e
        s_head = BS * s_token
        s_kv = Hkv * s_head
        s_layer = 2 * s_kv
        s_block = L * s_layer
        return PoolGeom(L, Hkv, Dh, e, NB, BS, s_layer, s_kv, s_block, s_token, s_head)

    @staticmethod
    def blkthd(L, Hkv, Dh, e, NB, BS) -> "PoolGeom":
        """(B,L,2,H) with H=[token][head][dim]: Eq. 5's right side with H untouched."""
        s_head = Dh * e
        s_token = Hkv * s_head
        s_kv = BS * s_token
        s_layer = 2 * s_kv
        s_block = L * s_layer
        return PoolGeom(L, Hkv, Dh, e, NB, BS, s_layer, s_kv, s_block, s_token, s_head)

    @property
    def bytes_per_token(self) -> int:
        return 2 * self.num_layers * self.num_kv_heads * self.head_dim * self.elem_bytes

    def span_bytes(self) -> int:
        """Bytes from the first to one past the last addressable element."""
        if self.plane_off is not None:
            return max(self.plane_off) + self.plane_bytes()
        return ((self.num_layers - 1) * self.s_layer + self.s_kv + (self.num_blocks - 1) * self.s_block
                + (self.block_size - 1) * self.s_token + (self.num_kv_heads - 1) * self.s_head
                + self.head_dim * self.elem_bytes)

    def _c(self, layer0: int = 0) -> _Pool:
        p = _Pool(self.num_layers, self.num_kv_heads, self.head_dim, self.elem_bytes,
                  self.num_blocks, self.block_size, self.s_layer, self.s_kv, self.s_block,
                  self.s_token, self.s_head, layer0, 0, None)
        if self.plane_off is not None:
            assert layer0 == 0, "a pool of separate planes is handed over whole"
            p._keep = np.asarray(self.plane_off, dtype=np.int64)     # kept alive by the struct object
            p.plane_off = p._keep.ctypes.data
        return p


def _u8(a: np.ndarray, writable: bool) -> int:
    assert a.dtype == np.uint8 and a.flags.c_contiguous, "oracle buffers are flat uint8 arrays"
    if writable:
        assert a.flags.writeable
    return a.ctypes.data


def _tab(t) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(t, dtype=np.int32))


def transfer(src: np.ndarray, sp: PoolGeom, dst: np.ndarray, dp: PoolGeom, src_tab, dst_tab, T: int,
             l0: int = 0, l1: int | None = None, src_layer0: int = 0, dst_layer0: int = 0) -> None:
    """dst[.., Dst[t//BS_d], t%BS_d, ..] := src[.., Src[t//BS_s], t%BS_s, ..] for t < T (in place).

    ``src`` / ``dst`` are flat uint8 buffers that start at layer ``*_layer0`` of their pool.
    """
    l1 = sp.num_layers if l1 is None else l1
    st, dt = _tab(src_tab), _tab(dst_tab)
    assert len(st) * sp.block_size >= T and len(dt) * dp.block_size >= T
    rc = _load().okv_transfer(_u8(src, False), C.byref(sp._c(src_layer0)), _u8(dst, True),
                              C.byref(dp._c(dst_layer0)), st.ctypes.data, dt.ctypes.data, T, l0, l1)
    if rc != 0:
        raise ValueError("oracle: block id out of range or shape mismatch")


def pack(src: np.ndarray, sp: PoolGeom, src_tab, T: int, staging: np.ndarray, req_tok_off: int,
         l0: int = 0, l1: int | None = None) -> None:
    l1 = sp.num_layers if l1 is None else l1
    st = _tab(src_tab)
    assert len(st) * sp.block_size >= T
    rc = _load().okv_pack(_u8(src, False), C.byref(sp._c()), st.ctypes.data, T, _u8(staging, True),
                          req_tok_off, l0, l1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def unpack(staging: np.ndarray, req_tok_off: int, dst: np.ndarray, dp: PoolGeom, dst_tab, T: int,
           l0: int = 0, l1: int | None = None) -> None:
    l1 = dp.num_layers if l1 is None else l1
    dt = _tab(dst_tab)
    assert len(dt) * dp.block_size >= T
    rc = _load().okv_unpack(_u8(staging, False), req_tok_off, _u8(dst, True), C.byref(dp._c()),
                            dt.ctypes.data, T, l0, l1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def pack_window(src: np.ndarray, sp: PoolGeom, src_tab, T: int, window: np.ndarray, req_tok_off: int,
                w0: int, w1: int) -> None:
    """Layers [w0,w1) of one request into a buffer that holds only those layers (reading A20)."""
    st = _tab(src_tab)
    assert len(st) * sp.block_size >= T
    rc = _load().okv_pack_window(_u8(src, False), C.byref(sp._c()), st.ctypes.data, T, _u8(window, True),
                                 req_tok_off, w0, w1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def unpack_window(window: np.ndarray, req_tok_off: int, dst: np.ndarray, dp: PoolGeom, dst_tab, T: int,
                  w0: int, w1: int) -> None:
    dt = _tab(dst_tab)
    assert len(dt) * dp.block_size >= T
    rc = _load().okv_unpack_window(_u8(window, False), req_tok_off, _u8(dst, True), C.byref(dp._c()),
                                   dt.ctypes.data, T, w0, w1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def pack_planes(src: np.ndarray, sp: PoolGeom, src_tab, T: int, window: np.ndarray, req_tok_off: int,
                p0: int, p1: int) -> None:
    """Planes [p0,p1) (plane = 2*layer + kv) of one request into a buffer that holds only those planes (A21)."""
    st = _tab(src_tab)
    assert len(st) * sp.block_size >= T and 0 <= p0 <= p1 <= 2 * sp.num_layers
    rc = _load().okv_pack_planes(_u8(src, False), C.byref(sp._c()), st.ctypes.data, T, _u8(window, True),
                                 req_tok_off, p0, p1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def unpack_planes(window: np.ndarray, req_tok_off: int, dst: np.ndarray, dp: PoolGeom, dst_tab, T: int,
                  p0: int, p1: int) -> None:
    dt = _tab(dst_tab)
    assert len(dt) * dp.block_size >= T and 0 <= p0 <= p1 <= 2 * dp.num_layers
    rc = _load().okv_unpack_planes(_u8(window, False), req_tok_off, _u8(dst, True), C.byref(dp._c()),
                                   dt.ctypes.data, T, p0, p1)
    if rc != 0:
        raise ValueError("oracle: block id out of range")


def align(src_tab, bs_s: int, dst_tab, bs_d: int, T: int):
    """Bidirectional segment alignment of one request -> list of (first_token, n_tokens).

    Either table may be ``None`` (that side is a dense buffer)."""
    st = _tab(src_tab) if src_tab is not None else None
    dt = _tab(dst_tab) if dst_tab is not None else None
    lib = _load()
    sp = st.ctypes.data if st is not None else None
    dp = dt.ctypes.data if dt is not None else None
    n = lib.okv_align(sp, bs_s, dp, bs_d, T, None, None, 0)
    first = np.zeros(max(n, 1), dtype=np.uint32)
    cnt = np.zeros(max(n, 1), dtype=np.uint32)
    n2 = lib.okv_align(sp, bs_s, dp, bs_d, T, first.ctypes.data, cnt.ctypes.data, n)
    assert n2 == n
    return [(int(first[i]), int(cnt[i])) for i in range(n)]


def count_segments(src_tab, bs_s: int, dst_tab, bs_d: int, T: int) -> int:
    st = _tab(src_tab) if src_tab is not None else None
    dt = _tab(dst_tab) if dst_tab is not None else None
    return int(_load().okv_align(st.ctypes.data if st is not None else None, bs_s,
                                 dt.ctypes.data if dt is not None else None, bs_d, T, None, None, 0))


def blockwise_calls(n_blocks: int, num_layers: int) -> int:
    """Calls of the per-block-per-layer-per-K|V scheme."""
    return int(_load().okv_blockwise_calls(n_blocks, num_layers))
