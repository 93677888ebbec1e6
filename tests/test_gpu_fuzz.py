"""`-m gpu` seeded differential fuzz: random shapes, layouts (named and padded STRIDED), block-size pairs, block
tables, batch compositions, operations and tunings — the CUDA path against the CPU oracle, bit for bit over
whole buffers (sentinel-filled).  Every case is reproducible from its index."""
import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import pools as P
from tests import gpu_common as G

pytestmark = pytest.mark.gpu

import os

LAYOUTS = ["lkbthd", "blkhtd", "blkthd", "padded"]
ELEM_BYTES = [2, 1, 2, 4]
# FLOWKV_FUZZ_OFFSET shifts the case indices (a soak run: FLOWKV_FUZZ_OFFSET=400 FLOWKV_FUZZ_CASES=4000 pytest ...)
FUZZ_OFFSET = int(os.environ.get("FLOWKV_FUZZ_OFFSET", "0"))
FUZZ_CASES = int(os.environ.get("FLOWKV_FUZZ_CASES", "400"))


def _geom(rng, layout, L, H, D, NB, BS, e=2, separate=False):
    """-> (oracle geometry, strides or None, plane offsets or None).  'padded' = token-major interior with padding
    after every block, K|V slab and layer (a STRIDED pool: separate allocations / alignment padding); with
    ``separate`` its layers — or every K and every V — sit at shuffled, gapped offsets of their own (reading A22: a
    tensor per layer, or per plane)."""
    if layout != "padded":
        return getattr(O.PoolGeom, layout)(L, H, D, e, NB, BS), None, None
    row, tok = D * e, H * D * e
    blk = BS * tok + 32 * int(rng.integers(0, 5))
    kv = NB * blk + 32 * int(rng.integers(0, 9))
    lay = 2 * kv + 32 * int(rng.integers(0, 3))
    g = O.PoolGeom(L, H, D, e, NB, BS, lay, kv, blk, tok, row)
    if not separate:
        return g, [lay, kv, blk, tok, row], None
    unit = 16 if rng.random() < 0.25 else 32               # a quarter of them only 16-byte aligned (128-bit path)
    planes = rng.random() < 0.5                            # K and V separate tensors too (A3), else stacked per layer
    n = 2 * L if planes else L
    size = g.plane_bytes() if planes else g.layer_bytes()
    off, pos = [0] * n, unit * int(rng.integers(0, 3))
    for i in rng.permutation(n):
        off[int(i)] = pos
        pos += size + unit * int(rng.integers(1, 6))
    g = g.with_plane_offsets(off) if planes else g.with_layer_offsets(off)
    return g, [lay, kv, blk, tok, row], list(g.plane_off)


def _pools(rng, idx, L, H, D, e, lay_s, bs_s, NBs, lay_d, bs_d, NBd):
    """Both pools of a case: oracle geometries, device buffers (src random bits, dst sentinel) and descriptors."""
    gs, ss, los = _geom(rng, lay_s, L, H, D, NBs, bs_s, e, separate=lay_s == "padded" and idx % 2 == 0)
    gd, sd, lod = _geom(rng, lay_d, L, H, D, NBd, bs_d, e, separate=lay_d == "padded" and idx % 2 == 1)
    src_buf, dst_buf = P.alloc_bytes(gs.span_bytes()), P.alloc_bytes(gd.span_bytes())
    P.fill_values(src_buf, "bits", "fp16", 9000 + idx)
    P.fill_sentinel(dst_buf)
    src = F.make_pool(src_buf.data_ptr(), L, H, D, e, NBs, bs_s, "strided" if ss else lay_s, ss, plane_offsets=los)
    dst = F.make_pool(dst_buf.data_ptr(), L, H, D, e, NBd, bs_d, "strided" if sd else lay_d, sd, plane_offsets=lod)
    return gs, gd, ss, sd, src_buf, dst_buf, src, dst


def _table(rng, n, NB, p_cont):
    """n distinct block ids; continues +1 with probability p_cont when that id is still free."""
    free = np.ones(NB, bool)
    out, cur = [], -2
    for _ in range(n):
        if cur + 1 < NB and cur >= 0 and free[cur + 1] and rng.random() < p_cont:
            cur += 1
        else:
            cur = int(rng.choice(np.nonzero(free)[0]))
        free[cur] = False
        out.append(cur)
    return np.asarray(out, np.int32)


def _case(idx):
    rng = np.random.default_rng(9000 + idx)
    L = int(rng.integers(1, 5))
    H = int(rng.choice([1, 2, 3, 4, 8]))
    e = ELEM_BYTES[idx % 4]                        # half the cases 2-byte, a quarter fp8 (1), a quarter fp32 (4)
    D = int(rng.choice([16, 32, 48, 128, 256])) // e          # rows of 16 .. 256 bytes at every element size
    bs_s, bs_d = int(2 ** rng.integers(0, 6)), int(2 ** rng.integers(0, 6))
    lay_s, lay_d = str(rng.choice(LAYOUTS)), str(rng.choice(LAYOUTS))
    if rng.random() < 0.35:                       # favour the congruent pairs that take the flat path
        lay_d, bs_d = lay_s, bs_s
    n_req = int(rng.integers(1, 5))
    Ts = [int(rng.integers(0, 200)) if rng.random() < 0.9 else 0 for _ in range(n_req)]
    ns = [-(-t // bs_s) for t in Ts]
    nd = [-(-t // bs_d) for t in Ts]
    NBs, NBd = sum(ns) + int(rng.integers(1, 6)), sum(nd) + int(rng.integers(1, 6))
    stab = _table(rng, sum(ns), NBs, float(rng.choice([0.0, 0.5, 0.9])))
    dtab = _table(rng, sum(nd), NBd, float(rng.choice([0.0, 0.5, 0.9, 1.0])))
    if rng.random() < 0.2 and n_req > 1 and ns[0] and ns[1]:      # prefix sharing on the src side (A9)
        k = min(ns[0], ns[1])
        stab[ns[0]:ns[0] + k] = stab[:k]
    reqs, so, do = [], 0, 0
    for t, a, b in zip(Ts, ns, nd):
        reqs.append((t, stab[so:so + a].copy(), dtab[do:do + b].copy()))
        so += a
        do += b
    tuning = {}
    if rng.random() < 0.3:
        tuning["variant"] = "bulk"
    if rng.random() < 0.5:
        tuning["tile_bytes"] = int(2 ** rng.integers(10, 17))
        if tuning.get("variant") == "bulk":
            tuning["tile_bytes"] = min(tuning["tile_bytes"], 65536)
    if rng.random() < 0.4:
        thr = int(2 ** rng.integers(5, 10))
        tuning["threads"] = thr
        tuning["group_threads"] = int(2 ** rng.integers(5, int(np.log2(thr)) + 1))
    if rng.random() < 0.3:
        tuning["tile_order"] = int(rng.integers(1, 3))
    if rng.random() < 0.3:
        tuning["cache_hint"] = int(rng.integers(1, 4))
    if rng.random() < 0.3:
        tuning["max_sms"], tuning["ctas_per_sm"] = int(rng.integers(1, 9)), int(rng.integers(1, 4))
    if rng.random() < 0.5:
        tuning["plan_in_params"] = 1
    op = str(rng.choice(["transfer", "layers", "pack_unpack", "windows"]))
    return rng, (L, H, D, e), (lay_s, bs_s, NBs), (lay_d, bs_d, NBd), reqs, tuning, op


@pytest.mark.parametrize("idx", range(FUZZ_OFFSET, FUZZ_OFFSET + FUZZ_CASES))
def test_fuzz_against_oracle(idx):
    rng, (L, H, D, e), (lay_s, bs_s, NBs), (lay_d, bs_d, NBd), reqs, tuning, op = _case(idx)
    gs, gd, ss, sd, src_buf, dst_buf, src, dst = _pools(rng, idx, L, H, D, e, lay_s, bs_s, NBs, lay_d, bs_d, NBd)
    src_np = P.to_numpy(src_buf)
    freqs = [F.Request(t, a, b) for t, a, b in reqs]
    total = sum(t for t, _, _ in reqs)
    tokb = H * D * e
    what = f"case {idx}: {lay_s}{bs_s}->{lay_d}{bs_d} L{L} H{H} D{D} e{e} T={[t for t, _, _ in reqs]} {tuning} {op}"
    plan = F.flowkv_plan(src, dst, freqs, F.FLOWKV_CHECK_DST_ALIAS, tuning or None)
    if tuning.get("variant") == "bulk" and plan.stats["mode_transfer"] == 2 and not ss and not sd and total:
        # named layouts in rows mode: the bulk variant is honoured (TMA tensor path), not silently replaced
        assert plan.stats["variant"] == F.FLOWKV_VARIANT_BULK, what

    def expect_transfer(l0=0, l1=L):
        exp = np.full(gd.span_bytes(), P.SENTINEL_BYTE, np.uint8)
        for t, a, b in reqs:
            O.transfer(src_np, gs, exp, gd, a, b, t, l0, l1)
        return exp

    assert plan.stats["n_segments"] == sum(O.count_segments(a, bs_s, b, bs_d, t) for t, a, b in reqs), what
    n0 = F.flowkv_launch_count()
    if op == "transfer":
        plan.transfer()
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if total else 0), what
        G.assert_same(P.to_numpy(dst_buf), expect_transfer(), what)
    elif op == "layers":
        l0 = int(rng.integers(0, L + 1))
        l1 = int(rng.integers(l0, L + 1))
        F.flowkv_transfer_layers(plan, l0, l1)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if total and l1 > l0 else 0), what
        G.assert_same(P.to_numpy(dst_buf), expect_transfer(l0, l1), what)
    elif op == "pack_unpack":
        nbytes = plan.stats["staging_bytes"]
        staging = P.alloc_bytes(nbytes + 32)
        P.fill_sentinel(staging)
        plan.pack(staging.data_ptr(), nbytes)
        plan.unpack(staging.data_ptr(), nbytes)
        torch.cuda.synchronize()
        exp = np.full(nbytes + 32, P.SENTINEL_BYTE, np.uint8)
        off = 0
        for t, a, _ in reqs:
            O.pack(src_np, gs, a, t, exp, off)
            off += t
        G.assert_same(P.to_numpy(staging), exp, what + " (wire bytes)")
        G.assert_same(P.to_numpy(dst_buf), expect_transfer(), what + " (unpack)")
    else:
        cut = int(rng.integers(0, L + 1))
        for w0, w1 in ((0, cut), (cut, L)):
            nb = F.flowkv_window_bytes(plan, w0, w1)
            assert nb == total * 2 * (w1 - w0) * tokb
            win = P.alloc_bytes(nb + 32)
            P.fill_sentinel(win)
            F.flowkv_pack_window(plan, win.data_ptr(), nb, w0, w1)
            F.flowkv_unpack_window(plan, win.data_ptr(), nb, w0, w1)
            torch.cuda.synchronize()
            exp = np.full(nb + 32, P.SENTINEL_BYTE, np.uint8)
            off = 0
            for t, a, _ in reqs:
                O.pack_window(src_np, gs, a, t, exp, off, w0, w1)
                off += t
            G.assert_same(P.to_numpy(win), exp, what + f" (window [{w0},{w1}))")
        G.assert_same(P.to_numpy(dst_buf), expect_transfer(), what + " (windows unpacked)")
    G.assert_same(P.to_numpy(src_buf), src_np, what + " (src unchanged)")
    plan.destroy()


def _device_tables(reqs, width_s, width_d):
    """Padded 2-D tables (pad value -7: must never be read as a block id in use) and lengths, on the device."""
    n = len(reqs)
    st = np.full((n, width_s), -7, np.int32)
    dt = np.full((n, width_d), -7, np.int32)
    for i, (_, a, b) in enumerate(reqs):
        st[i, :len(a)] = a
        dt[i, :len(b)] = b
    lens = np.asarray([t for t, _, _ in reqs], np.uint32)
    to = lambda x: torch.from_numpy(x.view(np.int32) if x.dtype == np.uint32 else x).cuda()
    return to(st), to(dt), to(lens)


@pytest.mark.parametrize("idx", range(FUZZ_OFFSET, FUZZ_OFFSET + max(1, FUZZ_CASES * 3 // 10)))
def test_fuzz_table_driven_transfer(idx):
    """flowkv_transfer_tables: the kernel walks device-resident padded block tables itself (no plan) — same seeded
    cases as above, whole dst pool against the oracle, one launch, error flag stays clear."""
    rng, (L, H, D, e), (lay_s, bs_s, NBs), (lay_d, bs_d, NBd), reqs, tuning, _ = _case(idx)
    gs, gd, ss, sd, src_buf, dst_buf, src, dst = _pools(rng, idx, L, H, D, e, lay_s, bs_s, NBs, lay_d, bs_d, NBd)
    src_np = P.to_numpy(src_buf)
    max_t = max(t for t, _, _ in reqs) + int(rng.integers(0, 40))
    ws, wd = -(-max_t // bs_s) + int(rng.integers(0, 3)), -(-max_t // bs_d) + int(rng.integers(0, 3))
    st, dt, lens = _device_tables(reqs, max(ws, 1), max(wd, 1))
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    tn = {k: v for k, v in tuning.items() if k in ("threads", "group_threads", "max_sms", "ctas_per_sm")}
    if idx % 5 == 0:                        # narrow CTAs with the group left on auto (must clamp, not divide by zero)
        tn = {"threads": 32 if idx % 10 == 0 else 64}
    n0 = F.flowkv_launch_count()
    l0, l1 = 0, L
    if idx % 3 == 1:                        # layer-range form: one launch per range, the other layers stay untouched
        l0 = int(rng.integers(0, L + 1))
        l1 = int(rng.integers(l0, L + 1))
        F.flowkv_transfer_tables_layers(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), len(reqs), st.shape[1],
                                        dt.shape[1], max_t, l0, l1, flag.data_ptr(), tn or None)
    else:
        F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), len(reqs), st.shape[1], dt.shape[1],
                                 max_t, flag.data_ptr(), tn or None)
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() - n0 == (1 if max_t and l1 > l0 else 0)
    exp = np.full(gd.span_bytes(), P.SENTINEL_BYTE, np.uint8)
    for t, a, b in reqs:
        O.transfer(src_np, gs, exp, gd, a, b, t, l0, l1)
    what = f"tables case {idx} layers [{l0},{l1}): {lay_s}{bs_s}->{lay_d}{bs_d} L{L} H{H} D{D} e{e} T={[t for t, _, _ in reqs]} {tn}"
    G.assert_same(P.to_numpy(dst_buf), exp, what)
    assert int(flag.item()) == 0, what
    G.assert_same(P.to_numpy(src_buf), src_np, what + " (src unchanged)")


@pytest.mark.parametrize("idx", range(FUZZ_OFFSET, FUZZ_OFFSET + max(1, FUZZ_CASES * 3 // 10)))
def test_fuzz_table_driven_pack_unpack_windows(idx):
    """flowkv_pack_tables / flowkv_unpack_tables: device-resident tables and cumulative lengths, layer windows split
    at a random layer; each window == the oracle's okv_pack_window, unpacking them rebuilds the oracle's transfer;
    a window buffer that is too small raises flag bit 2 and is left untouched."""
    rng, (L, H, D, e), (lay_s, bs_s, NBs), (lay_d, bs_d, NBd), reqs, tuning, _ = _case(idx)
    gs, gd, ss, sd, src_buf, dst_buf, src, dst = _pools(rng, idx, L, H, D, e, lay_s, bs_s, NBs, lay_d, bs_d, NBd)
    src_np = P.to_numpy(src_buf)
    Ts = [t for t, _, _ in reqs]
    total, max_t = sum(Ts), max(Ts) + int(rng.integers(0, 9))
    st, dt, _ = _device_tables(reqs, max(1, -(-max_t // bs_s)), max(1, -(-max_t // bs_d)))
    cu = torch.from_numpy(np.concatenate([[0], np.cumsum(Ts)]).astype(np.int64)).cuda()
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    tn = {k: v for k, v in tuning.items() if k in ("threads", "group_threads", "max_sms", "ctas_per_sm")} or None
    if idx % 5 == 0:
        tn = {"threads": 32 if idx % 10 == 0 else 64}
    tokb = H * D * e
    cut = int(rng.integers(0, L + 1))
    what = f"tables windows case {idx}: {lay_s}{bs_s}->{lay_d}{bs_d} L{L} H{H} D{D} e{e} T={Ts} cut={cut} {tn}"
    for w0, w1 in ((0, cut), (cut, L)):
        nb = total * 2 * (w1 - w0) * tokb
        win = P.alloc_bytes(nb + 32)
        P.fill_sentinel(win)
        n0 = F.flowkv_launch_count()
        F.flowkv_pack_tables(src, st.data_ptr(), cu.data_ptr(), len(reqs), st.shape[1], max_t, win.data_ptr(), nb, w0, w1,
                             flag.data_ptr(), tn)
        F.flowkv_unpack_tables(dst, dt.data_ptr(), cu.data_ptr(), len(reqs), dt.shape[1], max_t, win.data_ptr(), nb, w0, w1,
                               flag.data_ptr(), tn)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (2 if max_t and w1 > w0 else 0), what
        exp = np.full(nb + 32, P.SENTINEL_BYTE, np.uint8)
        off = 0
        for t, a, _ in reqs:
            O.pack_window(src_np, gs, a, t, exp, off, w0, w1)
            off += t
        G.assert_same(P.to_numpy(win), exp, what + f" window [{w0},{w1})")
    exp = np.full(gd.span_bytes(), P.SENTINEL_BYTE, np.uint8)
    for t, a, b in reqs:
        O.transfer(src_np, gs, exp, gd, a, b, t)
    G.assert_same(P.to_numpy(dst_buf), exp, what + " (windows unpacked)")
    assert int(flag.item()) == 0, what
    if total and L:
        nb = total * 2 * L * tokb
        small = P.alloc_bytes(nb)
        P.fill_sentinel(small)
        F.flowkv_pack_tables(src, st.data_ptr(), cu.data_ptr(), len(reqs), st.shape[1], max_t, small.data_ptr(), nb - 16, 0, L,
                             flag.data_ptr(), tn)
        torch.cuda.synchronize()
        assert int(flag.item()) & 2, what + " (capacity flag)"
        last = max(i for i, t in enumerate(Ts) if t)           # the request that would cross the end is skipped whole
        lo = int(np.cumsum([0] + Ts)[last]) * 2 * L * tokb
        assert np.all(P.to_numpy(small)[lo:] == P.SENTINEL_BYTE), what + " (bytes of the skipped request)"
