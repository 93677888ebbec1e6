"""Pins of the CPU oracle against things other than itself (all CPU, `-m "not gpu"`).

Each test names the plausible oracle mistake it would catch.  Nothing here touches the CUDA path.
"""
import json
import os

import numpy as np
import pytest

from oracle import oracle as O
from tests import helpers as Hh

GOLD = os.path.join(os.path.dirname(__file__), "golden")
SENT = 0xA5


def _rand_pool(rng, nbytes):
    return rng.integers(0, 256, size=nbytes, dtype=np.uint8)


def _geom(layout, L, H, D, NB, BS):
    return getattr(O.PoolGeom, layout)(L, H, D, 2, NB, BS)


# ---------------------------------------------------------------------------------------
# element placement
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", ["lkbthd", "blkhtd", "blkthd"])
def test_same_layout_full_blocks_equals_numpy_fancy_indexing(layout):
    """Catches: wrong stride order, swapped src/dst table, K|V or layer axis mix-up."""
    rng = np.random.default_rng(1)
    L, H, D, NB, BS, n = 3, 2, 8, 11, 4, 6
    g = _geom(layout, L, H, D, NB, BS)
    src = _rand_pool(rng, g.span_bytes())
    dst = np.full(g.span_bytes(), SENT, np.uint8)
    Src = rng.permutation(NB)[:n]
    Dst = rng.permutation(NB)[:n]
    O.transfer(src, g, dst, g, Src, Dst, n * BS)
    exp = np.full(g.span_bytes(), SENT, np.uint8)
    ev = Hh.logical_view(exp, layout, L, NB, BS, H, D)
    sv = Hh.logical_view(src, layout, L, NB, BS, H, D)
    ev[:, :, Dst] = sv[:, :, Src]
    assert np.array_equal(dst, exp)


@pytest.mark.parametrize("bs_s,bs_d,src_layout,dst_layout", [
    (4, 4, "lkbthd", "blkhtd"), (2, 8, "lkbthd", "blkhtd"), (8, 2, "blkhtd", "lkbthd"), (4, 16, "lkbthd", "lkbthd"),
    (4, 4, "lkbthd", "blkthd"), (8, 2, "blkthd", "blkhtd"), (2, 4, "blkhtd", "blkthd"),
])
def test_layout_and_block_size_conversion_equals_numpy_reshape(bs_s, bs_d, src_layout, dst_layout):
    """Full blocks on both sides: gather -> flatten tokens -> regroup into dst blocks.
    Catches: head/token transposition errors, wrong div/mod block size on one side."""
    rng = np.random.default_rng(2)
    L, H, D = 2, 3, 8
    T = 32
    ns, nd = T // bs_s, T // bs_d
    NBs, NBd = ns + 3, nd + 2
    gs, gd = _geom(src_layout, L, H, D, NBs, bs_s), _geom(dst_layout, L, H, D, NBd, bs_d)
    src = _rand_pool(rng, gs.span_bytes())
    dst = np.full(gd.span_bytes(), SENT, np.uint8)
    Src, Dst = rng.permutation(NBs)[:ns], rng.permutation(NBd)[:nd]
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    sv = Hh.logical_view(src, src_layout, L, NBs, bs_s, H, D)
    toks = sv[:, :, Src].reshape(L, 2, T, H, D)
    exp = np.full(gd.span_bytes(), SENT, np.uint8)
    ev = Hh.logical_view(exp, dst_layout, L, NBd, bs_d, H, D)
    ev[:, :, Dst] = toks.reshape(L, 2, nd, bs_d, H, D)
    assert np.array_equal(dst, exp)


def test_eq5_reorder_is_a_pure_axis_permutation():
    """Eq. 5: (L,2,B,H) -> (B,L,2,H) with identity tables and full blocks is numpy's
    transpose(2,0,1,3) of the same bytes.  Catches: a blkthd stride that is not the (B,L,2,H) order."""
    rng = np.random.default_rng(21)
    L, H, D, NB, BS = 3, 2, 8, 5, 4
    gs, gd = _geom("lkbthd", L, H, D, NB, BS), _geom("blkthd", L, H, D, NB, BS)
    src = _rand_pool(rng, gs.span_bytes())
    dst = np.full(gd.span_bytes(), SENT, np.uint8)
    ident = np.arange(NB)
    O.transfer(src, gs, dst, gd, ident, ident, NB * BS)
    Hbytes = BS * H * D * 2
    exp = src.reshape(L, 2, NB, Hbytes).transpose(2, 0, 1, 3).reshape(-1)
    assert np.array_equal(dst, exp)
    back = np.full(gs.span_bytes(), SENT, np.uint8)
    O.transfer(dst, gd, back, gs, ident, ident, NB * BS)
    assert np.array_equal(back, src)


def test_self_describing_pool_lands_where_definition_says():
    """src rows carry their own (l,c,block,tok,h) in their first 5 words; after the move each dst row
    named by the definition must carry the coordinates computed directly from the tables.
    Independent of the oracle's src addressing.  Catches: off-by-one in t//BS, t%BS, wrong table side."""
    rng = np.random.default_rng(3)
    L, H, D, NBs, NBd, bs_s, bs_d, T = 2, 2, 8, 9, 5, 4, 8, 27
    gs, gd = _geom("lkbthd", L, H, D, NBs, bs_s), _geom("blkhtd", L, H, D, NBd, bs_d)
    src = np.zeros(gs.span_bytes(), np.uint8)
    sv = Hh.logical_view(src, "lkbthd", L, NBs, bs_s, H, D)
    l, c, b, t, h = np.meshgrid(np.arange(L), np.arange(2), np.arange(NBs), np.arange(bs_s), np.arange(H), indexing="ij")
    for k, a in enumerate((l, c, b, t, h)):
        sv[..., k] = a + 1
    Src = rng.permutation(NBs)[:-(-T // bs_s)]
    Dst = rng.permutation(NBd)[:-(-T // bs_d)]
    dst = np.zeros(gd.span_bytes(), np.uint8)
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    dv = Hh.logical_view(dst, "blkhtd", L, NBd, bs_d, H, D)
    seen = 0
    for tt in range(T):
        for ll in range(L):
            for cc in range(2):
                for hh in range(H):
                    row = dv[ll, cc, Dst[tt // bs_d], tt % bs_d, hh]
                    assert list(row[:5]) == [ll + 1, cc + 1, Src[tt // bs_s] + 1, tt % bs_s + 1, hh + 1]
                    seen += 1
    # and nothing else was written (rows not named stay zero)
    assert np.count_nonzero(dv[..., 0]) == seen


def test_identity_tables_is_memcmp_prefix():
    """Identity tables + identical geometry: dst prefix == src prefix byte for byte."""
    rng = np.random.default_rng(4)
    L, H, D, NB, BS = 1, 2, 8, 6, 4
    g = _geom("blkhtd", 1, H, D, NB, BS)   # L=1 blkhtd: a block is one contiguous span
    src = _rand_pool(rng, g.span_bytes())
    dst = np.full(g.span_bytes(), SENT, np.uint8)
    O.transfer(src, g, dst, g, np.arange(4), np.arange(4), 4 * BS)
    n = 4 * g.s_block
    assert dst[:n].tobytes() == src[:n].tobytes()
    assert np.all(dst[n:] == SENT)


@pytest.mark.parametrize("T", [0, 1, 5, 8, 9, 15])
def test_partial_last_block_and_untouched_bytes(T):
    """Reading A4: only t < T is copied; every other dst byte keeps the sentinel; src unchanged.
    Catches: whole-block copies, tail spill, writes into src."""
    rng = np.random.default_rng(5)
    L, H, D, NB, BS = 2, 2, 8, 6, 4
    gs, gd = _geom("lkbthd", L, H, D, NB, BS), _geom("blkhtd", L, H, D, NB, BS)
    src = _rand_pool(rng, gs.span_bytes())
    src0 = src.copy()
    dst = np.full(gd.span_bytes(), SENT, np.uint8)
    nb = -(-T // BS)
    Src, Dst = rng.permutation(NB)[:nb], rng.permutation(NB)[:nb]
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    assert np.array_equal(src, src0)
    exp = np.full(gd.span_bytes(), SENT, np.uint8)
    ev, sv = Hh.logical_view(exp, "blkhtd", L, NB, BS, H, D), Hh.logical_view(src, "lkbthd", L, NB, BS, H, D)
    for t in range(T):
        ev[:, :, Dst[t // BS], t % BS] = sv[:, :, Src[t // BS], t % BS]
    assert np.array_equal(dst, exp)
    assert np.count_nonzero(dst != SENT) <= T * gs.bytes_per_token


def test_all_65536_bit_patterns_survive():
    """Raw-bit fidelity: NaN payloads, -0, denormals, Inf.  Catches: any pass through a float type."""
    L, H, D, BS = 1, 2, 64, 16
    NB = 65536 // (2 * BS * H * D)  # 16 blocks -> 65,536 elements
    g = _geom("lkbthd", L, H, D, NB, BS)
    src = np.arange(65536, dtype=np.uint16).view(np.uint8).copy()
    assert src.size == g.span_bytes()
    dst = np.zeros_like(src)
    perm = np.random.default_rng(6).permutation(NB)
    O.transfer(src, g, dst, g, perm, np.arange(NB), NB * BS)
    sv, dv = Hh.logical_view(src, "lkbthd", L, NB, BS, H, D), Hh.logical_view(dst, "lkbthd", L, NB, BS, H, D)
    assert np.array_equal(dv, sv[:, :, perm])
    assert np.array_equal(np.sort(dst.view(np.uint16)), np.arange(65536, dtype=np.uint16))


def test_layer_range_and_layer_slab():
    """Layer windows: [l0,l1) touches only those layers; a slab handed in with layer0 gives the same bytes."""
    rng = np.random.default_rng(7)
    L, H, D, NB, BS, T = 4, 2, 8, 5, 4, 14
    g = _geom("lkbthd", L, H, D, NB, BS)
    src = _rand_pool(rng, g.span_bytes())
    Src, Dst = rng.permutation(NB)[:4], rng.permutation(NB)[:4]
    full = np.full(g.span_bytes(), SENT, np.uint8)
    O.transfer(src, g, full, g, Src, Dst, T)
    part = np.full(g.span_bytes(), SENT, np.uint8)
    O.transfer(src, g, part, g, Src, Dst, T, l0=1, l1=3)
    assert np.array_equal(part[g.s_layer:3 * g.s_layer], full[g.s_layer:3 * g.s_layer])
    assert np.all(part[:g.s_layer] == SENT) and np.all(part[3 * g.s_layer:] == SENT)
    slab = np.full(g.s_layer, SENT, np.uint8)
    O.transfer(src[2 * g.s_layer:3 * g.s_layer].copy(), g, slab, g, Src, Dst, T, l0=2, l1=3, src_layer0=2, dst_layer0=2)
    assert np.array_equal(slab, full[2 * g.s_layer:3 * g.s_layer])


def test_out_of_range_block_id_rejected():
    g = _geom("lkbthd", 1, 1, 8, 4, 4)
    src = np.zeros(g.span_bytes(), np.uint8)
    dst = np.zeros(g.span_bytes(), np.uint8)
    with pytest.raises(ValueError):
        O.transfer(src, g, dst, g, [4], [0], 4)
    with pytest.raises(ValueError):
        O.transfer(src, g, dst, g, [0], [-1], 4)


# ---------------------------------------------------------------------------------------
# pack / unpack (wire format reading A12)
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", ["lkbthd", "blkhtd"])
def test_pack_equals_numpy_gather_and_unpack_inverts(layout):
    """staging[request][layer][K|V][token][head][dim].  Catches: wrong request offset, plane stride T_r,
    token/head order in the wire format."""
    rng = np.random.default_rng(8)
    L, H, D, NB, BS = 2, 3, 8, 12, 4
    g = _geom(layout, L, H, D, NB, BS)
    src = _rand_pool(rng, g.span_bytes())
    Ts = [7, 0, 12, 5]
    perm = rng.permutation(NB)
    tabs, off = [], 0
    for T in Ts:
        nb = -(-T // BS)
        tabs.append(perm[off:off + nb]); off += nb
    bpt = g.bytes_per_token
    staging = np.full(sum(Ts) * bpt, SENT, np.uint8)
    sv = Hh.logical_view(src, layout, L, NB, BS, H, D)
    exp_parts, tok_off = [], 0
    for T, tab in zip(Ts, tabs):
        O.pack(src, g, tab, T, staging, tok_off)
        tok_off += T
        exp_parts.append(sv[:, :, tab].reshape(L, 2, len(tab) * BS, H, D)[:, :, :T].reshape(-1))
    assert np.array_equal(staging.view(np.uint16), np.concatenate(exp_parts))
    # unpack through DIFFERENT dst tables == transfer src->dst directly
    gd = _geom("blkhtd" if layout == "lkbthd" else "lkbthd", L, H, D, NB, BS * 2)
    dperm = rng.permutation(NB)
    d1 = np.full(gd.span_bytes(), SENT, np.uint8)
    d2 = np.full(gd.span_bytes(), SENT, np.uint8)
    tok_off = doff = 0
    for T, tab in zip(Ts, tabs):
        nb = -(-T // (BS * 2))
        dtab = dperm[doff:doff + nb]; doff += nb
        O.unpack(staging, tok_off, d1, gd, dtab, T)
        O.transfer(src, g, d2, gd, tab, dtab, T)
        tok_off += T
    assert np.array_equal(d1, d2)


@pytest.mark.parametrize("layout", ["lkbthd", "blkthd"])
def test_layer_window_equals_planes_cut_out_of_the_wire_format(layout):
    """Reading A20: a window [w0,w1) is numpy's gather restricted to those layers, i.e. the slab of planes
    [2*w0, 2*w1) of each request's region of the (already pinned) full wire format; the window [0,L) IS the
    wire format; unpacking disjoint windows rebuilds unpack of the whole.  Catches: a window base that still
    uses 2*L planes per token, a plane index not rebased to w0, K|V order inside a layer."""
    rng = np.random.default_rng(18)
    L, H, D, NB, BS = 4, 2, 8, 12, 4
    g = _geom(layout, L, H, D, NB, BS)
    src = _rand_pool(rng, g.span_bytes())
    Ts = [7, 12, 0, 5]
    perm = rng.permutation(NB)
    tabs, off = [], 0
    for T in Ts:
        nb = -(-T // BS)
        tabs.append(perm[off:off + nb]); off += nb
    tokb = H * D * 2
    sv = Hh.logical_view(src, layout, L, NB, BS, H, D)
    full = np.zeros(sum(Ts) * g.bytes_per_token, np.uint8)
    tok_off = 0
    for T, tab in zip(Ts, tabs):
        O.pack(src, g, tab, T, full, tok_off)
        tok_off += T
    for w0, w1 in [(0, 4), (1, 3), (3, 4), (2, 2)]:
        win = np.full(sum(Ts) * 2 * (w1 - w0) * tokb + 16, SENT, np.uint8)
        exp_parts, cut_parts, tok_off = [], [], 0
        for T, tab in zip(Ts, tabs):
            O.pack_window(src, g, tab, T, win, tok_off, w0, w1)
            exp_parts.append(sv[w0:w1, :, tab].reshape(w1 - w0, 2, len(tab) * BS, H, D)[:, :, :T].reshape(-1))
            base = tok_off * g.bytes_per_token
            cut_parts.append(full[base + 2 * w0 * T * tokb: base + 2 * w1 * T * tokb])
            tok_off += T
        body = win[:-16]
        assert np.array_equal(body.view(np.uint16), np.concatenate(exp_parts))
        assert np.array_equal(body, np.concatenate(cut_parts))
        assert np.all(win[-16:] == SENT)
        if (w0, w1) == (0, 4):
            assert np.array_equal(body, full)
    # unpack of windows [0,1) + [1,4) == unpack of the whole wire format
    gd = _geom("blkhtd", L, H, D, NB, BS * 2)
    dperm = rng.permutation(NB)
    d1 = np.full(gd.span_bytes(), SENT, np.uint8)
    d2 = np.full(gd.span_bytes(), SENT, np.uint8)
    for w0, w1 in [(0, 1), (1, 4)]:
        win = np.zeros(sum(Ts) * 2 * (w1 - w0) * tokb, np.uint8)
        tok_off = doff = 0
        for T, tab in zip(Ts, tabs):
            nb = -(-T // (BS * 2))
            O.pack_window(src, g, tab, T, win, tok_off, w0, w1)
            tok_off += T
        tok_off = doff = 0
        for T, tab in zip(Ts, tabs):
            nb = -(-T // (BS * 2))
            O.unpack_window(win, tok_off, d1, gd, dperm[doff:doff + nb], T, w0, w1)
            tok_off += T; doff += nb
    tok_off = doff = 0
    for T, tab in zip(Ts, tabs):
        nb = -(-T // (BS * 2))
        O.unpack(full, tok_off, d2, gd, dperm[doff:doff + nb], T)
        tok_off += T; doff += nb
    assert np.array_equal(d1, d2)


def test_pack_unpack_identity_and_round_trip():
    """unpack(pack(pool,T),T) restores every named slot; transfer S->D then D->S restores src slots."""
    rng = np.random.default_rng(9)
    L, H, D, NB, BS, T = 2, 2, 8, 7, 4, 22
    g = _geom("lkbthd", L, H, D, NB, BS)
    pool = _rand_pool(rng, g.span_bytes())
    tab = rng.permutation(NB)[:6]
    staging = np.zeros(T * g.bytes_per_token, np.uint8)
    O.pack(pool, g, tab, T, staging, 0)
    back = np.full(g.span_bytes(), SENT, np.uint8)
    O.unpack(staging, 0, back, g, tab, T)
    pv, bv = Hh.logical_view(pool, "lkbthd", L, NB, BS, H, D), Hh.logical_view(back, "lkbthd", L, NB, BS, H, D)
    for t in range(T):
        assert np.array_equal(bv[:, :, tab[t // BS], t % BS], pv[:, :, tab[t // BS], t % BS])
    assert np.count_nonzero(back != SENT) <= T * g.bytes_per_token
    gd = _geom("blkhtd", L, H, D, 4, 8)
    mid = np.zeros(gd.span_bytes(), np.uint8)
    dtab = rng.permutation(4)[:3]
    O.transfer(pool, g, mid, gd, tab, dtab, T)
    again = np.full(g.span_bytes(), SENT, np.uint8)
    O.transfer(mid, gd, again, g, dtab, tab, T)
    assert np.array_equal(again, back)


# ---------------------------------------------------------------------------------------
# plan oracle: bidirectional segment alignment
# ---------------------------------------------------------------------------------------
def _expand(t):
    return list(range(*t["arange"])) if isinstance(t, dict) else t


def test_golden_alignment_fixtures():
    with open(os.path.join(GOLD, "align_examples.json")) as f:
        gold = json.load(f)
    for case in gold["cases"]:
        got = O.align(_expand(case["src"]), case["bs_src"], _expand(case["dst"]), case["bs_dst"], case["tokens"])
        assert got == [tuple(x) for x in case["expect"]], case["cite"]
        assert O.count_segments(_expand(case["src"]), case["bs_src"], _expand(case["dst"]), case["bs_dst"],
                                case["tokens"]) == len(case["expect"])
    for c in gold["blockwise_calls"]:
        assert O.blockwise_calls(c["n_blocks"], c["num_layers"]) == c["expect"], c["cite"]


def test_alignment_equals_token_level_definition_random():
    """Oracle works on granule ids; the definition is restated here on TOKEN slots.  Catches wrong
    granule scaling (BS/g), wrong gcd, missed break on one side, tail clamp."""
    rng = np.random.default_rng(10)
    for _ in range(300):
        bs_s, bs_d = (int(x) for x in rng.choice([1, 2, 4, 8, 16], size=2))
        T = int(rng.integers(0, 90))
        ns, nd = -(-T // bs_s), -(-T // bs_d)
        # tables with long-ish runs so that merges actually happen
        def tab(n):
            out, cur = [], int(rng.integers(0, 50))
            for _ in range(n):
                out.append(cur)
                cur = cur + 1 if rng.random() < 0.7 else int(rng.integers(0, 200))
            return out
        S, Dd = tab(ns), tab(nd)
        got = O.align(S, bs_s, Dd, bs_d, T)
        exp = Hh.segments_from_cuts(Hh.cuts_by_definition(S, bs_s, Dd, bs_d, T), T)
        assert got == exp
        if T:
            Hh.check_segment_invariants(got, S, bs_s, Dd, bs_d, T)
        # one-sided (pack / unpack) plans
        assert O.align(S, bs_s, None, 0, T) == Hh.segments_from_cuts(Hh.cuts_by_definition(S, bs_s, None, 0, T), T)
        assert O.align(None, 0, Dd, bs_d, T) == Hh.segments_from_cuts(Hh.cuts_by_definition(None, 0, Dd, bs_d, T), T)


def test_alignment_is_the_unique_minimal_partition_bruteforce():
    """Exhaustive: every way to cut a tiny request; the oracle's list is THE minimal legal partition
    (so 'number of segments == number of maximal consecutive-id runs', north_star)."""
    for bs_s, bs_d in [(2, 2), (2, 4), (4, 2), (1, 2)]:
        for T in (5, 8, 9):
            ns, nd = -(-T // bs_s), -(-T // bs_d)
            pool_s, pool_d = ns + 1, nd + 1
            rng = np.random.default_rng(100 + T + 10 * bs_s + bs_d)
            all_s = list(Hh.injective_tables(pool_s, ns))
            all_d = list(Hh.injective_tables(pool_d, nd))
            pick_s = [all_s[i] for i in rng.choice(len(all_s), size=min(12, len(all_s)), replace=False)]
            pick_d = [all_d[i] for i in rng.choice(len(all_d), size=min(12, len(all_d)), replace=False)]
            for S in pick_s:
                for Dd in pick_d:
                    best, parts = Hh.brute_force_min_partition(S, bs_s, Dd, bs_d, T)
                    got = O.align(list(S), bs_s, list(Dd), bs_d, T)
                    assert len(got) == best and parts == [got]


def test_random_permutation_table_gives_one_segment_per_block():
    """BASELINE.json configs[0]: run length 1 => 63 segments for 1000 tokens."""
    from paper_2504_03775_b200 import synth
    w = synth.config1_tiny()
    r = w.requests[0]
    assert O.count_segments(r.src_blocks, 16, r.dst_blocks, 16, r.num_tokens) == 63
    assert O.blockwise_calls(len(r.src_blocks), w.shape.num_layers) == 252


def test_expected_break_rate_independent_sides():
    """Independent geometric runs (mean 2 src, mean 16 dst): P(break) = 1 - (1/2)(15/16) = 0.531."""
    rng = np.random.default_rng(11)
    n = 40000

    def tab(p):
        out, cur = [], 0
        for _ in range(n):
            out.append(cur)
            cur = cur + 1 if rng.random() >= p else cur + 2 + int(rng.integers(0, 5))
        return out
    segs = O.count_segments(tab(0.5), 16, tab(1 / 16), 16, n * 16)
    assert abs(segs / n - (1 - 0.5 * 15 / 16)) < 0.01


# ---------------------------------------------------------------------------------------
# element sizes other than 2 bytes (reading A14: elements move as `elem_bytes` raw bytes; fp8 = 1, fp32 = 4)
# These reach okv_copy_elem's generic branch, which no 2-byte test touches.
# ---------------------------------------------------------------------------------------
ELEM_SIZES = [1, 4, 8]


def _geom_e(layout, L, H, D, e, NB, BS):
    return getattr(O.PoolGeom, layout)(L, H, D, e, NB, BS)


@pytest.mark.parametrize("e", ELEM_SIZES)
@pytest.mark.parametrize("layout", ["lkbthd", "blkhtd", "blkthd"])
def test_elem_sizes_same_layout_equals_numpy_fancy_indexing(e, layout):
    """numpy indexes whole `e`-byte items (uint8 / uint32 / uint64 views).  Catches: a dim stride that is not
    elem_bytes, a generic-branch copy that drops, repeats or reorders bytes of an element."""
    rng = np.random.default_rng(30 + e)
    L, H, D, NB, BS, n = 2, 3, 8, 9, 4, 5
    g = _geom_e(layout, L, H, D, e, NB, BS)
    assert g.span_bytes() == L * 2 * NB * BS * H * D * e
    src = _rand_pool(rng, g.span_bytes())
    dst = np.full(g.span_bytes(), SENT, np.uint8)
    Src, Dst = rng.permutation(NB)[:n], rng.permutation(NB)[:n]
    O.transfer(src, g, dst, g, Src, Dst, n * BS)
    exp = np.full(g.span_bytes(), SENT, np.uint8)
    ev, sv = Hh.logical_view(exp, layout, L, NB, BS, H, D, e), Hh.logical_view(src, layout, L, NB, BS, H, D, e)
    ev[:, :, Dst] = sv[:, :, Src]
    assert np.array_equal(dst, exp)


@pytest.mark.parametrize("e", ELEM_SIZES)
@pytest.mark.parametrize("bs_s,bs_d,src_layout,dst_layout,T", [
    (4, 4, "lkbthd", "blkhtd", 13), (2, 8, "lkbthd", "blkhtd", 16), (8, 2, "blkhtd", "lkbthd", 11), (4, 8, "blkthd", "blkhtd", 9)])
def test_elem_sizes_conversion_partial_block_and_untouched_bytes(e, bs_s, bs_d, src_layout, dst_layout, T):
    """Layout + block-size conversion with a partial last block, token by token in numpy item views; every other
    dst byte keeps the sentinel.  Catches: head/token transposition or tail spill that only shows at e != 2."""
    rng = np.random.default_rng(40 + e)
    L, H, D = 2, 2, 4
    ns, nd = -(-T // bs_s), -(-T // bs_d)
    NBs, NBd = ns + 2, nd + 2
    gs, gd = _geom_e(src_layout, L, H, D, e, NBs, bs_s), _geom_e(dst_layout, L, H, D, e, NBd, bs_d)
    src = _rand_pool(rng, gs.span_bytes())
    src0 = src.copy()
    dst = np.full(gd.span_bytes(), SENT, np.uint8)
    Src, Dst = rng.permutation(NBs)[:ns], rng.permutation(NBd)[:nd]
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    exp = np.full(gd.span_bytes(), SENT, np.uint8)
    ev, sv = Hh.logical_view(exp, dst_layout, L, NBd, bs_d, H, D, e), Hh.logical_view(src, src_layout, L, NBs, bs_s, H, D, e)
    for t in range(T):
        ev[:, :, Dst[t // bs_d], t % bs_d] = sv[:, :, Src[t // bs_s], t % bs_s]
    assert np.array_equal(dst, exp)
    assert np.array_equal(src, src0)


@pytest.mark.parametrize("e", ELEM_SIZES)
def test_elem_sizes_wire_format_windows_and_unpack(e):
    """Wire format A12 and layer windows A20 in `e`-byte items: pack == numpy gather, a window == the planes cut out
    of the wire format, unpack(pack) == transfer.  Catches: a bytes-per-token that assumes 2-byte elements."""
    rng = np.random.default_rng(50 + e)
    L, H, D, NB, BS = 3, 2, 4, 10, 4
    g = _geom_e("blkhtd", L, H, D, e, NB, BS)
    assert g.bytes_per_token == 2 * L * H * D * e
    src = _rand_pool(rng, g.span_bytes())
    Ts = [6, 0, 9]
    perm = rng.permutation(NB)
    tabs, off = [], 0
    for T in Ts:
        tabs.append(perm[off:off + -(-T // BS)]); off += -(-T // BS)
    sv = Hh.logical_view(src, "blkhtd", L, NB, BS, H, D, e)
    staging = np.full(sum(Ts) * g.bytes_per_token, SENT, np.uint8)
    parts, tok_off = [], 0
    for T, tab in zip(Ts, tabs):
        O.pack(src, g, tab, T, staging, tok_off)
        tok_off += T
        parts.append(sv[:, :, tab].reshape(L, 2, len(tab) * BS, H, D)[:, :, :T].reshape(-1))
    assert np.array_equal(staging.view(Hh.ELEM_DTYPE[e]), np.concatenate(parts))
    tokb = H * D * e
    w0, w1 = 1, 3
    win = np.full(sum(Ts) * 2 * (w1 - w0) * tokb, SENT, np.uint8)
    cut, tok_off = [], 0
    for T, tab in zip(Ts, tabs):
        O.pack_window(src, g, tab, T, win, tok_off, w0, w1)
        base = tok_off * g.bytes_per_token
        cut.append(staging[base + 2 * w0 * T * tokb: base + 2 * w1 * T * tokb])
        tok_off += T
    assert np.array_equal(win, np.concatenate(cut))
    gd = _geom_e("lkbthd", L, H, D, e, NB, BS * 2)
    dperm = rng.permutation(NB)
    d1, d2 = np.full(gd.span_bytes(), SENT, np.uint8), np.full(gd.span_bytes(), SENT, np.uint8)
    d3 = np.full(gd.span_bytes(), SENT, np.uint8)
    tok_off = doff = 0
    for T, tab in zip(Ts, tabs):
        nb = -(-T // (BS * 2))
        dtab = dperm[doff:doff + nb]; doff += nb
        O.unpack(staging, tok_off, d1, gd, dtab, T)
        O.transfer(src, g, d2, gd, tab, dtab, T)
        O.unpack_window(win, tok_off, d3, gd, dtab, T, w0, w1)
        tok_off += T
    assert np.array_equal(d1, d2)
    lay = gd.s_layer
    assert np.array_equal(d3[w0 * lay:w1 * lay], d2[w0 * lay:w1 * lay])
    assert np.all(d3[:w0 * lay] == SENT) and np.all(d3[w1 * lay:] == SENT)


def test_elem_size_is_only_how_a_row_is_cut_into_items():
    """The same bytes described as (Dh=16,e=1), (8,2), (4,4), (2,8) are the same rows, so every description must
    move the same bytes.  Catches: any place where elem_bytes enters other than through Dh*e."""
    rng = np.random.default_rng(60)
    L, H, NB, BS, T = 2, 3, 7, 4, 18
    outs = []
    for D, e in [(16, 1), (8, 2), (4, 4), (2, 8)]:
        gs, gd = _geom_e("lkbthd", L, H, D, e, NB, BS), _geom_e("blkhtd", L, H, D, e, NB, BS * 2)
        r = np.random.default_rng(61)
        src = _rand_pool(r, gs.span_bytes())
        Src, Dst = r.permutation(NB)[:5], r.permutation(NB)[:3]
        dst = np.full(gd.span_bytes(), SENT, np.uint8)
        O.transfer(src, gs, dst, gd, Src, Dst, T)
        outs.append(dst)
    for o in outs[1:]:
        assert np.array_equal(o, outs[0])


def test_all_256_byte_patterns_and_fp32_specials_survive():
    """Raw-bit fidelity at e = 1 (every fp8 code) and e = 4 (NaN payloads, -0, Inf, denormals as uint32)."""
    L, H, D, BS, NB = 1, 1, 16, 4, 4
    g = _geom_e("lkbthd", L, H, D, 1, NB, BS)                 # 2*4*4*16 = 512 one-byte elements
    src = np.tile(np.arange(256, dtype=np.uint8), 2)
    assert src.size == g.span_bytes()
    dst = np.zeros_like(src)
    perm = np.asarray([2, 0, 3, 1])
    O.transfer(src, g, dst, g, perm, np.arange(NB), NB * BS)
    sv, dv = Hh.logical_view(src, "lkbthd", L, NB, BS, H, D, 1), Hh.logical_view(dst, "lkbthd", L, NB, BS, H, D, 1)
    assert np.array_equal(dv, sv[:, :, perm])
    assert np.array_equal(np.sort(dst), np.sort(src))
    g4 = _geom_e("lkbthd", L, H, 4, 4, NB, BS)
    special = np.asarray([0x7FC00001, 0xFFC12345, 0x7F800000, 0xFF800000, 0x80000000, 0x00000001, 0x807FFFFF, 0x7FFFFFFF],
                         np.uint32)
    src4 = np.resize(special, g4.span_bytes() // 4).copy()
    src4[::3] ^= np.arange(src4[::3].size, dtype=np.uint32) << 8      # make rows distinguishable
    dst4 = np.zeros(g4.span_bytes(), np.uint8)
    O.transfer(src4.view(np.uint8), g4, dst4, g4, perm, np.arange(NB), NB * BS)
    s4, d4 = Hh.logical_view(src4.view(np.uint8), "lkbthd", L, NB, BS, H, 4, 4), Hh.logical_view(dst4, "lkbthd", L, NB, BS, H, 4, 4)
    assert np.array_equal(d4, s4[:, :, perm])


# ---------------------------------------------------------------------------------------
# plane windows (reading A21): the wire format cut at plane granularity
# ---------------------------------------------------------------------------------------
@pytest.mark.parametrize("layout", ["lkbthd", "blkhtd"])
def test_plane_window_equals_planes_cut_out_of_the_wire_format(layout):
    """A window [p0,p1) of planes (plane = 2*layer + kv) is numpy's gather restricted to those planes == the slab of
    planes [p0,p1) of each request's region of the (pinned) wire format; even-aligned plane windows ARE layer windows;
    unpacking disjoint plane windows rebuilds unpack of the whole.  Catches: K|V order inside a layer (plane % 2),
    a plane index not rebased to p0, a per-token size that still counts whole layers."""
    rng = np.random.default_rng(28)
    L, H, D, NB, BS = 3, 2, 8, 12, 4
    g = _geom(layout, L, H, D, NB, BS)
    src = _rand_pool(rng, g.span_bytes())
    Ts = [7, 12, 0, 5]
    perm = rng.permutation(NB)
    tabs, off = [], 0
    for T in Ts:
        nb = -(-T // BS)
        tabs.append(perm[off:off + nb]); off += nb
    tokb = H * D * 2
    sv = Hh.logical_view(src, layout, L, NB, BS, H, D).reshape(2 * L, NB, BS, H, D)      # [plane, block, token, head, dim]
    full = np.zeros(sum(Ts) * g.bytes_per_token, np.uint8)
    tok_off = 0
    for T, tab in zip(Ts, tabs):
        O.pack(src, g, tab, T, full, tok_off)
        tok_off += T
    for p0, p1 in [(0, 6), (1, 2), (1, 4), (3, 6), (5, 5), (2, 4)]:
        win = np.full(sum(Ts) * (p1 - p0) * tokb + 16, SENT, np.uint8)
        exp_parts, cut_parts, tok_off = [], [], 0
        for T, tab in zip(Ts, tabs):
            O.pack_planes(src, g, tab, T, win, tok_off, p0, p1)
            exp_parts.append(sv[p0:p1][:, tab].reshape(p1 - p0, len(tab) * BS, H, D)[:, :T].reshape(-1))
            base = tok_off * g.bytes_per_token
            cut_parts.append(full[base + p0 * T * tokb: base + p1 * T * tokb])
            tok_off += T
        body = win[:-16]
        assert np.array_equal(body.view(np.uint16), np.concatenate(exp_parts)) and np.array_equal(body, np.concatenate(cut_parts))
        assert np.all(win[-16:] == SENT)
        if p0 % 2 == 0 and p1 % 2 == 0:
            lw = np.zeros(body.size, np.uint8)
            tok_off = 0
            for T, tab in zip(Ts, tabs):
                O.pack_window(src, g, tab, T, lw, tok_off, p0 // 2, p1 // 2)
                tok_off += T
            assert np.array_equal(body, lw)
    gd = _geom("blkhtd" if layout == "lkbthd" else "lkbthd", L, H, D, NB, BS * 2)
    dperm = rng.permutation(NB)
    d1, d2 = np.full(gd.span_bytes(), SENT, np.uint8), np.full(gd.span_bytes(), SENT, np.uint8)
    for p0, p1 in [(0, 1), (1, 5), (5, 6)]:
        win = np.zeros(sum(Ts) * (p1 - p0) * tokb, np.uint8)
        tok_off = 0
        for T, tab in zip(Ts, tabs):
            O.pack_planes(src, g, tab, T, win, tok_off, p0, p1)
            tok_off += T
        tok_off = doff = 0
        for T, tab in zip(Ts, tabs):
            nb = -(-T // (BS * 2))
            O.unpack_planes(win, tok_off, d1, gd, dperm[doff:doff + nb], T, p0, p1)
            tok_off += T; doff += nb
    tok_off = doff = 0
    for T, tab in zip(Ts, tabs):
        nb = -(-T // (BS * 2))
        O.unpack(full, tok_off, d2, gd, dperm[doff:doff + nb], T)
        tok_off += T; doff += nb
    assert np.array_equal(d1, d2)


def test_golden_hand_worked_transfer_and_wire_format():
    """tests/golden/transfer_example.json: a 5-token request worked by hand (block tables [2,0,1] -> [1,0], src block 2
    LKBTHD, dst block 4 BLKHTD, partial blocks on both sides).  The offsets are evaluated here from the layout formulas
    stated in the fixture, not by the oracle or by numpy reshapes.  Catches what the numpy pins share with each other:
    a consistent misreading of an axis order."""
    with open(os.path.join(GOLD, "transfer_example.json")) as f:
        fx = json.load(f)
    L, H, D = fx["shape"]["L"], fx["shape"]["Hkv"], fx["shape"]["Dh"]
    gs = _geom("lkbthd", L, H, D, fx["src"]["num_blocks"], fx["src"]["block_size"])
    gd = _geom("blkhtd", L, H, D, fx["dst"]["num_blocks"], fx["dst"]["block_size"])
    src = np.zeros(gs.span_bytes() // 2, np.uint16)
    for c in range(2):
        for b in range(3):
            for t in range(2):
                for h in range(H):
                    off = ((c * 3 + b) * 2 + t) * 2 * 8 + h * 8
                    src[off:off + 8] = 1000 * c + 100 * b + 10 * t + h
    dst = np.full(gd.span_bytes() // 2, fx["dst"]["prefill"], np.uint16)
    rq = fx["request"]
    O.transfer(src.view(np.uint8), gs, dst.view(np.uint8), gd, rq["src_blocks"], rq["dst_blocks"], rq["num_tokens"])
    exp = np.full(dst.size, fx["expect_dst_rows"]["every_other_element"], np.uint16)
    for blk, c, h, tok, val in fx["expect_dst_rows"]["rows"]:
        off = blk * 128 + c * 64 + h * 32 + tok * 8
        exp[off:off + 8] = val
    assert np.array_equal(dst, exp)
    wire = np.full(rq["num_tokens"] * gs.bytes_per_token // 2, 65535, np.uint16)
    O.pack(src.view(np.uint8), gs, rq["src_blocks"], rq["num_tokens"], wire.view(np.uint8), 0)
    expw = np.full(wire.size, 65535, np.uint16)
    for c, t, h, val in fx["expect_wire"]["rows"]:
        off = ((c * 5 + t) * 2 + h) * 8
        expw[off:off + 8] = val
    assert np.array_equal(wire, expw)
    back = np.full(dst.size, 65535, np.uint16)
    O.unpack(wire.view(np.uint8), 0, back.view(np.uint8), gd, rq["dst_blocks"], rq["num_tokens"])
    assert np.array_equal(back, exp)


# ---------------------------------------------------------------------------------------
# reading A22: pools whose layers are separate allocations ("separate tensor structures across all layer
# dimensions" — the cache the paper starts from).  Pinned against numpy arrays that really ARE separate.
# ---------------------------------------------------------------------------------------
def _scatter_layers(rng, layers, gap=48):
    """Place separate per-layer arrays (uint8, flat) at shuffled, gapped offsets of one buffer -> (buffer, offsets)."""
    order = rng.permutation(len(layers))
    off, pos = [0] * len(layers), 16 * int(rng.integers(0, 4))
    for l in order:
        off[l] = pos
        pos += layers[l].size + 16 * int(rng.integers(1, gap // 16 + 1))
    buf = rng.integers(0, 256, size=pos, dtype=np.uint8)
    for l, a in enumerate(layers):
        buf[off[l]:off[l] + a.size] = a
    return buf, off


@pytest.mark.parametrize("e", [1, 2, 4])
@pytest.mark.parametrize("dst_separate", [False, True])
def test_separate_layer_tensors_equal_numpy_fancy_indexing_layer_by_layer(e, dst_separate):
    """Every src layer is its own [2][NB][BS][H][D] array somewhere in memory (shuffled order, gaps in between);
    the move must equal `dst_l[:, Dst] = src_l[:, Src]` for every layer separately.  Catches: a layer offset applied
    to the wrong layer, s_layer still added, K|V stride taken from the stacked pool, gaps overwritten."""
    rng = np.random.default_rng(2200 + e)
    L, H, D, NB, BS, n = 4, 2, 16 // e * 2, 7, 4, 5
    dt = Hh.ELEM_DTYPE[e]
    src_layers = [rng.integers(0, 256, size=2 * NB * BS * H * D * e, dtype=np.uint8) for _ in range(L)]
    src, soff = _scatter_layers(rng, src_layers)
    one = O.PoolGeom.lkbthd(1, H, D, e, NB, BS)                       # geometry of ONE layer tensor
    gs = O.PoolGeom(L, H, D, e, NB, BS, one.s_layer, one.s_kv, one.s_block, one.s_token, one.s_head).with_layer_offsets(soff)
    assert gs.span_bytes() <= src.size
    Src, Dst = rng.permutation(NB)[:n], rng.permutation(NB)[:n]
    T = n * BS - 3                                                    # partial last block (A4)
    if dst_separate:
        dst_layers = [np.full(2 * NB * BS * H * D * e, SENT, np.uint8) for _ in range(L)]
        dst, doff = _scatter_layers(rng, dst_layers)
        gd = O.PoolGeom(L, H, D, e, NB, BS, one.s_layer, one.s_kv, one.s_block, one.s_token, one.s_head).with_layer_offsets(doff)
    else:
        gd = O.PoolGeom.lkbthd(L, H, D, e, NB, BS)
        dst = np.full(gd.span_bytes(), SENT, np.uint8)
        doff = [l * gd.s_layer for l in range(L)]
    exp = dst.copy()
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    per_layer = 2 * NB * BS * H * D * e
    for l in range(L):
        sv = src_layers[l].view(dt).reshape(2, NB * 0 + NB, BS, H, D)
        ev = exp[doff[l]:doff[l] + per_layer].view(dt).reshape(2, NB, BS, H, D)
        full = T // BS
        ev[:, Dst[:full]] = sv[:, Src[:full]]
        ev[:, Dst[full], :T % BS] = sv[:, Src[full], :T % BS]
    assert np.array_equal(dst, exp)


def test_separate_layers_at_uniform_offsets_are_the_stacked_pool():
    """layer_off[l] = l * s_layer must give exactly what the stacked (L,2,B,H) pool gives — wire format included.
    Catches: layer_off used on one side of pack/unpack only, or ignored by the window functions."""
    rng = np.random.default_rng(2210)
    L, H, D, NB, BS, T = 3, 2, 8, 6, 4, 18
    g = _geom("lkbthd", L, H, D, NB, BS)
    gl = g.with_layer_offsets([l * g.s_layer for l in range(L)])
    src = _rand_pool(rng, g.span_bytes())
    tab = rng.permutation(NB)[:-(-T // BS)]
    a, b = np.full(T * g.bytes_per_token, SENT, np.uint8), np.full(T * g.bytes_per_token, SENT, np.uint8)
    O.pack(src, g, tab, T, a, 0)
    O.pack(src, gl, tab, T, b, 0)
    assert np.array_equal(a, b)
    wa, wb = np.full(T * 2 * 2 * H * D * 2, SENT, np.uint8), np.full(T * 2 * 2 * H * D * 2, SENT, np.uint8)
    O.pack_window(src, g, tab, T, wa, 0, 1, 3)
    O.pack_window(src, gl, tab, T, wb, 0, 1, 3)
    assert np.array_equal(wa, wb)
    da, db = np.full(g.span_bytes(), SENT, np.uint8), np.full(g.span_bytes(), SENT, np.uint8)
    O.unpack(a, 0, da, g, tab, T)
    O.unpack(a, 0, db, gl, tab, T)
    assert np.array_equal(da, db)


def test_separate_layers_into_one_block_major_tensor_is_eq5():
    """The migration Eq. 5 describes: per-layer tensors (L x [2][B][H]) -> ONE (B,L,2,H) tensor, identity
    tables: equals numpy stack + transpose.  Catches: a layer landing in another layer's slot of the block."""
    rng = np.random.default_rng(2220)
    L, H, D, NB, BS = 3, 2, 8, 5, 4
    Hbytes = BS * H * D * 2
    layers = [rng.integers(0, 256, size=2 * NB * Hbytes, dtype=np.uint8) for _ in range(L)]
    src, soff = _scatter_layers(rng, layers)
    one = O.PoolGeom.lkbthd(1, H, D, 2, NB, BS)
    gs = O.PoolGeom(L, H, D, 2, NB, BS, one.s_layer, one.s_kv, one.s_block, one.s_token, one.s_head).with_layer_offsets(soff)
    gd = _geom("blkthd", L, H, D, NB, BS)
    dst = np.full(gd.span_bytes(), SENT, np.uint8)
    ident = np.arange(NB)
    O.transfer(src, gs, dst, gd, ident, ident, NB * BS)
    exp = np.stack([a.reshape(2, NB, Hbytes) for a in layers]).transpose(2, 0, 1, 3).reshape(-1)
    assert np.array_equal(dst, exp)


@pytest.mark.parametrize("layout_in_plane", ["token_major", "head_major"])
def test_separate_k_and_v_tensors_per_layer_equal_numpy_fancy_indexing_plane_by_plane(layout_in_plane):
    """Readings A22 + A3: K and V of every layer are tensors of their own ([NB][BS][H][D] or [NB][H][BS][D]) at shuffled,
    gapped offsets; the move must equal `dst_p[Dst] = src_p[Src]` for each of the 2L planes separately.  Catches: K and
    V offsets swapped (2*l + c vs 2*c + l or l + c*L), s_kv still added on top of a plane offset, a plane offset applied
    to the neighbouring layer."""
    rng = np.random.default_rng(2230)
    L, H, D, NB, BS, n, e = 3, 2, 8, 6, 4, 4, 2
    per = NB * BS * H * D * e
    src_planes = [rng.integers(0, 256, size=per, dtype=np.uint8) for _ in range(2 * L)]
    src, soff = _scatter_layers(rng, src_planes)
    dst_planes = [np.full(per, SENT, np.uint8) for _ in range(2 * L)]
    dst, doff = _scatter_layers(rng, dst_planes)
    row = D * e
    if layout_in_plane == "token_major":
        s_head, s_token = row, H * row
        view = lambda a: a.view(np.uint16).reshape(NB, BS, H, D)
    else:
        s_token, s_head = row, BS * row
        view = lambda a: a.view(np.uint16).reshape(NB, H, BS, D).transpose(0, 2, 1, 3)
    s_block = BS * H * row
    bogus_kv, bogus_layer = 5 * per + 16, 11 * per + 32          # must not be used once plane offsets are given
    gs = O.PoolGeom(L, H, D, e, NB, BS, bogus_layer, bogus_kv, s_block, s_token, s_head).with_plane_offsets(soff)
    gd = O.PoolGeom(L, H, D, e, NB, BS, bogus_layer, bogus_kv, s_block, s_token, s_head).with_plane_offsets(doff)
    Src, Dst = rng.permutation(NB)[:n], rng.permutation(NB)[:n]
    T = n * BS - 1
    exp = dst.copy()
    O.transfer(src, gs, dst, gd, Src, Dst, T)
    full = T // BS
    for p in range(2 * L):
        sv = view(src_planes[p])
        ev = view(exp[doff[p]:doff[p] + per])
        ev[Dst[:full]] = sv[Src[:full]]
        ev[Dst[full], :T % BS] = sv[Src[full], :T % BS]
    assert np.array_equal(dst, exp)
    # the wire format sees the planes in order 2*l + c whatever their addresses are
    wire = np.full(T * gs.bytes_per_token, SENT, np.uint8)
    O.pack(src, gs, Src, T, wire, 0)
    toks = np.stack([np.concatenate([view(src_planes[p])[b] for b in Src])[:T] for p in range(2 * L)])     # [plane][t][h][d]
    assert np.array_equal(wire.view(np.uint16), toks.reshape(-1))
