"""Host logic of the product library (CPU, no device): exports, validation, alignment, schedule.

The library's segment list is compared with (i) the oracle's plan function, (ii) the test-side
definition in tests/helpers.py, (iii) the hand-worked fixtures in tests/golden/."""
import ctypes as C
import json
import os
import re

import numpy as np
import pytest

from oracle import oracle as O
from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import synth
from tests import helpers as Hh

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FAKE = 0x7F0000000000  # never dereferenced by flowkv_plan_host


def _pool(layout, L=2, H=2, D=8, NB=16, BS=4, base=FAKE, e=2):
    return F.make_pool(base, L, H, D, e, NB, BS, layout)


def _segs(plan):
    return [(s["request"], s["first_token"], s["n_tokens"]) for s in plan.segments]


def test_library_exports_every_symbol_the_header_declares():
    hdr = open(os.path.join(ROOT, "include", "flowkv.h")).read()
    declared = set(re.findall(r"FLOWKV_API\s+[\w\s\*]+?\b(flowkv_\w+)\s*\(", hdr))
    assert declared == set(F.EXPORTS), declared ^ set(F.EXPORTS)
    lib = C.CDLL(F.LIB_PATH)
    for name in declared:
        assert hasattr(lib, name), name


def test_struct_sizes_match_header_layout():
    assert C.sizeof(F.flowkv_pool) == 8 + 8 * 4 + 5 * 8 + 8          # + plane_offsets (FLOWKV_VERSION 4)
    assert F.flowkv_pool.plane_offsets.offset == 80
    assert C.sizeof(F.flowkv_request) == 32
    assert C.sizeof(F.flowkv_segment) == 40
    assert C.sizeof(F.flowkv_tuning) == 48
    assert C.sizeof(F.flowkv_plan_stats) == 9 * 8 + 16 * 4
    assert F.flowkv_plan_stats.n_flat_chunks.offset == 9 * 8 + 15 * 4


def test_named_layout_strides():
    p = _pool("lkbthd", L=32, H=8, D=128, NB=16384, BS=16)
    assert list(p.stride_bytes) == [2 * 16384 * 32768, 16384 * 32768, 32768, 2048, 256]
    q = _pool("blkhtd", L=80, H=8, D=128, NB=10, BS=64)
    assert list(q.stride_bytes) == [262144, 131072, 20971520, 256, 16384]
    # the oracle's geometry helper must agree (two independent statements of Eq. 5's two orders)
    g = O.PoolGeom.blkhtd(80, 8, 128, 2, 10, 64)
    assert [g.s_layer, g.s_kv, g.s_block, g.s_token, g.s_head] == list(q.stride_bytes)
    assert F.pool_bytes(q) == g.span_bytes()
    # blkthd = (B,L,2,H) with H untouched: a block is 2*L*BS*Hkv*Dh*e = 2 MiB at the 8B shape
    t = _pool("blkthd", L=32, H=8, D=128, NB=7, BS=16)
    assert list(t.stride_bytes) == [65536, 32768, 2 * 1024 * 1024, 2048, 256]
    gt = O.PoolGeom.blkthd(32, 8, 128, 2, 7, 16)
    assert [gt.s_layer, gt.s_kv, gt.s_block, gt.s_token, gt.s_head] == list(t.stride_bytes)


@pytest.mark.parametrize("case", json.load(open(os.path.join(ROOT, "tests", "golden", "align_examples.json")))["cases"])
def test_alignment_matches_hand_worked_fixtures(case):
    def tab(x):
        return np.arange(*x["arange"], dtype=np.int32) if isinstance(x, dict) else np.asarray(x, np.int32)
    s, d = tab(case["src"]), tab(case["dst"])
    src = _pool("lkbthd", NB=int(s.max()) + 1, BS=case["bs_src"])
    dst = _pool("lkbthd", NB=int(d.max()) + 1, BS=case["bs_dst"])
    plan = F.flowkv_plan_host(src, dst, [F.Request(case["tokens"], s, d)])
    assert [[a, n] for _, a, n in _segs(plan)] == case["expect"], case["cite"]


def test_alignment_equals_oracle_and_definition_on_random_tables():
    rng = np.random.default_rng(7)
    for it in range(300):
        bs_s, bs_d = int(2 ** rng.integers(0, 4)), int(2 ** rng.integers(0, 4))
        T = int(rng.integers(1, 60))
        ns, nd = -(-T // bs_s), -(-T // bs_d)
        NBs, NBd = ns + int(rng.integers(0, 4)), nd + int(rng.integers(0, 4))
        # tables with runs: random walk that continues +1 with probability 0.6
        def table(n, NB):
            perm = []
            free = set(range(NB))
            cur = None
            while len(perm) < n:
                if cur is not None and cur + 1 in free and rng.random() < 0.6:
                    cur = cur + 1
                else:
                    cur = int(rng.choice(sorted(free)))
                free.discard(cur)
                perm.append(cur)
            return np.asarray(perm, np.int32)
        S, D = table(ns, NBs), table(nd, NBd)
        plan = F.flowkv_plan_host(_pool("lkbthd", NB=NBs, BS=bs_s), _pool("blkhtd", NB=NBd, BS=bs_d),
                                  [F.Request(T, S, D)], F.FLOWKV_CHECK_DST_ALIAS)
        got = [(a, n) for _, a, n in _segs(plan)]
        assert got == O.align(S, bs_s, D, bs_d, T)
        assert got == Hh.segments_from_cuts(Hh.cuts_by_definition(S, bs_s, D, bs_d, T), T)
        Hh.check_segment_invariants(got, S, bs_s, D, bs_d, T)
        st = plan.stats
        assert st["n_segments"] == len(got) and st["total_tokens"] == T


def test_segment_fields_point_at_the_right_slots():
    S = np.asarray([5, 6, 7, 20, 21, 9, 3, 4], np.int32)
    D = np.asarray([0, 1], np.int32)
    plan = F.flowkv_plan_host(_pool("lkbthd", NB=32, BS=16), _pool("blkhtd", NB=2, BS=64), [F.Request(120, S, D)])
    segs = plan.segments
    assert [(s["src_block"], s["src_tok_off"], s["dst_block"], s["dst_tok_off"], s["n_tokens"]) for s in segs] == \
        [(5, 0, 0, 0, 48), (20, 0, 0, 48, 32), (9, 0, 1, 16, 16), (3, 0, 1, 32, 24)]


def test_batch_segments_never_cross_requests_and_staging_offsets():
    # request 1 continues request 0's ids on both sides: still two segments (reading A10)
    r0 = F.Request(32, np.asarray([4, 5], np.int32), np.asarray([0, 1], np.int32))
    r1 = F.Request(20, np.asarray([6, 7], np.int32), np.asarray([2, 3], np.int32))
    r2 = F.Request(0, np.zeros(0, np.int32), np.zeros(0, np.int32))
    plan = F.flowkv_plan_host(_pool("lkbthd", BS=16), _pool("lkbthd", BS=16), [r0, r2, r1])
    assert _segs(plan) == [(0, 0, 32), (2, 0, 20)]
    assert [s["staging_tok_off"] for s in plan.segments] == [0, 32]
    st = plan.stats
    assert st["n_requests"] == 3 and st["total_tokens"] == 52
    assert st["payload_bytes"] == 52 * 2 * 2 * 2 * 8 * 2 == st["staging_bytes"]


def test_config_segment_counts():
    """cfg1: permutation table => one segment per block (63); cfg2: ~208; contiguous both sides => 1."""
    w = synth.config1_tiny()
    sp = F.make_pool(FAKE, 2, 2, 64, 2, 128, 16, "lkbthd")
    plan = F.flowkv_plan_host(sp, sp, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks) for r in w.requests])
    assert plan.stats["n_segments"] == 63
    assert plan.stats["mode_transfer"] == 1 and plan.stats["mode_pack"] == 1 and plan.stats["mode_unpack"] == 1
    w = synth.config2_llama8b_13k()
    r = w.requests[0]
    s8 = F.make_pool(FAKE, 32, 8, 128, 2, 16384, 16, "lkbthd")
    d8 = F.make_pool(FAKE, 32, 8, 128, 2, 1024, 16, "lkbthd")
    plan = F.flowkv_plan_host(s8, d8, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)])
    assert plan.stats["n_segments"] == synth.n_runs(r.src_blocks) == O.count_segments(r.src_blocks, 16, r.dst_blocks, 16, 13312)
    assert plan.stats["payload_bytes"] == 1_744_830_464
    w = synth.config5_point(131072, 0)
    r = w.requests[0]
    plan = F.flowkv_plan_host(F.make_pool(FAKE, 32, 8, 128, 2, w.src.num_blocks, 16), F.make_pool(FAKE, 32, 8, 128, 2, w.dst.num_blocks, 16),
                              [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)])
    assert plan.stats["n_segments"] == 1


def test_hetero_layout_uses_rows_mode_and_chunks_cover_every_token_once():
    w = synth.config4_hetero(n_requests=3, num_layers=2)
    sp = F.make_pool(FAKE, 2, 8, 128, 2, w.src.num_blocks, 16, "lkbthd")
    dp = F.make_pool(FAKE, 2, 8, 128, 2, w.dst.num_blocks, 64, "blkhtd")
    plan = F.flowkv_plan_host(sp, dp, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks) for r in w.requests])
    st = plan.stats
    assert st["mode_transfer"] == 2          # rows
    assert st["mode_pack"] == 1              # lkbthd -> dense is contiguous
    assert st["mode_unpack"] == 2            # dense -> blkhtd is a head/token transposition
    exp = sum(O.count_segments(r.src_blocks, 16, r.dst_blocks, 64, r.num_tokens) for r in w.requests)
    assert st["n_segments"] == exp


@pytest.mark.parametrize("mutate,status", [
    (lambda s, d, r: setattr(r, "src_blocks", np.asarray([0, 1, 99], np.int32)), F.FLOWKV_ERR_BLOCK_OOB),
    (lambda s, d, r: setattr(r, "dst_blocks", np.asarray([0, -1, 2], np.int32)), F.FLOWKV_ERR_BLOCK_OOB),
    (lambda s, d, r: setattr(r, "src_blocks", np.asarray([0, 1], np.int32)), F.FLOWKV_ERR_TABLE_LEN),
    (lambda s, d, r: setattr(r, "dst_blocks", np.asarray([0, 1, 2, 3], np.int32)), F.FLOWKV_ERR_TABLE_LEN),
    (lambda s, d, r: setattr(r, "dst_blocks", np.asarray([3, 1, 3], np.int32)), F.FLOWKV_ERR_DST_ALIAS),
    (lambda s, d, r: setattr(d, "head_dim", 16), F.FLOWKV_ERR_SHAPE_MISMATCH),
    (lambda s, d, r: setattr(s, "base", FAKE + 8), F.FLOWKV_ERR_ALIGN),
    (lambda s, d, r: setattr(s, "block_size", 3), F.FLOWKV_ERR_UNSUPPORTED),
    (lambda s, d, r: setattr(s, "base", None), F.FLOWKV_ERR_INVALID_ARG),
])
def test_validation_errors(mutate, status):
    s, d = _pool("lkbthd", NB=8, BS=4), _pool("lkbthd", NB=8, BS=4)
    r = F.Request(10, np.asarray([0, 1, 2], np.int32), np.asarray([4, 5, 6], np.int32))
    mutate(s, d, r)
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_plan_host(s, d, [r], F.FLOWKV_CHECK_DST_ALIAS)
    assert ei.value.status == status, str(ei.value)
    assert F.flowkv_status_string(status) == ei.value.name


def test_row_not_multiple_of_16_bytes_is_rejected():
    with pytest.raises(F.FlowKVError) as ei:
        p = _pool("lkbthd", D=4)      # 8-byte rows
        F.flowkv_plan_host(p, p, [])
    assert ei.value.status == F.FLOWKV_ERR_ALIGN


def test_host_plan_cannot_run_and_empty_batch_is_ok():
    p = _pool("lkbthd")
    plan = F.flowkv_plan_host(p, p, [])
    assert plan.stats["n_segments"] == 0 and plan.stats["payload_bytes"] == 0
    with pytest.raises(F.FlowKVError) as ei:
        plan.transfer()
    assert ei.value.status == F.FLOWKV_ERR_UNSUPPORTED
    plan.destroy()
    plan.destroy()   # idempotent


def test_no_device_means_loud_failure_not_fallback():
    """On a machine without a GPU flowkv_plan (device variant) must fail with FLOWKV_ERR_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("has a GPU")
    p = _pool("lkbthd")
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_plan(p, p, [F.Request(4, np.asarray([0], np.int32), np.asarray([1], np.int32))])
    assert ei.value.status == F.FLOWKV_ERR_CUDA
    # the plan-free calls validate on the host first, then need a device: no silent success, no CPU path
    for call in (lambda: F.flowkv_transfer_tables(p, p, FAKE, FAKE, FAKE, 1, 1, 1, 4),
                 lambda: F.flowkv_transfer_tables_layers(p, p, FAKE, FAKE, FAKE, 1, 1, 1, 4, 0, 1),
                 lambda: F.flowkv_pack_tables(p, FAKE, FAKE, 1, 1, 4, FAKE, 1 << 20, 0, 1),
                 lambda: F.flowkv_unpack_tables(p, FAKE, FAKE, 1, 1, 4, FAKE, 1 << 20, 0, 1)):
        with pytest.raises(F.FlowKVError) as ei:
            call()
        assert ei.value.status == F.FLOWKV_ERR_CUDA
    with pytest.raises(F.FlowKVError) as ei:       # argument errors come before any device call
        F.flowkv_transfer_tables_layers(p, p, FAKE, FAKE, FAKE, 1, 1, 1, 4, 2, 1)
    assert ei.value.status == F.FLOWKV_ERR_INVALID_ARG
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_transfer_tables(p, p, FAKE, FAKE, FAKE, 1, 1, 1, 400)      # tables too short for max_tokens
    assert ei.value.status == F.FLOWKV_ERR_TABLE_LEN
    for thr in (32, 64):       # threads below the default group with the group on auto must not divide by zero
        with pytest.raises(F.FlowKVError) as ei:
            F.flowkv_transfer_tables(p, p, FAKE, FAKE, FAKE, 1, 1, 1, 4, 0, {"threads": thr})
        assert ei.value.status == F.FLOWKV_ERR_CUDA


def test_tile_schedule_respects_tile_bytes():
    s8 = F.make_pool(FAKE, 32, 8, 128, 2, 16384, 16, "lkbthd")
    d8 = F.make_pool(FAKE, 32, 8, 128, 2, 1024, 16, "lkbthd")
    w = synth.config2_llama8b_13k()
    r = w.requests[0]
    for tile in (8192, 32768, 65536):
        plan = F.flowkv_plan_host(s8, d8, [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks)], 0, {"tile_bytes": tile})
        st = plan.stats
        # every segment of n blocks (32 KiB per block-plane) needs ceil(n*32768/tile) chunks
        runs = np.diff(np.concatenate([[0], np.nonzero(np.diff(r.src_blocks) != 1)[0] + 1, [len(r.src_blocks)]]))
        assert st["n_chunks_transfer"] == int(sum(-(-int(n) * 32768 // tile) for n in runs))
        assert st["tile_bytes"] == tile and st["n_planes"] == 64


@pytest.mark.parametrize("layout", ["blkhtd", "blkthd"])
def test_block_major_pairs_use_flat_whole_block_spans(layout):
    """Both pools (B,L,2,H) with the same interior (Eq. 5): a run of n whole blocks that is
    consecutive on both sides is ONE byte range of n * 2*L*BS*Hkv*Dh*e bytes (Fig. 5); only a
    partial last block needs per-plane work.  Chunk counts follow in closed form."""
    L, H, D, BS = 4, 2, 64, 16
    blk = 2 * L * BS * H * D * 2                      # 32 KiB
    sp, dp = _pool(layout, L, H, D, 64, BS), _pool(layout, L, H, D, 64, BS)
    S = np.asarray([5, 6, 7, 8, 20, 21, 40], np.int32)
    Dt = np.asarray([0, 1, 2, 3, 4, 5, 6], np.int32)
    for T, tile in [(7 * BS, 65536), (7 * BS - 5, 65536), (7 * BS - 5, 16384), (3, 65536)]:
        nb = -(-T // BS)
        plan = F.flowkv_plan_host(sp, dp, [F.Request(T, S[:nb], Dt[:nb])], 0, {"tile_bytes": tile})
        st = plan.stats
        assert st["mode_transfer"] == 3
        segs = [(a, n) for _, a, n in _segs(plan)]
        assert segs == O.align(S[:nb], BS, Dt[:nb], BS, T)
        slots = 1                                      # an entry owns up to 32 tile slots of one range:
        while blk % tile == 0 and slots < 32 and (blk // tile) % (2 * slots) == 0:
            slots *= 2                                 # the largest power of two dividing the tiles of a block
        piece = tile * slots
        flat = sum(-(-(n // BS) * blk // piece) for _, n in segs)
        ragged = sum(1 for _, n in segs if n % BS)
        assert st["n_flat_chunks"] == flat and st["n_chunks_transfer"] == flat + ragged
    # fully contiguous on both sides, whole blocks: one segment, and 7 blocks * 32 KiB / 64 KiB tiles = 4 spans
    plan = F.flowkv_plan_host(sp, dp, [F.Request(7 * BS, np.arange(10, 17, dtype=np.int32), Dt)])
    assert plan.stats["n_segments"] == 1 and plan.stats["n_flat_chunks"] == plan.stats["n_chunks_transfer"]
    # differing interiors or block sizes are NOT flat
    other = "blkthd" if layout == "blkhtd" else "blkhtd"
    assert F.flowkv_plan_host(sp, _pool(other, L, H, D, 64, BS), [F.Request(16, S[:1], Dt[:1])]).stats["mode_transfer"] == 2
    d32 = _pool(layout, L, H, D, 64, 32)
    assert F.flowkv_plan_host(sp, d32, [F.Request(16, S[:1], Dt[:1])]).stats["mode_transfer"] == 2
    # a padded block-major pool (blocks do not abut) is not flat either
    strides = list(sp.stride_bytes)
    strides[F.LAYOUTS["strided"]] += 256            # index 2 == FLOWKV_S_BLOCK
    pad = F.make_pool(FAKE, L, H, D, 2, 64, BS, "strided", strides)
    assert F.flowkv_plan_host(pad, pad, [F.Request(16, S[:1], Dt[:1])]).stats["mode_transfer"] == 2


def test_descending_runs_never_merge_and_tile_space_limit():
    """Reading A8: ids that step by -1 are not one transfer (memory order would be reversed), so a table in
    descending order gives one segment per block.  And the documented limit: a batch whose tile space
    (schedule entries x planes) reaches 2^31 is refused with FLOWKV_ERR_UNSUPPORTED instead of overflowing the
    32-bit tile index of the kernels."""
    n = 1 << 20
    desc = np.arange(n - 1, -1, -1, dtype=np.int32)
    small = F.make_pool(FAKE, 2, 1, 8, 2, n, 1, "lkbthd")
    plan = F.flowkv_plan_host(small, small, [F.Request(4096, desc[:4096], desc[:4096])],
                              F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK)
    assert plan.stats["n_segments"] == 4096 == O.count_segments(desc[:4096], 1, desc[:4096], 1, 4096)
    plan.destroy()
    deep = F.make_pool(FAKE, 1024, 1, 8, 2, n, 1, "lkbthd")           # 2048 planes x 2^20 entries = 2^31 tiles
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_plan_host(deep, deep, [F.Request(n, desc, desc)], F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK)
    assert ei.value.status == F.FLOWKV_ERR_UNSUPPORTED
    ok = F.flowkv_plan_host(deep, deep, [F.Request(n - 1, desc[:n - 1], desc[:n - 1])],
                            F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK)
    assert ok.stats["n_chunks_transfer"] == n - 1


def test_planning_from_several_threads_at_once():
    """Header: 'distinct plans may be used from distinct threads; flowkv_last_error() is thread-local'.  ctypes
    releases the GIL during the call, so these planners really run concurrently."""
    import threading
    w = synth.config3_batched(n_requests=6, num_layers=2)
    sp = F.make_pool(FAKE, 2, 8, 128, 2, w.src.num_blocks, 16, "lkbthd")
    dp = F.make_pool(FAKE, 2, 8, 128, 2, w.dst.num_blocks, 16, "lkbthd")
    reqs = [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks) for r in w.requests]
    ref = _segs(F.flowkv_plan_host(sp, dp, reqs))
    bad = F.Request(16, np.asarray([w.src.num_blocks], np.int32), np.asarray([0], np.int32))   # BLOCK_OOB
    errors = []

    def worker(k):
        try:
            for i in range(40):
                if (i + k) % 4 == 0:
                    try:
                        F.flowkv_plan_host(sp, dp, [bad])
                        errors.append("bad request accepted")
                    except F.FlowKVError as e:
                        if e.status != F.FLOWKV_ERR_BLOCK_OOB or "src block id" not in str(e):
                            errors.append(f"wrong error text in thread {k}: {e}")
                else:
                    p = F.flowkv_plan_host(sp, dp, reqs)
                    if _segs(p) != ref:
                        errors.append(f"thread {k}: segments differ")
                    p.destroy()
        except Exception as e:  # pragma: no cover
            errors.append(repr(e))

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(6)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors[:3]


def test_header_is_plain_c_and_the_library_links_from_c(tmp_path):
    """include/flowkv.h compiles as C99 (-pedantic) and a C program reaches the planner through the ABI: the
    hand-worked example of SURVEY §8c gives (0,48,5,0) (48,32,20,3) (80,16,9,5) (96,24,3,6)."""
    import subprocess
    exe = tmp_path / "plan_host"
    src = os.path.join(ROOT, "tests", "c_abi", "plan_host.c")
    libdir = os.path.dirname(F.LIB_PATH)
    subprocess.check_call(["gcc", "-std=c99", "-pedantic", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), src,
                           "-o", str(exe), "-L", libdir, "-lflowkv", f"-Wl,-rpath,{libdir}"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=60)
    assert out.returncode == 0, out.stderr
    got = [tuple(int(x) for x in line.split()) for line in out.stdout.strip().splitlines()]
    assert got == [(0, 48, 5, 0), (48, 32, 20, 3), (80, 16, 9, 5), (96, 24, 3, 6)]


def test_bulk_variant_falls_back_when_two_ring_slots_cannot_fit_shared_memory():
    """in span mode a chunk is at least one token's plane bytes; a token of 128 KiB needs ring slots that
    do not fit 227 KB twice.  The plan must not promise a TMA launch it cannot make: it runs the register path and
    says so in stats.variant (all validation happens in flowkv_plan)."""
    big = F.make_pool(FAKE, 1, 64, 1024, 2, 8, 1, "lkbthd")          # tok_bytes = 64*1024*2 = 128 KiB
    p = F.flowkv_plan_host(big, big, [F.Request(2, np.array([0, 1], np.int32), np.array([2, 3], np.int32))], 0,
                           {"variant": "bulk"})
    assert p.stats["variant"] == F.FLOWKV_VARIANT_LDST
    small = F.make_pool(FAKE, 1, 8, 128, 2, 8, 16, "lkbthd")
    q = F.flowkv_plan_host(small, small, [F.Request(16, np.array([0], np.int32), np.array([1], np.int32))], 0,
                           {"variant": "bulk"})
    assert q.stats["variant"] == F.FLOWKV_VARIANT_BULK and q.stats["smem_bytes"] <= 227 * 1024


def test_request_batch_marshalled_once_plans_like_the_list():
    """flowkv.RequestBatch (the C array built once) gives the same plan as passing the Python requests, can be reused
    across calls, and an empty batch is fine."""
    w = synth.config3_batched(n_requests=5, num_layers=2)
    src = F.make_pool(FAKE, 2, 8, 128, 2, w.src.num_blocks, 16, "lkbthd")
    dst = F.make_pool(FAKE, 2, 8, 128, 2, w.dst.num_blocks, 16, "lkbthd")
    reqs = [F.Request(r.num_tokens, r.src_blocks, r.dst_blocks) for r in w.requests]
    batch = F.RequestBatch(reqs)
    assert len(batch) == 5
    a = F.flowkv_plan_host(src, dst, reqs, F.FLOWKV_CHECK_DST_ALIAS)
    for _ in range(3):
        b = F.flowkv_plan_host(src, dst, batch, F.FLOWKV_CHECK_DST_ALIAS)
        assert b.stats == a.stats and b.segments == a.segments
    assert F.flowkv_plan_host(src, dst, F.RequestBatch([])).stats["n_segments"] == 0
    # the schedule walks scattered batches in dst-address order, the reported segments stay in request / token order
    segs = a.segments
    assert [(s["request"], s["first_token"]) for s in segs] == sorted((s["request"], s["first_token"]) for s in segs)


def test_pools_whose_layers_are_separate_allocations_on_the_host_side():
    """flowkv_pool.plane_offsets (reading A22; `layer_offsets=` of the binding is its stacked-K|V special case; P:L98 'separate tensor structures across all layer dimensions'): the
    alignment is unchanged (layers play no part in it), a token-major pool stays in span mode, two block-major pools
    are no longer flat (a block is not one byte range), a misaligned offset is refused, the layer stride is ignored."""
    L, NB, BS = 3, 16, 4
    stab, dtab = [5, 6, 7, 1, 2], [0, 1, 2, 3, 9]
    req = [F.Request(18, stab, dtab)]
    plain = F.flowkv_plan_host(_pool("lkbthd", L=L), _pool("lkbthd", L=L), req)
    one = O.PoolGeom.lkbthd(1, 2, 8, 2, NB, BS)
    off = [4096 + one.layer_bytes(), 0, 3 * 4096 + 2 * one.layer_bytes()]            # shuffled, gapped
    sep = F.make_pool(FAKE + 65536, L, 2, 8, 2, NB, BS, "lkbthd", layer_offsets=[o - 4096 for o in off])   # negative too
    p = F.flowkv_plan_host(sep, _pool("lkbthd", L=L), req)
    assert _segs(p) == _segs(plain) and p.stats["n_segments"] == O.count_segments(stab, BS, dtab, BS, 18)
    assert p.stats["mode_transfer"] == 1 and p.stats["mode_pack"] == 1                # span: strides inside a layer decide
    assert F.pool_bytes(sep) == max(off) - 4096 + one.layer_bytes()
    # block-major + block-major would be flat; with separate layers on one side it is not
    bm = _pool("blkthd", L=L)
    assert F.flowkv_plan_host(bm, _pool("blkthd", L=L), req).stats["mode_transfer"] == 3
    bms = F.make_pool(FAKE, L, 2, 8, 2, NB, BS, "blkthd", layer_offsets=[l * bm.stride_bytes[0] for l in range(L)])
    assert F.flowkv_plan_host(bms, _pool("blkthd", L=L), req).stats["mode_transfer"] == 2
    # the layer stride is ignored (may be anything, even 0) once offsets are given
    st = list(sep.stride_bytes)
    st[0] = 0
    z = F.make_pool(FAKE, L, 2, 8, 2, NB, BS, "strided", st, layer_offsets=off)
    assert _segs(F.flowkv_plan_host(z, _pool("lkbthd", L=L), req)) == _segs(plain)
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_plan_host(F.make_pool(FAKE, L, 2, 8, 2, NB, BS, "lkbthd", layer_offsets=[0, 4104, 8192]), _pool("lkbthd", L=L), req)
    assert ei.value.status == F.FLOWKV_ERR_ALIGN and "plane offset" in str(ei.value)
    # fully separate K and V tensors per layer: 2L plane offsets; both the layer and the K|V stride are ignored
    po = [4096 * (7 * p_ % 6) + 16 * p_ for p_ in range(2 * L)]
    zz = list(sep.stride_bytes)
    zz[0] = zz[1] = 0
    kvsep = F.make_pool(FAKE, L, 2, 8, 2, NB, BS, "strided", zz, plane_offsets=po)
    pk = F.flowkv_plan_host(kvsep, _pool("lkbthd", L=L), req)
    assert _segs(pk) == _segs(plain) and pk.stats["mode_transfer"] == 1 and pk.stats["vec_bytes"] == 16
    assert F.pool_bytes(kvsep) == max(po) + O.PoolGeom.lkbthd(1, 2, 8, 2, NB, BS).plane_bytes()
    with pytest.raises(F.FlowKVError):
        F.make_pool(FAKE, L, 2, 8, 2, NB, BS, "strided", zz)                      # without offsets those strides are required
    # 32-byte vectors need 32-byte aligned offsets
    v32 = F.flowkv_plan_host(F.make_pool(FAKE, L, 2, 16, 2, NB, BS, "lkbthd", layer_offsets=[0, 1 << 20, 2 << 20]),
                             _pool("lkbthd", L=L, D=16), req)
    v16 = F.flowkv_plan_host(F.make_pool(FAKE, L, 2, 16, 2, NB, BS, "lkbthd", layer_offsets=[0, (1 << 20) + 16, 2 << 20]),
                             _pool("lkbthd", L=L, D=16), req)
    assert v32.stats["vec_bytes"] == 32 and v16.stats["vec_bytes"] == 16


def test_alignment_properties_under_hypothesis():
    """Property test (hypothesis): batches of 1-4 requests, block sizes 1-64 on each side, tables drawn as runs, two-sided
    and one-sided plans.  The library's segments == the oracle's okv_align == the test-side definition, request by
    request; segments never cross requests; staging offsets are the prefix sums of the lengths."""
    from hypothesis import given, settings, strategies as st, HealthCheck

    @st.composite
    def batches(draw):
        bs_s, bs_d = 2 ** draw(st.integers(0, 6)), 2 ** draw(st.integers(0, 6))
        lens = draw(st.lists(st.integers(0, 150), min_size=1, max_size=4))
        sides = draw(st.sampled_from(["both", "src", "dst"]))
        seed = draw(st.integers(0, 2 ** 31 - 1))
        p_cont = draw(st.sampled_from([0.0, 0.3, 0.7, 1.0]))
        return bs_s, bs_d, lens, sides, seed, p_cont

    def tables(rng, lens, bs, p_cont):
        need = [-(-t // bs) for t in lens]
        NB = sum(need) + int(rng.integers(1, 5))
        free, out, cur = np.ones(NB, bool), [], -2
        for n in need:
            tab = []
            for _ in range(n):
                if cur >= 0 and cur + 1 < NB and free[cur + 1] and rng.random() < p_cont:
                    cur += 1
                else:
                    cur = int(rng.choice(np.nonzero(free)[0]))
                free[cur] = False
                tab.append(cur)
            out.append(np.asarray(tab, np.int32))
        return out, NB

    @settings(max_examples=250, deadline=None, suppress_health_check=list(HealthCheck))
    @given(batches())
    def check(b):
        bs_s, bs_d, lens, sides, seed, p_cont = b
        rng = np.random.default_rng(seed)
        S, NBs = tables(rng, lens, bs_s, p_cont)
        D, NBd = tables(rng, lens, bs_d, p_cont)
        src = _pool("lkbthd", NB=NBs, BS=bs_s) if sides != "dst" else None
        dst = _pool("blkhtd", NB=NBd, BS=bs_d) if sides != "src" else None
        reqs = [F.Request(t, S[i] if src is not None else None, D[i] if dst is not None else None) for i, t in enumerate(lens)]
        plan = F.flowkv_plan_host(src, dst, reqs, F.FLOWKV_CHECK_DST_ALIAS if dst is not None else 0)
        segs = plan.segments
        off = 0
        for i, t in enumerate(lens):
            mine = [(s["first_token"], s["n_tokens"]) for s in segs if s["request"] == i]
            s_tab, d_tab = (S[i] if src is not None else None), (D[i] if dst is not None else None)
            exp = Hh.segments_from_cuts(Hh.cuts_by_definition(s_tab, bs_s, d_tab, bs_d, t), t) if t else []
            assert mine == exp, (b, i)
            if src is not None and dst is not None:
                assert mine == O.align(S[i], bs_s, D[i], bs_d, t)
            assert all(s["staging_tok_off"] == off for s in segs if s["request"] == i)
            off += t
        assert [s["request"] for s in segs] == sorted(s["request"] for s in segs)
        assert plan.stats["total_tokens"] == sum(lens)

    check()


def test_library_version_matches_header_and_binding():
    """flowkv_version() == FLOWKV_VERSION of include/flowkv.h == the version the ctypes struct layouts were written
    for (the binding refuses to load a library of another version: flowkv_pool grew in version 4)."""
    hdr = open(os.path.join(ROOT, "include", "flowkv.h")).read()
    v = int(re.search(r"#define FLOWKV_VERSION (\d+)", hdr).group(1))
    assert F._lib.flowkv_version() == v == F.FLOWKV_VERSION


def test_pool_from_tensors_describes_per_layer_tensors_in_place():
    """`pools.pool_from_tensors` (host part, CPU tensors stand in for device ones): base = the lowest data pointer,
    plane offsets = pointer distances in plane order 2*l + c, shape and element size from the tensors; K|V stacked per
    layer and separate K / V lists give the same kind of descriptor; the planner accepts it."""
    import torch
    from paper_2504_03775_b200 import pools as P
    L, NB, BS, H, D = 3, 6, 4, 2, 8
    layers = [torch.zeros(2, NB, BS, H, D, dtype=torch.bfloat16) for _ in range(L)]
    p = P.pool_from_tensors(layers=layers)
    base = min(t.data_ptr() for t in layers)
    per = NB * BS * H * D * 2
    assert (p.base, p.num_layers, p.num_kv_heads, p.head_dim, p.elem_bytes, p.num_blocks, p.block_size) == (base, L, H, D, 2, NB, BS)
    assert list(p._plane_offsets_keep) == [t.data_ptr() - base + c * per for t in layers for c in (0, 1)]
    ks = [torch.zeros(NB, BS, H, D, dtype=torch.float16) for _ in range(L)]
    vs = [torch.zeros(NB, BS, H, D, dtype=torch.float16) for _ in range(L)]
    q = P.pool_from_tensors(k_layers=ks, v_layers=vs)
    b2 = min(t.data_ptr() for t in ks + vs)
    assert list(q._plane_offsets_keep) == [t.data_ptr() - b2 for kv in zip(ks, vs) for t in kv]
    req = [F.Request(18, [5, 0, 1, 2, 3], [0, 1, 2, 4, 5])]
    st = F.flowkv_plan_host(q, _pool("lkbthd", L=L, H=H, D=D, NB=NB, BS=BS), req).stats
    assert st["n_segments"] == O.count_segments([5, 0, 1, 2, 3], BS, [0, 1, 2, 4, 5], BS, 18) and st["mode_transfer"] == 1
    with pytest.raises(AssertionError):
        P.pool_from_tensors(layers=[layers[0], layers[1][:, :3]])          # shapes must agree
