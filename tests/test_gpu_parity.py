"""`-m gpu` parity: the CUDA path (through the C-ABI) against the CPU oracle, bit for bit.

Sizes: small enough for the token-by-token oracle to finish in seconds, yet spanning many tiles and
ragged tails.  Full-size configs are in test_gpu_fullsize.py."""
import itertools

import numpy as np
import pytest
import torch

from oracle import oracle as O
from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import pools as P
from paper_2504_03775_b200 import synth
from tests import gpu_common as G

pytestmark = pytest.mark.gpu

TUNINGS = [
    None,
    {"variant": "ldst", "cache_hint": 1, "group_threads": 32, "threads": 128, "tile_bytes": 4096},
    {"variant": "ldst", "cache_hint": 2, "group_threads": 64, "threads": 256, "tile_bytes": 8192, "tile_order": 2},
    {"variant": "ldst", "cache_hint": 3, "threads": 512, "tile_bytes": 65536, "ctas_per_sm": 2, "plan_in_params": 1},
    {"variant": "bulk", "tile_bytes": 16384, "stages": 4, "plan_in_params": 1},
    {"variant": "bulk", "tile_bytes": 4096, "stages": 16, "ctas_per_sm": 2, "tile_order": 2},
    {"variant": "ldst", "max_sms": 3, "ctas_per_sm": 1},
]


@pytest.mark.parametrize("tuning", TUNINGS)
def test_cfg1_tiny_every_variant(tuning):
    """BASELINE.json configs[0]: 1000 tokens, permutation src table (63 segments), ragged last block."""
    w = synth.config1_tiny()
    dp, plan, _ = G.run_transfer_and_check(w, tuning)
    assert plan.stats["n_segments"] == 63


@pytest.mark.parametrize("tuning", [None, {"variant": "bulk"}])
def test_cfg2_shape_two_layers(tuning):
    """configs[1] with L=2: same tables (832 blocks, ~208 runs over a 16,384-block pool => 64-bit offsets
    inside one plane up to 512 MiB), 2 GiB src pool."""
    w = synth.config2_llama8b_13k(num_layers=2)
    G.run_transfer_and_check(w, tuning)


@pytest.mark.parametrize("tuning", [None, {"variant": "bulk", "tile_bytes": 32768}])
def test_cfg3_batched_small(tuning):
    """configs[2] scaled: 6 requests, L=2, src runs of mean 2, dst runs of mean 16, one batch, one launch."""
    w = synth.config3_batched(n_requests=6, num_layers=2)
    G.run_transfer_and_check(w, tuning)


@pytest.mark.parametrize("tuning", [None, {"cache_hint": 1, "group_threads": 32, "tile_bytes": 8192},
                                    {"tile_bytes": 131072, "threads": 512}])
def test_cfg4_hetero_layout_and_block_size(tuning):
    """configs[3] scaled: src BS16 LKBTHD -> dst BS64 BLKHTD, 3 requests, L=2; partial 64-token dst blocks."""
    w = synth.config4_hetero(n_requests=3, num_layers=2)
    assert any(r.num_tokens % 64 for r in w.requests)
    G.run_transfer_and_check(w, tuning)


@pytest.mark.parametrize("src_layout,dst_layout,bs_s,bs_d", [
    ("blkhtd", "lkbthd", 64, 16), ("blkhtd", "blkhtd", 16, 16), ("blkhtd", "blkhtd", 8, 32),
    ("lkbthd", "lkbthd", 32, 8), ("lkbthd", "blkhtd", 16, 16),
])
def test_other_layout_pairs(src_layout, dst_layout, bs_s, bs_d):
    lengths = [777, 64, 1, 300]
    w = synth.make_workload("pairs", 11, synth.Shape(3, 4, 64, "bf16"), lengths,
                            src_layout, bs_s, ("geometric", 3.0), None, dst_layout, bs_d, ("geometric", 2.0), None)
    G.run_transfer_and_check(w, None, fill="bits")


@pytest.mark.parametrize("heads,dim", [(3, 40), (5, 8), (1, 72), (7, 24)])
def test_non_power_of_two_heads_and_16_byte_rows(heads, dim):
    """Rows of 16/48/80/144 bytes and odd head counts: the 128-bit path and the generic div/mod path."""
    w = synth.make_workload("odd", 12, synth.Shape(2, heads, dim, "fp16"), [333, 17],
                            "lkbthd", 4, ("geometric", 2.0), None, "blkhtd", 8, ("contiguous",), None)
    G.run_transfer_and_check(w, None, fill="bits")
    w2 = synth.make_workload("odd2", 13, synth.Shape(2, heads, dim, "fp16"), [333, 17],
                             "lkbthd", 4, ("geometric", 2.0), None, "lkbthd", 4, ("geometric", 5.0), None)
    G.run_transfer_and_check(w2, None, fill="bits")
    G.run_transfer_and_check(w2, {"variant": "bulk"}, fill="bits")


def test_all_65536_bit_patterns_survive():
    """NaN payloads, +-Inf, -0, denormals: elements move as raw 16-bit words."""
    w = synth.make_workload("bits", 14, synth.Shape(1, 2, 64, "fp16"), [512], "lkbthd", 16, ("fixed", 1), 64,
                            "blkhtd", 32, ("contiguous",), None)
    dp = P.DevicePools(w)
    pat = torch.arange(65536, dtype=torch.int32, device="cuda").to(torch.int16)   # 65,536 distinct patterns
    nrep = dp.src_buf.numel() // 2 // 65536
    assert nrep >= 1
    dp.src_buf.view(torch.int16)[: nrep * 65536] = pat.repeat(nrep)
    src_np = P.to_numpy(dp.src_buf)
    plan = dp.plan()
    plan.transfer()
    torch.cuda.synchronize()
    exp = G.oracle_transfer(w, src_np)
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "bit patterns")


def test_brute_force_tiny_pools():
    """Every injective src table x a set of dst tables x every T in the last block, BS in {2,4}, incl.
    BS_s != BS_d and both layouts (SURVEY §8c 'everything, exhaustively')."""
    L, H, D = 2, 2, 8          # 16-byte rows
    shape = synth.Shape(L, H, D, "fp16")
    rng = np.random.default_rng(5)
    cases = 0
    for (bs_s, bs_d, lay_s, lay_d) in [(2, 2, "lkbthd", "lkbthd"), (4, 2, "lkbthd", "blkhtd"), (2, 4, "blkhtd", "lkbthd")]:
        NBs, NBd = 4, 4
        ssp, dsp = synth.PoolSpec(lay_s, bs_s, NBs), synth.PoolSpec(lay_d, bs_d, NBd)
        src_buf = P.alloc_bytes(ssp.bytes(shape))
        dst_buf = P.alloc_bytes(dsp.bytes(shape))
        P.fill_values(src_buf, "bits", "fp16", 99)
        src_np = P.to_numpy(src_buf)
        sdesc, ddesc = P.describe(ssp, shape, src_buf.data_ptr()), P.describe(dsp, shape, dst_buf.data_ptr())
        gs, gd = G.geom(ssp, shape), G.geom(dsp, shape)
        maxT = min(NBs * bs_s, NBd * bs_d, 8)
        for T in range(1, maxT + 1):
            ns, nd = -(-T // bs_s), -(-T // bs_d)
            dtabs = list(itertools.permutations(range(NBd), nd))
            for S in itertools.permutations(range(NBs), ns):
                for Dt in [dtabs[i] for i in rng.choice(len(dtabs), size=min(3, len(dtabs)), replace=False)]:
                    P.fill_sentinel(dst_buf)
                    plan = F.flowkv_plan(sdesc, ddesc, [F.Request(T, np.asarray(S, np.int32), np.asarray(Dt, np.int32))])
                    plan.transfer()
                    torch.cuda.synchronize()
                    exp = np.full(dsp.bytes(shape), P.SENTINEL_BYTE, np.uint8)
                    O.transfer(src_np, gs, exp, gd, S, Dt, T)
                    G.assert_same(P.to_numpy(dst_buf), exp, f"brute {lay_s}{bs_s}->{lay_d}{bs_d} T={T} S={S} D={Dt}")
                    assert plan.stats["n_segments"] == O.count_segments(np.asarray(S, np.int32), bs_s, np.asarray(Dt, np.int32), bs_d, T)
                    plan.destroy()
                    cases += 1
    assert cases > 500


@pytest.mark.parametrize("w_fn", [
    lambda: synth.config1_tiny(),
    lambda: synth.config4_hetero(n_requests=2, num_layers=2),
    lambda: synth.config3_batched(n_requests=4, num_layers=1),
])
@pytest.mark.parametrize("tuning", [None, {"variant": "bulk"}])
def test_pack_unpack_against_oracle_and_identity(w_fn, tuning):
    """pack == oracle pack (wire format A12); unpack == oracle unpack; unpack(pack(src)) == transfer(src)."""
    w = w_fn()
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    plan = dp.plan(0, tuning)
    nbytes = plan.stats["staging_bytes"]
    assert nbytes == w.payload_bytes
    staging = P.alloc_bytes(nbytes + 64)
    P.fill_sentinel(staging)
    n0 = F.flowkv_launch_count()
    plan.pack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() - n0 == 1
    got = P.to_numpy(staging)
    G.assert_same(got[:nbytes], G.oracle_pack(w, src_np), "pack")
    assert np.all(got[nbytes:] == P.SENTINEL_BYTE), "pack wrote past the wire size"
    plan.unpack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    via_staging = P.to_numpy(dp.dst_buf)
    G.assert_same(via_staging, G.oracle_unpack(w, got[:nbytes]), "unpack")
    G.assert_same(via_staging, G.oracle_transfer(w, src_np), "unpack(pack(src)) == transfer(src)")
    # one-sided plans reach the same bytes
    P.fill_sentinel(staging)
    p_only = F.flowkv_plan(dp.src, None, P.requests_of(w, dst=False), 0, tuning)
    p_only.pack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(staging)[:nbytes], got[:nbytes], "pack-only plan")
    with pytest.raises(F.FlowKVError):
        p_only.transfer()
    with pytest.raises(F.FlowKVError) as ei:
        plan.pack(staging.data_ptr(), nbytes - 1)
    assert ei.value.status == F.FLOWKV_ERR_STAGING_TOO_SMALL


def test_pack_to_unaligned_by_16_staging_and_mapped_pinned_host():
    """Staging at a 16-byte (not 32-byte) aligned address forces the 128-bit path; pinned host memory
    (the stand-in for the network endpoint) is written by the same kernel through UVA."""
    w = synth.config1_tiny()
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    plan = dp.plan()
    nbytes = plan.stats["staging_bytes"]
    exp = G.oracle_pack(w, src_np)
    big = P.alloc_bytes(nbytes + 64)
    off = 16 if big.data_ptr() % 32 == 0 else 0
    plan.pack(big.data_ptr() + off, nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(big)[off:off + nbytes], exp, "pack to 16-byte aligned staging")
    host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    host.fill_(P.SENTINEL_BYTE)
    plan.pack(host.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(host.numpy(), exp, "pack to pinned host")
    P.fill_sentinel(dp.dst_buf)
    plan.unpack(host.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "unpack from pinned host")


def test_round_trip_restores_source():
    """transfer(S->D) then transfer(D->S') with the tables swapped restores every named slot."""
    w = synth.config4_hetero(n_requests=2, num_layers=1)
    dp = P.DevicePools(w, fill="bits")
    dp.plan().transfer()
    back = P.alloc_bytes(w.src.bytes(w.shape))
    P.fill_sentinel(back)
    bdesc = P.describe(w.src, w.shape, back.data_ptr())
    reqs = [F.Request(r.num_tokens, r.dst_blocks, r.src_blocks) for r in w.requests]
    F.flowkv_plan(dp.dst, bdesc, reqs).transfer()
    torch.cuda.synchronize()
    src_np, back_np = P.to_numpy(dp.src_buf), P.to_numpy(back)
    # expected: sentinel everywhere except the request's token slots, which equal src (by the oracle, identity tables)
    exp = np.full(back_np.size, P.SENTINEL_BYTE, np.uint8)
    gs = G.geom(w.src, w.shape)
    for r in w.requests:
        O.transfer(src_np, gs, exp, gs, r.src_blocks, r.src_blocks, r.num_tokens)
    G.assert_same(back_np, exp, "round trip")


def test_empty_batches_launch_nothing():
    w = synth.config1_tiny()
    dp = P.DevicePools(w)
    n0 = F.flowkv_launch_count()
    for reqs in ([], [F.Request(0, np.zeros(0, np.int32), np.zeros(0, np.int32))]):
        plan = F.flowkv_plan(dp.src, dp.dst, reqs)
        plan.transfer()
        plan.pack(0, 0)
        plan.unpack(0, 0)
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() == n0
    assert np.all(P.to_numpy(dp.dst_buf) == P.SENTINEL_BYTE)


def test_shared_source_blocks_between_requests():
    """Prefix sharing (reading A9): two requests may name the same src blocks."""
    shape = synth.Shape(2, 2, 64, "fp16")
    ssp, dsp = synth.PoolSpec("lkbthd", 16, 32), synth.PoolSpec("lkbthd", 16, 32)
    r0 = synth.Request(40, np.asarray([3, 4, 9], np.int32), np.asarray([0, 1, 2], np.int32))
    r1 = synth.Request(60, np.asarray([3, 4, 20, 21], np.int32), np.asarray([10, 11, 12, 13], np.int32))
    w = synth.Workload("shared", 15, shape, ssp, dsp, [r0, r1], "uniform")
    G.run_transfer_and_check(w)


def test_non_default_stream_and_strided_pool():
    """A caller stream other than the current one, and a STRIDED pool (separate K and V tensors with padding)."""
    L, H, D, NB, BS = 2, 2, 64, 16, 8
    row, tok = D * 2, H * D * 2
    blk = BS * tok + 256          # padded blocks => not span-capable => rows mode
    kv = NB * blk + 4096
    lay = 2 * kv
    nbytes = L * lay
    src_buf, dst_buf = P.alloc_bytes(nbytes), P.alloc_bytes(nbytes)
    P.fill_values(src_buf, "bits", "fp16", 5)
    P.fill_sentinel(dst_buf)
    strides = [lay, kv, blk, tok, row]
    s = F.make_pool(src_buf.data_ptr(), L, H, D, 2, NB, BS, "strided", strides)
    d = F.make_pool(dst_buf.data_ptr(), L, H, D, 2, NB, BS, "strided", strides)
    S, Dt, T = np.asarray([5, 6, 1, 9], np.int32), np.asarray([2, 3, 4, 0], np.int32), 29
    stream = torch.cuda.Stream()
    plan = F.flowkv_plan(s, d, [F.Request(T, S, Dt)], 0, None, stream.cuda_stream)
    assert plan.stats["mode_transfer"] == 2
    plan.transfer(stream.cuda_stream)
    stream.synchronize()
    g = O.PoolGeom(L, H, D, 2, NB, BS, lay, kv, blk, tok, row)
    exp = np.full(nbytes, P.SENTINEL_BYTE, np.uint8)
    O.transfer(P.to_numpy(src_buf), g, exp, g, S, Dt, T)
    G.assert_same(P.to_numpy(dst_buf), exp, "strided pool")


def test_baselines_reach_the_same_bytes_and_count_calls():
    """Naive per-(block,layer,K|V) copies: calls == blocks*L*2; per-segment copies: segments*L*2."""
    w = synth.config1_tiny()
    dp = P.DevicePools(w)
    src_np = P.to_numpy(dp.src_buf)
    exp = G.oracle_transfer(w, src_np)
    calls = F.flowkv_baseline_blockwise(dp.src, dp.dst, dp.requests)
    torch.cuda.synchronize()
    assert calls == O.blockwise_calls(63, 2) == 252
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "blockwise baseline")
    P.fill_sentinel(dp.dst_buf)
    plan = dp.plan()
    calls = F.flowkv_baseline_segmentwise(plan)
    torch.cuda.synchronize()
    assert calls == plan.stats["n_segments"] * 4
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "segmentwise baseline")


def test_layer_range_operations():
    """flowkv_*_layers move exactly layers [l0,l1) (oracle: same loops restricted to those layers); an empty range
    launches nothing; a range outside [0,L] is rejected; the union of ranges equals the full operation."""
    w = synth.config4_hetero(n_requests=2, num_layers=5)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    gs, gd = G.geom(w.src, w.shape), G.geom(w.dst, w.shape)
    plan = dp.plan()
    nbytes = plan.stats["staging_bytes"]
    staging = P.alloc_bytes(nbytes)
    for l0, l1 in [(0, 0), (1, 3), (4, 5), (3, 3), (0, 5), (5, 5)]:
        P.fill_sentinel(dp.dst_buf)
        P.fill_sentinel(staging)
        n0 = F.flowkv_launch_count()
        F.flowkv_transfer_layers(plan, l0, l1)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if l1 > l0 else 0)
        exp = np.full(dp.dst_buf.numel(), P.SENTINEL_BYTE, np.uint8)
        for r in w.requests:
            O.transfer(src_np, gs, exp, gd, r.src_blocks, r.dst_blocks, r.num_tokens, l0, l1)
        G.assert_same(P.to_numpy(dp.dst_buf), exp, f"transfer_layers [{l0},{l1})")
        # pack / unpack of the same range through the wire format
        F.flowkv_pack_layers(plan, staging.data_ptr(), nbytes, l0, l1)
        torch.cuda.synchronize()
        exps = np.full(nbytes, P.SENTINEL_BYTE, np.uint8)
        off = 0
        for r in w.requests:
            O.pack(src_np, gs, r.src_blocks, r.num_tokens, exps, off, l0, l1)
            off += r.num_tokens
        got_s = P.to_numpy(staging)
        G.assert_same(got_s, exps, f"pack_layers [{l0},{l1})")
        P.fill_sentinel(dp.dst_buf)
        F.flowkv_unpack_layers(plan, staging.data_ptr(), nbytes, l0, l1)
        torch.cuda.synchronize()
        expu = np.full(dp.dst_buf.numel(), P.SENTINEL_BYTE, np.uint8)
        off = 0
        for r in w.requests:
            O.unpack(got_s, off, expu, gd, r.dst_blocks, r.num_tokens, l0, l1)
            off += r.num_tokens
        G.assert_same(P.to_numpy(dp.dst_buf), expu, f"unpack_layers [{l0},{l1})")
    for bad in [(2, 6), (3, 2), (6, 6)]:
        with pytest.raises(F.FlowKVError) as ei:
            F.flowkv_transfer_layers(plan, *bad)
        assert ei.value.status == F.FLOWKV_ERR_INVALID_ARG
    # union of disjoint ranges == the full transfer
    P.fill_sentinel(dp.dst_buf)
    for l0, l1 in [(3, 5), (0, 1), (1, 3)]:
        F.flowkv_transfer_layers(plan, l0, l1)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "union of layer ranges")


@pytest.mark.parametrize("n_chunks,ctas", [(0, 0), (1, 4), (3, 1), (100, 64)])
def test_transfer_via_pinned_host_pipeline(n_chunks, ctas):
    """pool -> pinned host -> pool with the two directions pipelined over layer chunks on two streams:
    dst == oracle transfer, host buffer == oracle pack, caller's stream order is enough to see both."""
    w = synth.config3_batched(n_requests=3, num_layers=6)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    stream = torch.cuda.Stream()
    plan = dp.plan(F.FLOWKV_PLAN_NO_TRANSFER, None, stream.cuda_stream)
    nbytes = plan.stats["staging_bytes"]
    host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    host.fill_(P.SENTINEL_BYTE)
    n0 = F.flowkv_launch_count()
    F.flowkv_transfer_via_host(plan, host.data_ptr(), nbytes, n_chunks, ctas, stream.cuda_stream)
    stream.synchronize()
    chunks = min(n_chunks, 6) if n_chunks else 6          # auto = min(L, 16)
    assert F.flowkv_launch_count() - n0 == 2 * chunks
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "via host: dst")
    G.assert_same(host.numpy(), G.oracle_pack(w, src_np), "via host: wire bytes")
    plan.destroy()


@pytest.mark.parametrize("layout", ["blkhtd", "blkthd"])
@pytest.mark.parametrize("tuning", [None, {"tile_bytes": 4096, "threads": 128, "group_threads": 32},
                                    {"tile_bytes": 16384, "ctas_per_sm": 1, "max_sms": 2, "cache_hint": 1},
                                    {"tile_order": 2, "group_threads": 64, "threads": 256},
                                    {"variant": "bulk"}, {"variant": "bulk", "tile_bytes": 4096, "stages": 3, "max_sms": 2,
                                                          "ctas_per_sm": 1, "plan_in_params": 1}])
def test_flat_mode_block_major_both_sides(layout, tuning):
    """S§8f NEXT-2 / Eq. 5 / Fig. 5: both pools (B,L,2,H) with the same interior.  Whole-block runs move as
    plane-free byte ranges, partial last blocks token-granular (A4) — all in ONE launch, bit-exact incl.
    the sentinel bytes of every untouched slot."""
    lengths = [777, 64, 1, 300, 16, 15, 0, 17]
    w = synth.make_workload("flat", 31, synth.Shape(3, 4, 64, "bf16"), lengths,
                            layout, 16, ("geometric", 3.0), None, layout, 16, ("geometric", 2.0), None)
    dp, plan, _ = G.run_transfer_and_check(w, tuning, fill="bits")
    st = plan.stats
    assert st["mode_transfer"] == 3 and st["n_flat_chunks"] > 0
    assert st["n_chunks_transfer"] - st["n_flat_chunks"] >= sum(1 for t in lengths if t % 16)
    assert st["variant"] == (F.FLOWKV_VARIANT_BULK if tuning and tuning.get("variant") == "bulk" else F.FLOWKV_VARIANT_LDST)


@pytest.mark.parametrize("upload", [0, 1])
def test_flat_mode_layer_ranges_and_pack_unpack(upload):
    """Layer-range launches of a flat plan fall back to its rows schedule; pack/unpack of block-major pools go
    through the dense wire format as before."""
    w = synth.make_workload("flatL", 32, synth.Shape(5, 2, 64, "fp16"), [100, 33, 48],
                            "blkthd", 16, ("geometric", 2.0), None, "blkthd", 16, ("contiguous",), None)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    gs, gd = G.geom(w.src, w.shape), G.geom(w.dst, w.shape)
    plan = dp.plan(0, {"plan_in_params": upload})
    assert plan.stats["mode_transfer"] == 3 and (plan.stats["plan_device_bytes"] > 0) == bool(upload)
    for l0, l1 in [(1, 3), (0, 5), (4, 5), (2, 2)]:
        P.fill_sentinel(dp.dst_buf)
        n0 = F.flowkv_launch_count()
        F.flowkv_transfer_layers(plan, l0, l1)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if l1 > l0 else 0)
        exp = np.full(dp.dst_buf.numel(), P.SENTINEL_BYTE, np.uint8)
        for r in w.requests:
            O.transfer(src_np, gs, exp, gd, r.src_blocks, r.dst_blocks, r.num_tokens, l0, l1)
        G.assert_same(P.to_numpy(dp.dst_buf), exp, f"flat plan, layers [{l0},{l1})")
    nbytes = plan.stats["staging_bytes"]
    staging = P.alloc_bytes(nbytes)
    plan.pack(staging.data_ptr(), nbytes)
    P.fill_sentinel(dp.dst_buf)
    plan.unpack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(staging), G.oracle_pack(w, src_np), "pack from blkthd")
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "unpack into blkthd")


@pytest.mark.parametrize("src_layout,dst_layout", [("lkbthd", "blkthd"), ("blkthd", "lkbthd"), ("blkthd", "blkhtd")])
def test_eq5_whole_pool_reorder(src_layout, dst_layout):
    """Eq. 5 as an operation: the whole pool re-ordered (L,2,B,H) <-> (B,L,2,H) with identity
    tables, one launch."""
    NB, BS = 24, 16
    ident = np.arange(NB, dtype=np.int32)
    shape = synth.Shape(4, 4, 64, "bf16")
    w = synth.Workload("eq5", 33, shape, synth.PoolSpec(src_layout, BS, NB), synth.PoolSpec(dst_layout, BS, NB),
                       [synth.Request(NB * BS, ident, ident)])
    G.run_transfer_and_check(w, None, fill="bits")


def test_baselines_on_block_major_pools_count_calls():
    """(B,L,2,H) pools: blockwise = one copy per whole block, segmentwise = one per segment (Fig. 5),
    plus per-plane copies for the partial last block; both reach the oracle's bytes."""
    L = 3
    w = synth.make_workload("bm_base", 34, synth.Shape(L, 2, 64, "fp16"), [16 * 9 + 5, 32],
                            "blkthd", 16, ("geometric", 3.0), None, "blkthd", 16, ("contiguous",), None)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    exp = G.oracle_transfer(w, src_np)
    calls = F.flowkv_baseline_blockwise(dp.src, dp.dst, dp.requests)
    torch.cuda.synchronize()
    assert calls == (9 + 2) + 2 * L
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "blockwise baseline, block-major")
    P.fill_sentinel(dp.dst_buf)
    plan = dp.plan()
    calls = F.flowkv_baseline_segmentwise(plan)
    torch.cuda.synchronize()
    segs = plan.segments
    assert calls == sum(1 for sg in segs if sg["n_tokens"] >= 16) + 2 * L
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "segmentwise baseline, block-major")


@pytest.mark.parametrize("n_blocks", [15, 16, 17, 95, 96, 97, 255, 256, 257, 511, 512, 513])
@pytest.mark.parametrize("variant", ["ldst", "bulk"])
def test_small_plans_travel_in_kernel_params(n_blocks, variant):
    """Step a4 'kernel params when small': a plan whose schedules have <= 512 entries is never uploaded
    (plan_device_bytes == 0) — transfer, pack and unpack read their entries from the parameter space, in the
    smallest of four forms (16 / 96 / 256 / 512 entries) that holds them; one entry more and the plan is uploaded
    as usual.  Both sides of every form boundary; same bytes either way."""
    T = n_blocks * 16 - 3
    w = synth.make_workload("inparams", 35, synth.Shape(2, 2, 64, "fp16"), [T],
                            "lkbthd", 16, ("permutation",), 1024, "lkbthd", 16, ("contiguous",), 600, "uniform")
    tuning = {"variant": variant, "tile_bytes": 4096}
    dp, plan, exp = G.run_transfer_and_check(w, tuning, fill="bits")
    st = plan.stats
    if st["n_chunks_transfer"] == n_blocks:          # the seeded permutation had no accidental +1 neighbours
        assert (st["plan_device_bytes"] == 0) == (n_blocks <= 512)
    src_np = P.to_numpy(dp.src_buf)
    nbytes = st["staging_bytes"]
    staging = P.alloc_bytes(nbytes)
    plan.pack(staging.data_ptr(), nbytes)
    P.fill_sentinel(dp.dst_buf)
    plan.unpack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(staging), G.oracle_pack(w, src_np), "pack")
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "unpack")
    forced = dp.plan(0, dict(tuning, plan_in_params=1))
    assert forced.stats["plan_device_bytes"] > 0
    P.fill_sentinel(dp.dst_buf)
    forced.transfer()
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "uploaded plan")


@pytest.mark.parametrize("w_fn", [
    lambda: synth.config3_batched(n_requests=3, num_layers=5),
    lambda: synth.config4_hetero(n_requests=2, num_layers=5),
])
def test_layer_window_pack_unpack(w_fn):
    """flowkv_pack_window / flowkv_unpack_window: a window holds only layers [l0,l1) as a self-contained dense
    message == those planes cut out of the oracle's wire format; unpacking the windows one by one rebuilds the
    oracle's transfer; bytes past the window are untouched; a short buffer is rejected."""
    w = w_fn()
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    full = G.oracle_pack(w, src_np)
    plan = dp.plan(F.FLOWKV_PLAN_NO_TRANSFER)
    L = w.shape.num_layers
    assert F.flowkv_window_bytes(plan, 0, L) == plan.stats["staging_bytes"]
    P.fill_sentinel(dp.dst_buf)
    for l0, l1 in [(0, 2), (2, 3), (3, 5), (4, 4)]:
        nb = F.flowkv_window_bytes(plan, l0, l1)
        assert nb == w.total_tokens * 2 * (l1 - l0) * w.shape.num_kv_heads * w.shape.head_dim * 2
        win = P.alloc_bytes(nb + 64)
        P.fill_sentinel(win)
        n0 = F.flowkv_launch_count()
        F.flowkv_pack_window(plan, win.data_ptr(), nb, l0, l1)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if l1 > l0 else 0)
        got = P.to_numpy(win)
        G.assert_same(got[:nb], G.oracle_pack_window(w, src_np, l0, l1), f"pack_window [{l0},{l1})")
        assert np.array_equal(got[:nb], G.window_of(full, w, l0, l1))
        assert np.all(got[nb:] == P.SENTINEL_BYTE)
        F.flowkv_unpack_window(plan, win.data_ptr(), nb, l0, l1)
        if nb:
            with pytest.raises(F.FlowKVError) as ei:
                F.flowkv_pack_window(plan, win.data_ptr(), nb - 1, l0, l1)
            assert ei.value.status == F.FLOWKV_ERR_STAGING_TOO_SMALL
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "windows [0,2)+[2,3)+[3,5) unpacked == transfer")
    with pytest.raises(F.FlowKVError):
        F.flowkv_window_bytes(plan, 3, 6)


@pytest.mark.parametrize("small", [False, True])
@pytest.mark.parametrize("n_chunks,ctas", [(0, 0), (1, 0), (4, 8), (6, 0), (9, 4), (100, 0)])
def test_transfer_via_pinned_host_with_copy_engines(n_chunks, ctas, small):
    """Copy-engine mode of flowkv_transfer_via_host: pack_window -> D2H memcpy -> H2D memcpy -> unpack_window per
    layer chunk through caller-provided device scratch.  dst == oracle transfer; the host buffer holds the chunks
    back to back, each == its layer window of the oracle's wire format."""
    L = 6
    if small:      # a plan small enough to ride in the kernel parameters (no upload)
        w = synth.make_workload("via_small", 37, synth.Shape(L, 2, 64, "fp16"), [200, 90],
                                "lkbthd", 16, ("geometric", 2.0), None, "blkhtd", 32, ("contiguous",), None)
    else:
        w = synth.config3_batched(n_requests=3, num_layers=L)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    stream = torch.cuda.Stream()
    plan = dp.plan(F.FLOWKV_PLAN_NO_TRANSFER, None, stream.cuda_stream)
    assert (plan.stats["plan_device_bytes"] == 0) == small
    nbytes = plan.stats["staging_bytes"]
    host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    host.fill_(P.SENTINEL_BYTE)
    sb = F.flowkv_via_host_scratch_bytes(plan, n_chunks)
    scratch = P.alloc_bytes(sb)
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_transfer_via_host(plan, host.data_ptr(), nbytes, n_chunks, ctas, stream.cuda_stream, scratch.data_ptr(), sb - 1)
    assert ei.value.status == F.FLOWKV_ERR_STAGING_TOO_SMALL
    n0 = F.flowkv_launch_count()
    F.flowkv_transfer_via_host(plan, host.data_ptr(), nbytes, n_chunks, ctas, stream.cuda_stream, scratch.data_ptr(), sb)
    stream.synchronize()
    launched = F.flowkv_launch_count() - n0
    if n_chunks:
        chunks = min(n_chunks, 2 * L)                                  # clamped to one chunk per plane
    else:       # default: the divisor of 2L nearest sqrt(payload / 400 KB) on a log scale, within [4, 64] (flowkv.h)
        target = min(64.0, max(4.0, np.sqrt(nbytes / 400e3)))
        cands = [d for d in range(min(2 * L, 4), min(2 * L, 64) + 1) if (2 * L) % d == 0]
        chunks = min(cands, key=lambda d: abs(np.log(d / target)))
    assert launched == 2 * chunks
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "via host (copy engines): dst")
    if chunks <= L:       # layer windows (A20)
        exp_host = np.concatenate([G.oracle_pack_window(w, src_np, L * c // chunks, L * (c + 1) // chunks) for c in range(chunks)])
    else:                 # more chunks than layers: plane windows (A21), the oracle's okv_pack_planes
        exp_host = np.concatenate([G.oracle_pack_planes(w, src_np, 2 * L * c // chunks, 2 * L * (c + 1) // chunks)
                                   for c in range(chunks)])
    G.assert_same(host.numpy(), exp_host, "via host (copy engines): chunked wire bytes")
    plan.destroy()


def test_peer_pool_over_cuda_ipc():
    """NEXT-3 / P:L90 'IPC' mode: the dst pool belongs to ANOTHER process (the decode side); this process maps it
    through CUDA IPC and flowkv_transfer stores straight into it — a one-sided put, one launch.  The owner then
    reads its own pool back and it must equal the oracle over every byte."""
    import queue
    import torch.multiprocessing as mp
    from paper_2504_03775_b200 import peer
    from tests import peer_child

    w = synth.config4_hetero(n_requests=2, num_layers=2)
    nbytes = w.dst.bytes(w.shape)
    ctx = mp.get_context("spawn")
    to_parent, to_child = ctx.Queue(), ctx.Queue()
    child = ctx.Process(target=peer_child.decode_side, args=(nbytes, P.SENTINEL_BYTE, to_parent, to_child), daemon=True)
    child.start()
    try:
        try:
            kind, handle = to_parent.get(timeout=180)
        except queue.Empty:
            pytest.skip("decode-side process did not come up")
        if kind == "error":
            pytest.skip(f"CUDA IPC export unavailable here: {handle}")
        try:
            remote = peer.import_pool(handle)
        except RuntimeError as e:
            pytest.skip(f"CUDA IPC import unavailable here: {e}")
        assert remote.numel() == nbytes
        src_buf = P.alloc_bytes(w.src.bytes(w.shape))
        P.fill_values(src_buf, "bits", w.shape.dtype, w.seed)
        src = P.describe(w.src, w.shape, src_buf.data_ptr())
        dst = P.describe(w.dst, w.shape, remote.data_ptr())           # the peer's memory
        n0 = F.flowkv_launch_count()
        plan = F.flowkv_plan(src, dst, P.requests_of(w), F.FLOWKV_CHECK_DST_ALIAS)
        plan.transfer()
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == 1
        to_child.put("written")
        kind, blob = to_parent.get(timeout=180)
        assert kind == "bytes", blob
        got = np.frombuffer(blob, dtype=np.uint8)
        G.assert_same(got, G.oracle_transfer(w, P.to_numpy(src_buf)), "peer pool over CUDA IPC")
        plan.destroy()
        del remote
        to_child.put("done")
        child.join(timeout=60)
    finally:
        if child.is_alive():
            child.kill()


@pytest.mark.parametrize("upload", [0, 1])
def test_transfer_is_cuda_graph_capturable(upload):
    """A built plan's transfer is one kernel launch and nothing else, so it can be captured into a CUDA graph and
    replayed (launch-bound small transfers: replay costs one graph launch).  Replays reach the oracle's bytes."""
    w = synth.config1_tiny()
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    stream = torch.cuda.Stream()
    plan = dp.plan(F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK, {"plan_in_params": upload}, stream.cuda_stream)
    stream.synchronize()                      # the plan upload (if any) is done before capture begins
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        plan.transfer(torch.cuda.current_stream().cuda_stream)
    exp = G.oracle_transfer(w, src_np)
    for _ in range(3):
        P.fill_sentinel(dp.dst_buf)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        G.assert_same(P.to_numpy(dp.dst_buf), exp, "graph replay")
    del g
    plan.destroy()


@pytest.mark.parametrize("layouts", [("lkbthd", "lkbthd"), ("lkbthd", "blkhtd"), ("blkthd", "blkthd")])
@pytest.mark.parametrize("tuning", [None, {"variant": "bulk"}, {"plan_in_params": 1, "tile_bytes": 4096}])
def test_guard_bands_around_both_pools_stay_intact(layouts, tuning):
    """Own bounds check (compute-sanitizer is installed but refused on the pool's boxes — exit code 86, "closed on this
    pool and stays closed", profiles/r03_sanitizer.md): each pool sits between two 64 KiB guard
    bands inside one allocation, the request names the FIRST and the LAST block of both pools and ends in a partial
    block; after transfer, pack and unpack every guard byte still holds its sentinel and dst == oracle."""
    GUARD = 64 << 10
    shape = synth.Shape(3, 2, 64, "fp16")
    NB, BS, T = 12, 16, 5 * 16 + 7
    stab = np.asarray([NB - 1, 0, 1, 5, 6, NB - 2], np.int32)
    dtab = np.asarray([0, NB - 2, NB - 1, 3, 4, 7], np.int32)
    ssp, dsp = synth.PoolSpec(layouts[0], BS, NB), synth.PoolSpec(layouts[1], BS, NB)
    w = synth.Workload("guard", 36, shape, ssp, dsp, [synth.Request(T, stab, dtab)])
    sbytes, dbytes = ssp.bytes(shape), dsp.bytes(shape)
    sbig, dbig = P.alloc_bytes(sbytes + 2 * GUARD), P.alloc_bytes(dbytes + 2 * GUARD)
    P.fill_sentinel(sbig)
    P.fill_sentinel(dbig)
    src_buf, dst_buf = sbig[GUARD:GUARD + sbytes], dbig[GUARD:GUARD + dbytes]
    P.fill_values(src_buf, "bits", "fp16", 36)
    src_np = P.to_numpy(src_buf)
    src = P.describe(ssp, shape, src_buf.data_ptr())
    dst = P.describe(dsp, shape, dst_buf.data_ptr())
    plan = F.flowkv_plan(src, dst, P.requests_of(w), F.FLOWKV_CHECK_DST_ALIAS, tuning)
    nbytes = plan.stats["staging_bytes"]
    stg_big = P.alloc_bytes(nbytes + 2 * GUARD)
    P.fill_sentinel(stg_big)
    plan.transfer()
    torch.cuda.synchronize()
    exp = G.oracle_transfer(w, src_np)
    G.assert_same(P.to_numpy(dst_buf), exp, "guarded transfer")
    plan.pack(stg_big.data_ptr() + GUARD, nbytes)
    P.fill_sentinel(dst_buf)
    plan.unpack(stg_big.data_ptr() + GUARD, nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dst_buf), exp, "guarded unpack(pack)")
    for name, big, n in (("src", sbig, sbytes), ("dst", dbig, dbytes), ("staging", stg_big, nbytes)):
        b = P.to_numpy(big)
        assert np.all(b[:GUARD] == P.SENTINEL_BYTE), f"{name}: bytes below the buffer were written"
        assert np.all(b[GUARD + n:] == P.SENTINEL_BYTE), f"{name}: bytes above the buffer were written"
    G.assert_same(P.to_numpy(src_buf), src_np, "src unchanged")


def test_launch_and_api_call_accounting():
    """SURVEY §8d 'launch accounting': a whole step (plan + transfer + destroy) of a small plan is ONE stream
    call — the launch; an uploaded plan adds allocation, upload, event record + wait and the stream-ordered free."""
    w = synth.config1_tiny()
    dp = P.DevicePools(w)
    xfer_only = F.FLOWKV_PLAN_NO_PACK | F.FLOWKV_PLAN_NO_UNPACK
    for upload, expect in ((0, 1), (1, 6)):
        c0, n0 = F.flowkv_api_call_count(), F.flowkv_launch_count()
        plan = dp.plan(xfer_only, {"plan_in_params": upload})
        plan.transfer()
        plan.destroy()
        assert F.flowkv_launch_count() - n0 == 1
        assert F.flowkv_api_call_count() - c0 == expect
    torch.cuda.synchronize()
    # the naive scheme: one call per block per layer per K|V
    c0 = F.flowkv_api_call_count()
    calls = F.flowkv_baseline_blockwise(dp.src, dp.dst, dp.requests)
    torch.cuda.synchronize()
    assert F.flowkv_api_call_count() - c0 == calls == 252


def test_product_path_from_plain_c_without_torch(tmp_path):
    """tests/c_abi/transfer_gpu.c: cudaMalloc'd pools, flowkv_plan + flowkv_transfer from C on its own stream, the
    whole dst pool against the oracle's C function — no Python, no torch in that process.  One launch."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    exe = tmp_path / "transfer_gpu"
    libdir, odir = os.path.dirname(F.LIB_PATH), os.path.join(root, "oracle")
    O.build()
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(root, "include"), "-I", f"{cuda}/include",
                           os.path.join(root, "tests", "c_abi", "transfer_gpu.c"), "-o", str(exe),
                           "-L", libdir, "-lflowkv", "-L", odir, "-lflowkv_oracle", "-L", f"{cuda}/lib64", "-lcudart",
                           f"-Wl,-rpath,{libdir}", f"-Wl,-rpath,{odir}", f"-Wl,-rpath,{cuda}/lib64"])
    out = subprocess.run([str(exe)], capture_output=True, text=True, timeout=120)
    assert out.returncode == 0, out.stderr + out.stdout
    assert out.stdout.strip() == "ok 1"


def test_table_driven_transfer_graph_replay_and_error_flag():
    """flowkv_transfer_tables captured ONCE in a CUDA graph; between replays only the CONTENTS of the device tables
    and lengths change (new requests, new block ids) and every replay lands where the oracle says.  A block id
    outside the pool raises the device error flag, skips that tile and touches nothing else."""
    shape = synth.Shape(3, 2, 64, "fp16")
    NBs, NBd, n_req, max_t = 64, 40, 3, 150
    ssp, dsp = synth.PoolSpec("lkbthd", 16, NBs), synth.PoolSpec("blkhtd", 32, NBd)
    src_buf, dst_buf = P.alloc_bytes(ssp.bytes(shape)), P.alloc_bytes(dsp.bytes(shape))
    P.fill_values(src_buf, "bits", "fp16", 41)
    src_np = P.to_numpy(src_buf)
    src, dst = P.describe(ssp, shape, src_buf.data_ptr()), P.describe(dsp, shape, dst_buf.data_ptr())
    gs, gd = G.geom(ssp, shape), G.geom(dsp, shape)
    ws, wd = -(-max_t // 16), -(-max_t // 32)
    st = torch.full((n_req, ws), -1, dtype=torch.int32, device="cuda")
    dt = torch.full((n_req, wd), -1, dtype=torch.int32, device="cuda")
    lens = torch.zeros(n_req, dtype=torch.int32, device="cuda")
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    stream = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), n_req, ws, wd, max_t,
                                 flag.data_ptr(), None, torch.cuda.current_stream().cuda_stream)
    rng = np.random.default_rng(42)
    for it in range(4):
        Ts = [int(rng.integers(0, max_t + 1)) for _ in range(n_req)]
        sperm, dperm = rng.permutation(NBs).astype(np.int32), rng.permutation(NBd).astype(np.int32)
        reqs, so, do = [], 0, 0
        hs, hd = np.full((n_req, ws), -1, np.int32), np.full((n_req, wd), -1, np.int32)
        for i, t in enumerate(Ts):
            a, b = sperm[so:so + -(-t // 16)], dperm[do:do + -(-t // 32)]
            so, do = so + len(a), do + len(b)
            hs[i, :len(a)], hd[i, :len(b)] = a, b
            reqs.append((t, a, b))
        st.copy_(torch.from_numpy(hs)); dt.copy_(torch.from_numpy(hd)); lens.copy_(torch.tensor(Ts, dtype=torch.int32))
        P.fill_sentinel(dst_buf)
        torch.cuda.synchronize()
        g.replay()
        torch.cuda.synchronize()
        exp = np.full(dsp.bytes(shape), P.SENTINEL_BYTE, np.uint8)
        for t, a, b in reqs:
            O.transfer(src_np, gs, exp, gd, a, b, t)
        G.assert_same(P.to_numpy(dst_buf), exp, f"graph replay {it} with new tables {Ts}")
        assert int(flag.item()) == 0
    # an id outside the pool: flagged, its tiles skipped, the rest of the batch still lands
    bad = hs.copy()
    victim = next(i for i, t in enumerate(Ts) if t > 0)
    bad[victim, 0] = NBs + 5
    st.copy_(torch.from_numpy(bad))
    P.fill_sentinel(dst_buf)
    torch.cuda.synchronize()
    g.replay()
    torch.cuda.synchronize()
    assert int(flag.item()) == 1
    exp = np.full(dsp.bytes(shape), P.SENTINEL_BYTE, np.uint8)
    for i, (t, a, b) in enumerate(reqs):
        if i != victim:
            O.transfer(src_np, gs, exp, gd, a, b, t)
    got = P.to_numpy(dst_buf)
    # every byte outside the victim's dst blocks is exactly the oracle's; inside them only tokens >= 16 may be written
    blk = 32 * shape.bytes_per_token
    mask = np.ones(got.size, bool)
    for b in reqs[victim][2]:
        mask[int(b) * blk:(int(b) + 1) * blk] = False
    assert np.array_equal(got[mask], exp[mask])
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), n_req, ws - 1, wd, max_t)
    assert ei.value.status == F.FLOWKV_ERR_TABLE_LEN


# ---------------------------------------------------------------------------------------------------------
# round 2: element sizes other than 2 bytes, table-driven layer ranges, the allocator wired through to bytes
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype,dim", [("fp8", 128), ("fp32", 64), ("fp8", 16), ("fp32", 12)])
@pytest.mark.parametrize("pair", [("lkbthd", 16, "lkbthd", 16), ("lkbthd", 16, "blkhtd", 64), ("blkthd", 16, "blkthd", 16)])
def test_one_and_four_byte_elements_every_operation(dtype, dim, pair):
    """fp8 KV (Llama-3-8B heads: rows of 128 B, the 256-bit path at 4 vectors per row; and 16-B rows) and fp32:
    planned transfer, pack / unpack, layer windows and the table-driven kernel against the oracle run with the
    same elem_bytes (its generic element copy, pinned in tests/test_oracle_pins.py)."""
    sl, sbs, dl, dbs = pair
    shape = synth.Shape(3, 8, dim, dtype)
    assert shape.elem_bytes in (1, 4)
    w = synth.make_workload(f"{dtype}_{sl}{sbs}_{dl}{dbs}", 777, shape, [333, 0, 1000, 17],
                            sl, sbs, ("geometric", 3.0), None, dl, dbs, ("geometric", 8.0), None)
    dp, plan, exp = G.run_transfer_and_check(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    nbytes = plan.stats["staging_bytes"]
    assert nbytes == w.total_tokens * 2 * 3 * 8 * dim * shape.elem_bytes
    staging = P.alloc_bytes(nbytes)
    P.fill_sentinel(dp.dst_buf)
    plan.pack(staging.data_ptr(), nbytes)
    plan.unpack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(staging), G.oracle_pack(w, src_np), "wire bytes")
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "unpack")
    wb = F.flowkv_window_bytes(plan, 1, 3)
    win = P.alloc_bytes(wb)
    F.flowkv_pack_window(plan, win.data_ptr(), wb, 1, 3)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(win), G.oracle_pack_window(w, src_np, 1, 3), "window [1,3)")
    # table-driven, same bytes
    P.fill_sentinel(dp.dst_buf)
    st, dt, lens, ws, wd, max_t = _padded_tables(w)
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    F.flowkv_transfer_tables(dp.src, dp.dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), len(w.requests), ws, wd, max_t,
                             flag.data_ptr())
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "table-driven")
    assert int(flag.item()) == 0


def _padded_tables(w):
    n = len(w.requests)
    max_t = max(r.num_tokens for r in w.requests)
    ws, wd = max(1, -(-max_t // w.src.block_size)), max(1, -(-max_t // w.dst.block_size))
    hs, hd = np.full((n, ws), -3, np.int32), np.full((n, wd), -3, np.int32)
    for i, r in enumerate(w.requests):
        hs[i, :len(r.src_blocks)], hd[i, :len(r.dst_blocks)] = r.src_blocks, r.dst_blocks
    lens = torch.tensor([r.num_tokens for r in w.requests], dtype=torch.int32, device="cuda")
    return torch.from_numpy(hs).cuda(), torch.from_numpy(hd).cuda(), lens, ws, wd, max_t


def test_table_driven_layer_ranges_parity_and_one_graph_of_layerwise_launches():
    """flowkv_transfer_tables_layers: (i) each range alone == the oracle's layer-range loop, other layers keep the
    sentinel, one launch per range, zero for an empty one; (ii) a layer-wise sender — one launch per layer — captured
    ONCE in a CUDA graph and replayed while the device tables change, whole pool against the oracle each time."""
    shape = synth.Shape(5, 2, 64, "fp16")
    L = shape.num_layers
    w = synth.make_workload("tables_layers", 4242, shape, [150, 31, 0, 64], "lkbthd", 16, ("geometric", 2.0), 64,
                            "blkhtd", 32, ("geometric", 4.0), 32)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    gs, gd = G.geom(w.src, shape), G.geom(w.dst, shape)
    st, dt, lens, ws, wd, max_t = _padded_tables(w)
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    n = len(w.requests)
    for l0, l1 in [(0, 1), (1, 4), (4, 5), (0, 5), (2, 2)]:
        P.fill_sentinel(dp.dst_buf)
        n0 = F.flowkv_launch_count()
        F.flowkv_transfer_tables_layers(dp.src, dp.dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), n, ws, wd, max_t, l0, l1,
                                        flag.data_ptr())
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if l1 > l0 else 0)
        exp = np.full(w.dst.bytes(shape), P.SENTINEL_BYTE, np.uint8)
        for r in w.requests:
            O.transfer(src_np, gs, exp, gd, r.src_blocks, r.dst_blocks, r.num_tokens, l0, l1)
        G.assert_same(P.to_numpy(dp.dst_buf), exp, f"table-driven layers [{l0},{l1})")
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_transfer_tables_layers(dp.src, dp.dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), n, ws, wd, max_t, 3, L + 1)
    assert ei.value.status == F.FLOWKV_ERR_INVALID_ARG
    # (ii) layer-wise sender inside one captured graph
    stream = torch.cuda.Stream()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=stream):
        for layer in range(L):
            F.flowkv_transfer_tables_layers(dp.src, dp.dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), n, ws, wd, max_t,
                                            layer, layer + 1, flag.data_ptr(), None, torch.cuda.current_stream().cuda_stream)
    rng = np.random.default_rng(7)
    for it in range(3):
        Ts = [int(rng.integers(0, max_t + 1)) for _ in range(n)]
        sperm = rng.permutation(w.src.num_blocks).astype(np.int32)
        dperm = rng.permutation(w.dst.num_blocks).astype(np.int32)
        hs, hd = np.full((n, ws), -1, np.int32), np.full((n, wd), -1, np.int32)
        reqs, so, do = [], 0, 0
        for i, t in enumerate(Ts):
            a, b = sperm[so:so + -(-t // 16)], dperm[do:do + -(-t // 32)]
            so, do = so + len(a), do + len(b)
            hs[i, :len(a)], hd[i, :len(b)] = a, b
            reqs.append((t, a, b))
        st.copy_(torch.from_numpy(hs)); dt.copy_(torch.from_numpy(hd)); lens.copy_(torch.tensor(Ts, dtype=torch.int32))
        P.fill_sentinel(dp.dst_buf)
        torch.cuda.synchronize()
        n0 = F.flowkv_launch_count()
        g.replay()
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() == n0          # replays launch from the graph, not through the library
        exp = np.full(w.dst.bytes(shape), P.SENTINEL_BYTE, np.uint8)
        for t, a, b in reqs:
            O.transfer(src_np, gs, exp, gd, a, b, t)
        G.assert_same(P.to_numpy(dp.dst_buf), exp, f"layer-wise graph replay {it}")
        assert int(flag.item()) == 0


def test_segment_allocator_tables_through_plan_and_transfer():
    """S§8f NEXT-1 end to end (P:L105 -> P:L107 -> the copy): a seeded alloc/free churn runs through flowkv_alloc_* for
    BOTH pools, the tables it hands out go into flowkv_plan + flowkv_transfer, the bytes are the oracle's, the segment
    count is okv_align's, and the product allocator handed out exactly what the oracle allocator does."""
    from oracle.allocator_oracle import OracleAllocator

    class OA:
        def __init__(self, nb):
            self.a = OracleAllocator(nb)

        def allocate(self, k):
            return self.a.allocate(k)

        def free(self, ids):
            self.a.release([int(i) for i in ids])

    w = synth.config3_batched(n_requests=5, num_layers=2, allocator=F.Allocator)
    wo = synth.config3_batched(n_requests=5, num_layers=2, allocator=OA)
    for a, b in zip(w.requests, wo.requests):
        assert np.array_equal(a.src_blocks, b.src_blocks) and np.array_equal(a.dst_blocks, b.dst_blocks)
    fifo = synth.config3_batched(n_requests=5, num_layers=2)
    dp, plan, _ = G.run_transfer_and_check(w)
    n_seg = sum(O.count_segments(r.src_blocks, 16, r.dst_blocks, 16, r.num_tokens) for r in w.requests)
    assert plan.stats["n_segments"] == n_seg
    fifo_seg = sum(O.count_segments(r.src_blocks, 16, r.dst_blocks, 16, r.num_tokens) for r in fifo.requests)
    assert n_seg * 3 < fifo_seg, (n_seg, fifo_seg)        # the allocator's point: far fewer, longer segments


# ---------------------------------------------------------------------------------------------------------
# rows mode through the TMA tensor path (cp.async.bulk.tensor): layout / block-size conversion by the TMA unit
# ---------------------------------------------------------------------------------------------------------
ROWS_TMA_TUNINGS = [
    {"variant": "bulk"},
    {"variant": "bulk", "stages": 4, "tile_bytes": 16384},
    {"variant": "bulk", "max_sms": 16, "ctas_per_sm": 2, "stages": 6},
    {"variant": "bulk", "plan_in_params": 1, "tile_order": 2, "tile_bytes": 8192},
]


@pytest.mark.parametrize("tuning", ROWS_TMA_TUNINGS)
def test_cfg4_hetero_through_the_tma_tensor_path(tuning):
    """configs[3] scaled (src BS16 LKBTHD -> dst BS64 BLKHTD, partial 64-token dst blocks, ragged request ends): the
    bulk variant is honoured in rows mode (stats.variant says so) and the whole dst pool is the oracle's."""
    w = synth.config4_hetero(n_requests=3, num_layers=2)
    dp, plan, _ = G.run_transfer_and_check(w, tuning)
    st = plan.stats
    assert st["mode_transfer"] == 2 and st["variant"] == F.FLOWKV_VARIANT_BULK and st["threads"] == 32, st
    assert st["smem_bytes"] <= 227 * 1024


@pytest.mark.parametrize("pair", [("lkbthd", 16, "blkhtd", 64), ("blkhtd", 64, "lkbthd", 16), ("blkhtd", 8, "blkhtd", 32),
                                  ("blkthd", 4, "blkhtd", 4), ("lkbthd", 1, "blkhtd", 2), ("blkhtd", 32, "blkthd", 16)])
@pytest.mark.parametrize("heads,dim,dtype", [(8, 128, "bf16"), (3, 40, "fp16"), (1, 8, "fp16"), (5, 16, "fp8"), (2, 64, "fp32")])
def test_rows_tma_layout_pairs_shapes_and_ragged_ends(pair, heads, dim, dtype):
    """Every rows-mode layout pair, odd head counts, 16-byte rows (tokens of 48 .. 2048 bytes: ragged chunks park
    tokens at 128-byte aligned shared-memory offsets), 1-, 2- and 4-byte elements; request lengths that end inside a
    block on both sides, an empty request and a one-token request; layer ranges ride the same maps."""
    sl, sbs, dl, dbs = pair
    shape = synth.Shape(3, heads, dim, dtype)
    w = synth.make_workload(f"rows_tma_{sl}{sbs}_{dl}{dbs}", 31337, shape, [97, 0, 1, 130, 64], sl, sbs, ("geometric", 3.0), None,
                            dl, dbs, ("geometric", 5.0), None)
    dp, plan, exp = G.run_transfer_and_check(w, {"variant": "bulk"}, fill="bits")
    assert plan.stats["variant"] == F.FLOWKV_VARIANT_BULK, plan.stats
    src_np = P.to_numpy(dp.src_buf)
    gs, gd = G.geom(w.src, shape), G.geom(w.dst, shape)
    for l0, l1 in [(0, 1), (1, 3), (2, 2)]:
        P.fill_sentinel(dp.dst_buf)
        n0 = F.flowkv_launch_count()
        F.flowkv_transfer_layers(plan, l0, l1)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == (1 if l1 > l0 else 0)
        e2 = np.full(w.dst.bytes(shape), P.SENTINEL_BYTE, np.uint8)
        for r in w.requests:
            O.transfer(src_np, gs, e2, gd, r.src_blocks, r.dst_blocks, r.num_tokens, l0, l1)
        G.assert_same(P.to_numpy(dp.dst_buf), e2, f"rows TMA layers [{l0},{l1})")
    # pack / unpack of a bulk rows plan run the register path (a dense side has no tensor map) and still match
    nbytes = plan.stats["staging_bytes"]
    staging = P.alloc_bytes(nbytes)
    P.fill_sentinel(dp.dst_buf)
    plan.pack(staging.data_ptr(), nbytes)
    plan.unpack(staging.data_ptr(), nbytes)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(staging), G.oracle_pack(w, src_np), "wire bytes of a bulk rows plan")
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "unpack of a bulk rows plan")


def test_rows_tma_falls_back_where_a_tensor_map_cannot_describe_the_pool():
    """A STRIDED pool whose layer stride is not twice its K|V stride has no uniform plane axis: the plan says LDST in
    stats.variant and the bytes are still the oracle's."""
    shape = synth.Shape(2, 2, 64, "fp16")
    L, H, D, NBs, NBd, bs = 2, 2, 64, 12, 10, 8
    row, tok = D * 2, H * D * 2
    blk, kv = bs * tok, NBs * bs * tok + 64
    lay = 2 * kv + 96
    gs = O.PoolGeom(L, H, D, 2, NBs, bs, lay, kv, blk, tok, row)
    gd = O.PoolGeom.blkhtd(L, H, D, 2, NBd, bs)
    src_buf, dst_buf = P.alloc_bytes(gs.span_bytes()), P.alloc_bytes(gd.span_bytes())
    P.fill_values(src_buf, "bits", "fp16", 5)
    P.fill_sentinel(dst_buf)
    src = F.make_pool(src_buf.data_ptr(), L, H, D, 2, NBs, bs, "strided", [lay, kv, blk, tok, row])
    dst = F.make_pool(dst_buf.data_ptr(), L, H, D, 2, NBd, bs, "blkhtd")
    a, b = np.asarray([3, 4, 9, 0], np.int32), np.asarray([7, 1, 2, 5], np.int32)
    plan = F.flowkv_plan(src, dst, [F.Request(29, a, b)], 0, {"variant": "bulk"})
    assert plan.stats["mode_transfer"] == 2 and plan.stats["variant"] == F.FLOWKV_VARIANT_LDST
    plan.transfer()
    torch.cuda.synchronize()
    exp = np.full(gd.span_bytes(), P.SENTINEL_BYTE, np.uint8)
    O.transfer(P.to_numpy(src_buf), gs, exp, gd, a, b, 29)
    G.assert_same(P.to_numpy(dst_buf), exp, "fallback")


def test_bench_starts_its_own_ranks_and_peer_mode_runs_on_one_gpu():
    """`python bench.py --gpus 2` with no launcher starts 2 ranks itself (one process per rank, torch.distributed
    rendezvous on 127.0.0.1); --peer makes rank r store into rank (r+1)%2's dst pool through CUDA IPC; --same-device puts
    both ranks on cuda:0 with a gloo control plane (there is one GPU here).  A functional check of the multi-rank
    path, not a scaling number: the line must report both ranks and one launch per step per rank 0."""
    import json
    import os
    import subprocess
    import sys
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ)
    for k in ("WORLD_SIZE", "RANK", "LOCAL_RANK", "MASTER_ADDR", "MASTER_PORT"):
        env.pop(k, None)
    out = subprocess.run([sys.executable, os.path.join(root, "bench.py"), "--gpus", "2", "--same-device", "--peer", "--config", "cfg1",
                          "--steps", "10", "--warmup", "3", "--no-e2e", "--no-baselines", "--no-cpu-baseline"],
                         capture_output=True, text=True, timeout=600, env=env, cwd=root)
    assert out.returncode == 0, out.stderr[-3000:]
    lines = [ln for ln in out.stdout.splitlines() if ln.startswith("{")]
    assert len(lines) == 1, out.stdout
    j = json.loads(lines[0])
    assert j["n_gpus"] == 2 and j["gpu_launches"] == 10 and j["launches_per_batch"] == 1.0
    assert "CUDA IPC" in j["run"]["dst"]
    # one record per rank: two processes, each launched its 10 kernels, moved its payload, and what it stored through the
    # IPC mapping reads back equal to its own src pool on sampled tokens
    pr = j["per_rank"]
    assert len(pr) == 2 and [r["rank"] for r in pr] == [0, 1] and pr[0]["pid"] != pr[1]["pid"]
    assert all(r["gpu_launches"] == 10 and r["payload_bytes_moved"] == 10 * j["config"]["payload_bytes"] for r in pr)
    assert all(r["peer_sample_matches_src"] is True for r in pr)


def test_hand_worked_golden_example_on_the_gpu():
    """tests/golden/transfer_example.json (5 tokens, block tables [2,0,1] -> [1,0], LKBTHD/2 -> BLKHTD/4): the CUDA path
    against the hand-worked values directly — register path, TMA tensor path and the table-driven kernel."""
    import json
    import os
    with open(os.path.join(os.path.dirname(__file__), "golden", "transfer_example.json")) as f:
        fx = json.load(f)
    src_h = np.zeros(2 * 3 * 2 * 2 * 8, np.uint16)
    for c in range(2):
        for b in range(3):
            for t in range(2):
                for h in range(2):
                    off = ((c * 3 + b) * 2 + t) * 2 * 8 + h * 8
                    src_h[off:off + 8] = 1000 * c + 100 * b + 10 * t + h
    exp = np.full(2 * 128, 65535, np.uint16)
    for blk, c, h, tok, val in fx["expect_dst_rows"]["rows"]:
        off = blk * 128 + c * 64 + h * 32 + tok * 8
        exp[off:off + 8] = val
    src_buf = torch.from_numpy(src_h.view(np.uint8).copy()).cuda()
    src = F.make_pool(src_buf.data_ptr(), 1, 2, 8, 2, 3, 2, "lkbthd")
    rq = fx["request"]
    a, b = np.asarray(rq["src_blocks"], np.int32), np.asarray(rq["dst_blocks"], np.int32)
    for tuning in (None, {"variant": "bulk"}, "tables"):
        dst_buf = torch.full((exp.size * 2,), 255, dtype=torch.uint8, device="cuda")
        dst = F.make_pool(dst_buf.data_ptr(), 1, 2, 8, 2, 2, 4, "blkhtd")
        if tuning == "tables":
            st, dt = torch.from_numpy(a[None, :].copy()).cuda(), torch.from_numpy(b[None, :].copy()).cuda()
            lens = torch.tensor([rq["num_tokens"]], dtype=torch.int32, device="cuda")
            F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), 1, 3, 2, rq["num_tokens"])
        else:
            plan = F.flowkv_plan(src, dst, [F.Request(rq["num_tokens"], a, b)], F.FLOWKV_CHECK_DST_ALIAS, tuning)
            if tuning:
                assert plan.stats["variant"] == F.FLOWKV_VARIANT_BULK
            plan.transfer()
        torch.cuda.synchronize()
        got = dst_buf.cpu().numpy().view(np.uint16)
        assert np.array_equal(got, exp), tuning


@pytest.mark.parametrize("tokens", synth.TABLE3_TOKENS)
def test_paper_table3_request_lengths(tokens):
    """The paper's own request sizes (Table 3: 500 .. 12,000 input tokens), L = 2: planned transfer
    (register and TMA paths), the table-free host route and the table-driven kernel all reach the oracle's dst pool;
    lengths that are no multiple of the block size leave the tail of the last block untouched (A4)."""
    w = synth.table3_point(tokens, num_layers=2)
    dp, plan, exp = G.run_transfer_and_check(w)
    assert plan.stats["n_segments"] == synth.n_runs(w.requests[0].src_blocks)
    plan.destroy()
    s = torch.cuda.current_stream().cuda_stream
    dp.dst_buf.fill_(P.SENTINEL_BYTE)
    pb = dp.plan(0, {"variant": "bulk"}, s)
    assert pb.stats["variant"] == F.FLOWKV_VARIANT_BULK
    pb.transfer(s)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), exp, f"table 3 T={tokens}: TMA bulk path")
    pb.destroy()
    # host route: pool -> pinned host -> pool
    dp.dst_buf.fill_(P.SENTINEL_BYTE)
    pv = dp.plan(F.FLOWKV_PLAN_NO_TRANSFER, None, s)
    nbytes = pv.stats["staging_bytes"]
    host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    sb = F.flowkv_via_host_scratch_bytes(pv, 0)
    scratch = P.alloc_bytes(sb)
    F.flowkv_transfer_via_host(pv, host.data_ptr(), nbytes, 0, 0, s, scratch.data_ptr(), sb)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), exp, f"table 3 T={tokens}: host route")
    pv.destroy()
    # table-driven: block tables and the length stay on the device
    r = w.requests[0]
    dp.dst_buf.fill_(P.SENTINEL_BYTE)
    st_ = torch.from_numpy(np.ascontiguousarray(r.src_blocks)).cuda()
    dt_ = torch.from_numpy(np.ascontiguousarray(r.dst_blocks)).cuda()
    nt = torch.tensor([tokens], dtype=torch.int32, device="cuda")
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    F.flowkv_transfer_tables(dp.src, dp.dst, st_.data_ptr(), dt_.data_ptr(), nt.data_ptr(), 1, len(r.src_blocks),
                             len(r.dst_blocks), tokens, flag.data_ptr(), None, s)
    torch.cuda.synchronize()
    assert int(flag.item()) == 0
    G.assert_same(P.to_numpy(dp.dst_buf), exp, f"table 3 T={tokens}: table-driven")


def test_distinct_plans_from_distinct_threads_on_distinct_streams():
    """Header: 'distinct plans may be used from distinct threads'.  Four threads, each with its own stream and pools,
    loop plan -> transfer (-> host route) -> destroy at once — uploaded plans and plans that ride in the kernel
    parameters — so the library's shared caches (pinned staging, plan memory pool, upload stream, recycled vectors,
    via-host helper streams) are hit concurrently; every dst pool must equal the oracle's."""
    import threading
    shape = synth.Shape(3, 4, 64, "bf16")
    works = []
    for k in range(4):
        lengths = [700 + 37 * k, 90, 1500 + k] if k % 2 == 0 else [8 + k]       # odd threads: tiny plans (kernel params)
        run = 2.0
        works.append(synth.make_workload(f"mt{k}", 9000 + k, shape, lengths, "lkbthd", 16,
                                         ("fixed", 1) if k % 2 == 0 else ("geometric", run), None,
                                         "blkhtd" if k == 2 else "lkbthd", 32 if k == 2 else 16, ("geometric", 3.0), None))
    dps = [P.DevicePools(w, fill="bits") for w in works]
    srcs = [P.to_numpy(dp.src_buf) for dp in dps]
    streams = [torch.cuda.Stream() for _ in works]
    hosts = [torch.empty(max(w.payload_bytes, 16), dtype=torch.uint8, pin_memory=True) for w in works]
    errors, uploaded = [], [False] * 4
    torch.cuda.synchronize()

    def worker(k):
        try:
            dp, s = dps[k], streams[k].cuda_stream
            for it in range(25):
                plan = dp.plan(F.FLOWKV_CHECK_DST_ALIAS, {"plan_in_params": 1} if k % 2 == 0 else None, s)   # even threads upload
                uploaded[k] = plan.stats["plan_device_bytes"] > 0
                plan.transfer(s)
                if it % 5 == 4:
                    sb = F.flowkv_via_host_scratch_bytes(plan, 3)
                    scratch = P.alloc_bytes(sb)
                    F.flowkv_transfer_via_host(plan, hosts[k].data_ptr(), hosts[k].numel(), 3, 0, s, scratch.data_ptr(), sb)
                    streams[k].synchronize()
                plan.destroy()
            streams[k].synchronize()
        except Exception as e:          # noqa: BLE001 — reported by the main thread
            errors.append(f"thread {k}: {e!r}")

    threads = [threading.Thread(target=worker, args=(k,)) for k in range(4)]
    for t in threads:
        t.start()
    for t in threads:
        t.join()
    assert not errors, errors
    assert uploaded[0] and uploaded[2] and not uploaded[1] and not uploaded[3], uploaded
    torch.cuda.synchronize()
    for k, w in enumerate(works):
        G.assert_same(P.to_numpy(dps[k].dst_buf), G.oracle_transfer(w, srcs[k]), f"thread {k} ({w.name})")
        G.assert_same(P.to_numpy(dps[k].src_buf), srcs[k], "src pool must not change")


def _separate_layers(rng, L, H, D, e, NB, BS, unit=32, planes=False):
    """A cache whose layers are separate allocations (reading A22): every layer a (2,NB,BS,H,D) tensor — or, with
    ``planes``, every K and every V a (NB,BS,H,D) tensor of its own (A3) — at a shuffled, gapped offset of one device
    buffer -> (oracle geometry, plane offsets, total bytes)."""
    one = O.PoolGeom.lkbthd(1, H, D, e, NB, BS)
    n = 2 * L if planes else L
    size = one.plane_bytes() if planes else one.layer_bytes()
    off, pos = [0] * n, unit * int(rng.integers(0, 4))
    for i in rng.permutation(n):
        off[int(i)] = pos
        pos += size + unit * int(rng.integers(1, 9))
    g = O.PoolGeom(L, H, D, e, NB, BS, one.s_layer, one.s_kv, one.s_block, one.s_token, one.s_head)
    g = g.with_plane_offsets(off) if planes else g.with_layer_offsets(off)
    return g, list(g.plane_off), pos


@pytest.mark.parametrize("dst_kind", ["lkbthd", "separate", "separate_kv", "blkthd", "blkhtd32"])
@pytest.mark.parametrize("tuning", [None, {"variant": "bulk"}, {"plan_in_params": 1, "tile_bytes": 4096}])
def test_pools_whose_layers_are_separate_allocations(dst_kind, tuning):
    """before Eq. 5 the cache is 'separate tensor structures across all layer dimensions'.  src = L tensors at
    scattered addresses (flowkv_pool.plane_offsets, base in the MIDDLE so some offsets are negative); dst = a stacked
    pool, another set of separate tensors (per layer, or per layer AND K|V: 2L tensors on both sides), or ONE (B,L,2,H) tensor — the paper's own migration — incl. a block-size
    change.  Transfer, layer range, pack / unpack, windows, the table-driven kernel and the memcpy baseline against
    the oracle over whole buffers (the gaps between the tensors stay untouched)."""
    rng = np.random.default_rng(4100 + len(dst_kind))
    L, H, D, e, NBs, BS = 5, 4, 64, 2, 40, 16
    gs, soff, sbytes = _separate_layers(rng, L, H, D, e, NBs, BS, planes=dst_kind == "separate_kv")
    src_buf = P.alloc_bytes(sbytes)
    P.fill_values(src_buf, "bits", "fp16", 4100)
    src_np = P.to_numpy(src_buf)
    mid = soff[4]
    src = F.make_pool(src_buf.data_ptr() + mid, L, H, D, e, NBs, BS, "lkbthd", plane_offsets=[o - mid for o in soff])
    if dst_kind in ("separate", "separate_kv"):
        NBd, bs_d = 24, BS
        gd, doff, dbytes = _separate_layers(rng, L, H, D, e, NBd, bs_d, unit=16, planes=dst_kind == "separate_kv")   # 16-byte aligned only: 128-bit path
        dst_buf = P.alloc_bytes(dbytes)
        dst = F.make_pool(dst_buf.data_ptr(), L, H, D, e, NBd, bs_d, "lkbthd", plane_offsets=doff)
    else:
        lay, bs_d = {"lkbthd": ("lkbthd", BS), "blkthd": ("blkthd", BS), "blkhtd32": ("blkhtd", 32)}[dst_kind]
        NBd = 24 * BS // bs_d
        gd = getattr(O.PoolGeom, lay)(L, H, D, e, NBd, bs_d)
        dst_buf = P.alloc_bytes(gd.span_bytes())
        dst = F.make_pool(dst_buf.data_ptr(), L, H, D, e, NBd, bs_d, lay)
    Ts = [150, 0, 77, 16]
    stab = rng.permutation(NBs)
    dtab = rng.permutation(NBd)
    reqs, so, do = [], 0, 0
    for t in Ts:
        a, b = -(-t // BS), -(-t // bs_d)
        reqs.append((t, stab[so:so + a].astype(np.int32), dtab[do:do + b].astype(np.int32)))
        so, do = so + a, do + b
    freqs = [F.Request(t, a, b) for t, a, b in reqs]
    s = torch.cuda.current_stream().cuda_stream

    def expect(l0=0, l1=L):
        exp = np.full(dst_buf.numel(), P.SENTINEL_BYTE, np.uint8)
        for t, a, b in reqs:
            O.transfer(src_np, gs, exp, gd, a, b, t, l0, l1)
        return exp

    what = f"separate layers -> {dst_kind} {tuning}"
    plan = F.flowkv_plan(src, dst, freqs, F.FLOWKV_CHECK_DST_ALIAS, tuning, s)
    st = plan.stats
    assert st["mode_transfer"] == (1 if dst_kind in ("lkbthd", "separate", "separate_kv") else 2)
    assert st["vec_bytes"] == (16 if dst_kind in ("separate", "separate_kv") else 32)
    if tuning and tuning.get("variant") == "bulk":      # span: the bulk ring; rows: no tensor map for such a pool
        assert st["variant"] == (F.FLOWKV_VARIANT_BULK if st["mode_transfer"] == 1 else F.FLOWKV_VARIANT_LDST)
    P.fill_sentinel(dst_buf)
    n0 = F.flowkv_launch_count()
    plan.transfer(s)
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() - n0 == 1
    G.assert_same(P.to_numpy(dst_buf), expect(), what + ": transfer")
    P.fill_sentinel(dst_buf)
    F.flowkv_transfer_layers(plan, 1, 4, s)
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dst_buf), expect(1, 4), what + ": layers [1,4)")
    # wire format and a window
    nbytes = st["staging_bytes"]
    staging = P.alloc_bytes(nbytes)
    P.fill_sentinel(staging)
    P.fill_sentinel(dst_buf)
    plan.pack(staging.data_ptr(), nbytes, s)
    plan.unpack(staging.data_ptr(), nbytes, s)
    torch.cuda.synchronize()
    wire = np.full(nbytes, P.SENTINEL_BYTE, np.uint8)
    off = 0
    for t, a, _ in reqs:
        O.pack(src_np, gs, a, t, wire, off)
        off += t
    G.assert_same(P.to_numpy(staging), wire, what + ": wire bytes")
    G.assert_same(P.to_numpy(dst_buf), expect(), what + ": unpack")
    nb = F.flowkv_window_bytes(plan, 2, 5)
    win = P.alloc_bytes(nb)
    F.flowkv_pack_window(plan, win.data_ptr(), nb, 2, 5, s)
    torch.cuda.synchronize()
    wexp = np.full(nb, P.SENTINEL_BYTE, np.uint8)
    off = 0
    for t, a, _ in reqs:
        O.pack_window(src_np, gs, a, t, wexp, off, 2, 5)
        off += t
    G.assert_same(P.to_numpy(win), wexp, what + ": window [2,5)")
    # memcpy baseline (token-major on both sides only) walks the same per-layer addresses
    if dst_kind in ("lkbthd", "separate", "separate_kv"):
        P.fill_sentinel(dst_buf)
        calls = F.flowkv_baseline_segmentwise(plan, s)
        torch.cuda.synchronize()
        assert calls == st["n_segments"] * 2 * L
        G.assert_same(P.to_numpy(dst_buf), expect(), what + ": segmentwise memcpy baseline")
    # the host route (pack windows -> pinned host -> unpack windows) walks the same per-layer addresses
    if tuning is None:
        host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
        sb = F.flowkv_via_host_scratch_bytes(plan, 7)
        scratch = P.alloc_bytes(sb)
        P.fill_sentinel(dst_buf)
        F.flowkv_transfer_via_host(plan, host.data_ptr(), nbytes, 7, 0, s, scratch.data_ptr(), sb)
        torch.cuda.synchronize()
        G.assert_same(P.to_numpy(dst_buf), expect(), what + ": host route")
    plan.destroy()
    # table-driven: nothing planned, tables on the device
    if tuning is None:
        n = len(reqs)
        ws, wd = max(len(a) for _, a, _ in reqs), max(len(b) for _, _, b in reqs)
        st_ = np.full((n, ws), -3, np.int32)
        dt_ = np.full((n, wd), -3, np.int32)
        for i, (_, a, b) in enumerate(reqs):
            st_[i, :len(a)], dt_[i, :len(b)] = a, b
        dst_t, ddt_t = torch.from_numpy(st_).cuda(), torch.from_numpy(dt_).cuda()
        lens = torch.tensor(Ts, dtype=torch.int32, device="cuda")
        flag = torch.zeros(1, dtype=torch.int32, device="cuda")
        P.fill_sentinel(dst_buf)
        F.flowkv_transfer_tables_layers(src, dst, dst_t.data_ptr(), ddt_t.data_ptr(), lens.data_ptr(), n, ws, wd, max(Ts), 0, 3,
                                        flag.data_ptr(), None, s)
        F.flowkv_transfer_tables_layers(src, dst, dst_t.data_ptr(), ddt_t.data_ptr(), lens.data_ptr(), n, ws, wd, max(Ts), 3, L,
                                        flag.data_ptr(), None, s)
        torch.cuda.synchronize()
        assert int(flag.item()) == 0
        G.assert_same(P.to_numpy(dst_buf), expect(), what + ": table-driven, two layer ranges")
    G.assert_same(P.to_numpy(src_buf), src_np, what + ": src unchanged")


def test_src_layers_as_really_separate_torch_allocations():
    """The same through REAL separate allocations: one torch tensor per layer (`DevicePools(separate_src_layers=True)`),
    offsets = differences of their device pointers (any sign, any size).  dst equals the oracle run layer by layer on
    each tensor's own bytes."""
    w = synth.config2_llama8b_13k(num_layers=3)
    dp = P.DevicePools(w, separate_src_layers=True)
    assert len({t.data_ptr() for t in dp.src_layers}) == 3 and dp.src.plane_offsets
    plan, s = dp.plan(F.FLOWKV_CHECK_DST_ALIAS), torch.cuda.current_stream().cuda_stream
    plan.transfer(s)
    torch.cuda.synchronize()
    r = w.requests[0]
    one_s = G.geom(w.src, w.shape, num_layers=1)
    gd = G.geom(w.dst, w.shape)
    exp = np.full(w.dst.bytes(w.shape), P.SENTINEL_BYTE, np.uint8)
    for l, t in enumerate(dp.src_layers):          # layer l of dst := layer 0 of the 1-layer pool that tensor l is
        O.transfer(P.to_numpy(t), one_s, exp[l * gd.s_layer:(l + 1) * gd.s_layer], G.geom(w.dst, w.shape, num_layers=1),
                   r.src_blocks, r.dst_blocks, r.num_tokens)
    G.assert_same(P.to_numpy(dp.dst_buf), exp, "separate torch tensors per layer")
    plan.destroy()


@pytest.mark.parametrize("reader", ["span_ldst", "rows_ldst", "span_bulk", "rows_tma", "tables", "span_ldst_uploaded"])
def test_back_to_back_dependent_transfers_see_each_others_writes(reader):
    """Programmatic dependent launch: every copy kernel lets the next one start early (launch_dependents at entry) and
    must wait for the previous grid's memory before touching any (griddepcontrol.wait).  Writer: pool0 -> pool1 as 48
    CTAs of ONE 1 MiB tile each — a grid that leaves most SMs free and runs for tens of microseconds, so the reader's
    CTAs are resident while it is still storing.  Reader: pool1 -> pool2 launched right behind it on the same stream,
    one of each kernel family.  pool2 must equal the oracle applied twice; with the wait removed from the kernels
    every one of these cases reads sentinel bytes (checked once by building the library without it)."""
    L, H, D, e, T = 24, 4, 64, 2, 2048                      # 512 B per token and plane: 1 MiB per plane
    lay2, bs2 = ("blkhtd", 32) if reader.startswith("rows") else ("lkbthd", 16)
    g0 = g1 = O.PoolGeom.lkbthd(L, H, D, e, T // 16, 16)
    g2 = getattr(O.PoolGeom, lay2)(L, H, D, e, T // bs2 + 3, bs2)
    b0, b1, b2 = P.alloc_bytes(g0.span_bytes()), P.alloc_bytes(g1.span_bytes()), P.alloc_bytes(g2.span_bytes())
    P.fill_values(b0, "bits", "fp16", 78)
    p0 = F.make_pool(b0.data_ptr(), L, H, D, e, T // 16, 16, "lkbthd")
    p1 = F.make_pool(b1.data_ptr(), L, H, D, e, T // 16, 16, "lkbthd")
    p2 = F.make_pool(b2.data_ptr(), L, H, D, e, T // bs2 + 3, bs2, lay2)
    ident = np.arange(T // 16, dtype=np.int32)
    tab2 = np.random.default_rng(78).permutation(T // bs2 + 3)[:T // bs2].astype(np.int32)
    s = torch.cuda.current_stream().cuda_stream
    writer = F.flowkv_plan(p0, p1, [F.Request(T, ident, ident)], 0, {"tile_bytes": 1 << 20, "threads": 512}, s)
    assert writer.stats["n_chunks_transfer"] == 1 and writer.stats["grid"] == 2 * L
    tun = {"span_ldst": None, "rows_ldst": None, "span_bulk": {"variant": "bulk"}, "rows_tma": {"variant": "bulk"},
           "tables": None, "span_ldst_uploaded": {"plan_in_params": 1}}[reader]
    rd = F.flowkv_plan(p1, p2, [F.Request(T, ident, tab2)], 0, tun, s)
    if reader in ("span_bulk", "rows_tma"):
        assert rd.stats["variant"] == F.FLOWKV_VARIANT_BULK
    st1, dt2 = torch.from_numpy(ident).cuda(), torch.from_numpy(tab2).cuda()
    lens = torch.tensor([T], dtype=torch.int32, device="cuda")
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    src_np = P.to_numpy(b0)
    e1 = np.full(g1.span_bytes(), P.SENTINEL_BYTE, np.uint8)
    O.transfer(src_np, g0, e1, g1, ident, ident, T)
    e2 = np.full(g2.span_bytes(), P.SENTINEL_BYTE, np.uint8)
    O.transfer(e1, g1, e2, g2, ident, tab2, T)
    for rep in range(4):
        P.fill_sentinel(b1)
        P.fill_sentinel(b2)
        torch.cuda.synchronize()
        writer.transfer(s)                                  # nothing between the two launches
        if reader == "tables":
            F.flowkv_transfer_tables(p1, p2, st1.data_ptr(), dt2.data_ptr(), lens.data_ptr(), 1, len(ident), len(tab2), T,
                                     flag.data_ptr(), None, s)
        else:
            rd.transfer(s)
        torch.cuda.synchronize()
        G.assert_same(P.to_numpy(b2), e2, f"{reader} behind a long writer, pass {rep}")
    assert int(flag.item()) == 0
    writer.destroy()
    rd.destroy()


@pytest.mark.parametrize("stages", [2, 3, 16])
@pytest.mark.parametrize("kind", ["span", "flat", "rows_tma"])
def test_tma_rings_over_many_iterations_on_one_cta(kind, stages):
    """One driving thread on ONE SM walks the whole batch: hundreds of turns of the mbarrier ring per CTA (phase parity
    flips every `stages` tiles, slots are reused as soon as their store has read them).  Span ring, flat ring and the
    TMA tensor path, ring depths 2 / 3 / 16, ragged request ends included; whole dst pool against the oracle."""
    lay_s, lay_d, bs_d = {"span": ("lkbthd", "lkbthd", 16), "flat": ("blkthd", "blkthd", 16), "rows_tma": ("lkbthd", "blkhtd", 64)}[kind]
    w = synth.make_workload(f"ring_{kind}", 611 + stages, synth.Shape(3, 4, 64, "bf16"), [1234, 777, 5],
                            lay_s, 16, ("geometric", 3.0), None, lay_d, bs_d, ("geometric", 5.0), None)
    tuning = {"variant": "bulk", "max_sms": 1, "ctas_per_sm": 1, "stages": stages, "tile_bytes": 4096}
    dp, plan, _ = G.run_transfer_and_check(w, tuning)
    st = plan.stats
    assert st["variant"] == F.FLOWKV_VARIANT_BULK and st["grid"] == 1 and st["stages"] == stages
    assert st["mode_transfer"] == {"span": 1, "flat": 3, "rows_tma": 2}[kind]
    assert (st["n_chunks_transfer"] * st["n_planes"] if kind != "flat" else st["n_chunks_transfer"]) >= 300     # turns of the ring
    plan.destroy()


@pytest.mark.parametrize("stages", [2, 3])
def test_tma_ring_slot_reuse_with_slow_stores_to_pinned_host(stages):
    """The ring may refill a slot only after the store that drained it has READ it (cp.async.bulk.wait_group.read).
    Make the stores slow and the loads fast — pack from HBM into mapped pinned host memory through the bulk variant,
    few CTAs with a short ring — the ordering the PTX model requires the wait for.  (On B200 a library built with that
    wait relaxed by one group still passes: one SM's TMA unit appears to work its queue in order.  The test pins the
    result, not the hardware's slack.)"""
    w = synth.make_workload("ring_host", 733, synth.Shape(4, 8, 128, "bf16"), [4096, 1000],
                            "lkbthd", 16, ("geometric", 4.0), None, "lkbthd", 16, ("contiguous",), None)
    dp = P.DevicePools(w, fill="bits")
    src_np = P.to_numpy(dp.src_buf)
    s = torch.cuda.current_stream().cuda_stream
    plan = dp.plan(F.FLOWKV_PLAN_NO_TRANSFER, {"variant": "bulk", "stages": stages, "max_sms": 4, "ctas_per_sm": 1,
                                               "tile_bytes": 32768}, s)
    assert plan.stats["variant"] == F.FLOWKV_VARIANT_BULK and plan.stats["stages"] == stages and plan.stats["grid"] == 4
    nbytes = plan.stats["staging_bytes"]
    host = torch.empty(nbytes, dtype=torch.uint8, pin_memory=True)
    exp = G.oracle_pack(w, src_np)
    for rep in range(2):
        host.fill_(P.SENTINEL_BYTE)
        plan.pack(host.data_ptr(), nbytes, s)
        torch.cuda.synchronize()
        G.assert_same(host.numpy(), exp, f"bulk pack to pinned host, pass {rep}")
    P.fill_sentinel(dp.dst_buf)
    plan.unpack(host.data_ptr(), nbytes, s)              # slow loads, fast stores: the other direction
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "bulk unpack from pinned host")
    plan.destroy()


def test_prefix_cache_hit_moves_only_the_suffix():
    """the controller 'identifies global cache prefix matches to ... reduce KV Cache transfer latency' — the decode
    side already holds the first t0 tokens.  The request then carries the tables from block t0 / BS on and
    num_tokens = T - t0 (flowkv.h): the cached prefix blocks of dst keep their bytes, the suffix lands exactly where the
    oracle puts tokens [t0, T) of the full request; segments are those of the full alignment clipped at t0."""
    L, H, D, e, T, t0 = 3, 4, 64, 2, 1000, 320                     # t0 a multiple of both block sizes (16, 32)
    gs, gd = O.PoolGeom.lkbthd(L, H, D, e, 80, 16), O.PoolGeom.blkhtd(L, H, D, e, 40, 32)
    rng = np.random.default_rng(86)
    stab = np.concatenate([np.arange(5, 25), rng.permutation(np.arange(30, 80))[:43]]).astype(np.int32)     # 63 blocks
    dtab = rng.permutation(40)[:32].astype(np.int32)
    src_buf, dst_buf = P.alloc_bytes(gs.span_bytes()), P.alloc_bytes(gd.span_bytes())
    P.fill_values(src_buf, "bits", "fp16", 86)
    P.fill_values(dst_buf, "bits", "fp16", 87)                      # the decode pool is full of other requests' bytes
    src_np, dst0 = P.to_numpy(src_buf), P.to_numpy(dst_buf)
    src = F.make_pool(src_buf.data_ptr(), L, H, D, e, 80, 16, "lkbthd")
    dst = F.make_pool(dst_buf.data_ptr(), L, H, D, e, 40, 32, "blkhtd")
    sub_s, sub_d = stab[t0 // 16:], dtab[t0 // 32:]
    plan = F.flowkv_plan(src, dst, [F.Request(T - t0, sub_s, sub_d)], F.FLOWKV_CHECK_DST_ALIAS)
    full = O.align(stab, 16, dtab, 32, T)
    clipped = [(max(a, t0) - t0, a + n - max(a, t0)) for a, n in full if a + n > t0]
    assert [(s_["first_token"], s_["n_tokens"]) for s_ in plan.segments] == clipped
    plan.transfer()
    torch.cuda.synchronize()
    # oracle: the FULL request into a scratch copy, then keep only what tokens [t0, T) wrote
    whole = dst0.copy()
    O.transfer(src_np, gs, whole, gd, stab, dtab, T)
    prefix_only = dst0.copy()
    O.transfer(src_np, gs, prefix_only, gd, stab[:t0 // 16], dtab[:t0 // 32], t0)
    exp = np.where(prefix_only != dst0, dst0, whole)                # undo the prefix tokens' writes
    exp2 = dst0.copy()
    O.transfer(src_np, gs, exp2, gd, sub_s, sub_d, T - t0)          # the same through the sub-tables
    assert np.array_equal(exp, exp2)
    G.assert_same(P.to_numpy(dst_buf), exp, "suffix after a prefix-cache hit")
    plan.destroy()


@pytest.mark.parametrize("split_kv", [False, True])
def test_pool_from_per_layer_torch_tensors(split_kv):
    """`pools.pool_from_tensors`: a cache held as per-layer torch tensors ([2,NB,BS,H,D] each, or separate K and V tensors
    per layer) is described in place (base = lowest pointer, plane offsets = pointer distances) and moved into one
    (B,L,2,H) tensor — Eq. 5's migration — in one launch; checked against torch indexing per plane (test-only) and the
    oracle run on each plane's own bytes."""
    L, NB, BS, H, D, T = 5, 48, 16, 4, 64, 700
    gen = torch.Generator(device="cuda").manual_seed(98)
    mk = lambda *shape: torch.randn(*shape, device="cuda", dtype=torch.bfloat16, generator=gen)
    if split_kv:
        ks, vs = [mk(NB, BS, H, D) for _ in range(L)], [mk(NB, BS, H, D) for _ in range(L)]
        src = P.pool_from_tensors(k_layers=ks, v_layers=vs)
        planes = [t for kv in zip(ks, vs) for t in kv]
    else:
        layers = [mk(2, NB, BS, H, D) for _ in range(L)]
        src = P.pool_from_tensors(layers=layers)
        planes = [t[c] for t in layers for c in (0, 1)]
    assert src.num_layers == L and src.elem_bytes == 2 and src.plane_offsets
    dst_t = torch.full((NB, L, 2, BS, H, D), -1.0, device="cuda", dtype=torch.bfloat16)         # one (B,L,2,H) tensor
    dst = F.make_pool(dst_t.data_ptr(), L, H, D, 2, NB, BS, "blkthd")
    rng = np.random.default_rng(98)
    stab, dtab = rng.permutation(NB)[:-(-T // BS)].astype(np.int32), rng.permutation(NB)[:-(-T // BS)].astype(np.int32)
    n0 = F.flowkv_launch_count()
    plan = F.flowkv_plan(src, dst, [F.Request(T, stab, dtab)], F.FLOWKV_CHECK_DST_ALIAS)
    plan.transfer()
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() - n0 == 1
    full, rem = T // BS, T % BS
    one = O.PoolGeom.lkbthd(1, H, D, 2, NB, BS)
    gplane = O.PoolGeom(1, H, D, 2, NB, BS, one.s_layer, one.s_kv, one.s_block, one.s_token, one.s_head).with_plane_offsets([0, 0])
    for p, t in enumerate(planes):
        l, c = p // 2, p % 2
        got = dst_t[:, l, c]                                             # [NB, BS, H, D]
        exp = torch.full_like(got, -1.0)
        exp[torch.from_numpy(dtab[:full]).long().cuda()] = t[torch.from_numpy(stab[:full]).long().cuda()]
        exp[int(dtab[full]), :rem] = t[int(stab[full]), :rem]
        assert torch.equal(got.view(torch.int16), exp.view(torch.int16)), f"plane {p}"
        # the oracle on this plane alone: a one-layer pool whose K and V plane are both this tensor (offsets [0, 0])
        o_src = t.contiguous().view(torch.uint8).cpu().numpy().reshape(-1)
        o_dst = torch.full_like(t, -1.0).view(torch.uint8).cpu().numpy().reshape(-1).copy()
        O.transfer(o_src, gplane, o_dst, gplane, stab, dtab, T)
        assert np.array_equal(o_dst, got.contiguous().view(torch.uint8).cpu().numpy().reshape(-1)), f"plane {p} (oracle)"
    plan.destroy()


# ---------------------------------------------------------------------------------------------------------
# round 3: contract violations the host cannot see, bounded caches, small parameter forms for separate-plane pools
# ---------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("separate", [False, True])
def test_table_driven_length_above_max_tokens_is_reported(separate):
    """A device-side length above the host's max_tokens: the grid was sized from max_tokens, so the tokens past it are
    not moved — the kernel must say so (error bit 4) instead of truncating silently; everything below max_tokens
    lands where the oracle puts it, nothing else is touched.  Both kernel forms (ordinary pool, per-plane offsets)."""
    shape = synth.Shape(2, 2, 64, "fp16")
    ssp, dsp = synth.PoolSpec("lkbthd", 16, 48), synth.PoolSpec("lkbthd", 16, 32)
    src_buf, dst_buf = P.alloc_bytes(ssp.bytes(shape)), P.alloc_bytes(dsp.bytes(shape))
    P.fill_values(src_buf, "bits", "fp16", 77)
    P.fill_sentinel(dst_buf)
    src_np = P.to_numpy(src_buf)
    dst = P.describe(dsp, shape, dst_buf.data_ptr())
    if separate:                                       # the same memory described plane by plane: the *_po kernel
        plane = ssp.num_blocks * 16 * 2 * 64 * 2
        src = F.make_pool(src_buf.data_ptr(), 2, 2, 64, 2, 48, 16, "lkbthd", plane_offsets=[p * plane for p in range(4)])
    else:
        src = P.describe(ssp, shape, src_buf.data_ptr())
    rng = np.random.default_rng(5)
    max_t, lens_h = 64, [64, 100, 17]                  # request 1 claims 100 tokens, the host said at most 64
    ws = wd = 7                                        # the tables do hold 100 tokens' worth of ids
    hs, hd = rng.permutation(48)[:21].astype(np.int32).reshape(3, 7), rng.permutation(32)[:21].astype(np.int32).reshape(3, 7)
    st, dt = torch.from_numpy(hs).cuda(), torch.from_numpy(hd).cuda()
    lens = torch.tensor(lens_h, dtype=torch.int32, device="cuda")
    flag = torch.zeros(1, dtype=torch.int32, device="cuda")
    F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), 3, ws, wd, max_t, flag.data_ptr())
    torch.cuda.synchronize()
    assert int(flag.item()) == 4
    gs, gd = G.geom(ssp, shape), G.geom(dsp, shape)
    exp = np.full(dsp.bytes(shape), P.SENTINEL_BYTE, np.uint8)
    for i, t in enumerate(lens_h):
        t = min(t, max_t)
        O.transfer(src_np, gs, exp, gd, hs[i, :-(-t // 16)], hd[i, :-(-t // 16)], t)
    G.assert_same(P.to_numpy(dst_buf), exp, "tokens below max_tokens move, the rest is reported, not moved")
    flag.zero_()                                       # within the bound: no bit
    lens.copy_(torch.tensor([64, 64, 17], dtype=torch.int32))
    F.flowkv_transfer_tables(src, dst, st.data_ptr(), dt.data_ptr(), lens.data_ptr(), 3, ws, wd, max_t, flag.data_ptr())
    torch.cuda.synchronize()
    assert int(flag.item()) == 0


@pytest.mark.parametrize("tokens", [40, 600, 3000, 20000])
def test_separate_plane_pools_in_every_parameter_form(tokens):
    """Pools with plane_offsets and a schedule of 3 / 38 / 188 / 1250 entries: the 512-byte, 3 KiB and 16 KiB parameter
    forms of the *_po kernels and the uploaded schedule, span and rows mode, against the oracle."""
    shape = synth.Shape(2, 2, 64, "fp16")
    for dst_layout, dst_bs in (("lkbthd", 16), ("blkhtd", 64)):
        w = synth.make_workload(f"po_tiers_{tokens}_{dst_layout}", 8800 + tokens, shape, [tokens], "lkbthd", 16, ("fixed", 1), None,
                                dst_layout, dst_bs, ("contiguous",), None, value_dist="bits")
        dp = P.DevicePools(w, separate_src_layers=True)
        src_np = np.concatenate([P.to_numpy(t) for t in dp.src_layers])
        plan = dp.plan(F.FLOWKV_CHECK_DST_ALIAS)
        n0 = F.flowkv_launch_count()
        plan.transfer(torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
        assert F.flowkv_launch_count() - n0 == 1
        assert (plan.stats["plan_device_bytes"] == 0) == (plan.stats["n_chunks_transfer"] <= 512)
        G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), w.name)


def test_plane_offset_tables_stay_bounded_and_trim_gives_them_back():
    """4,000 distinct plane_offsets tables (a server that keeps re-allocating its per-layer tensors): the library holds
    at most 64 + those that live plans reference; a table an alive plan uses survives any number of evictions and the
    plan still moves the right bytes; flowkv_trim() drops what nobody holds."""
    shape = synth.Shape(2, 2, 64, "fp16")
    w = synth.make_workload("po_cache", 8900, shape, [700], "lkbthd", 16, ("geometric", 2.0), None,
                            "lkbthd", 16, ("contiguous",), None, value_dist="bits")
    dp = P.DevicePools(w, separate_src_layers=True)
    src_np = np.concatenate([P.to_numpy(t) for t in dp.src_layers])
    s = torch.cuda.current_stream().cuda_stream
    F.flowkv_trim()
    base_tables = F.flowkv_cache_counts()["plane_offset_tables"]
    keeper = dp.plan(F.FLOWKV_CHECK_DST_ALIAS, None, s)              # holds dp.src's table for the whole test
    assert F.flowkv_cache_counts()["plane_offset_tables"] == base_tables + 1
    plane = 64 * 16 * 2 * 64 * 2
    big = P.alloc_bytes(4 * plane + 16 * 4000 + 4096)
    for i in range(4000):                                             # 4,000 pools that differ in one plane offset
        offs = [0, plane, 2 * plane, 3 * plane + 16 * (i + 1)]
        pool = F.make_pool(big.data_ptr(), 2, 2, 64, 2, 64, 16, "lkbthd", plane_offsets=offs)
        F.flowkv_plan(pool, None, [F.Request(16, np.array([i % 64], np.int32), None)], 0, None, s).destroy()
        if i % 500 == 0:
            assert F.flowkv_cache_counts()["plane_offset_tables"] <= 64 + 1 + base_tables
    assert F.flowkv_cache_counts()["plane_offset_tables"] <= 64 + 1 + base_tables
    keeper.transfer(s)                                                # its table was never evicted
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "plan that outlived 4,000 cache insertions")
    F.flowkv_trim()
    assert F.flowkv_cache_counts()["plane_offset_tables"] == base_tables + 1        # only the keeper's (and what earlier tests still hold)
    keeper.destroy()
    F.flowkv_trim()
    assert F.flowkv_cache_counts()["plane_offset_tables"] == base_tables
    dp.plan(F.FLOWKV_CHECK_DST_ALIAS, None, s).transfer(s)            # and everything still works afterwards
    torch.cuda.synchronize()
    G.assert_same(P.to_numpy(dp.dst_buf), G.oracle_transfer(w, src_np), "after trim")
