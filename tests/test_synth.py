"""Seeded input generators: structure of the tables they draw (CPU)."""
import numpy as np

from paper_2504_03775_b200 import synth


def _check_tables(w):
    for side, spec in (("src_blocks", w.src), ("dst_blocks", w.dst)):
        allids = np.concatenate([getattr(r, side) for r in w.requests]) if w.requests else np.zeros(0, np.int32)
        assert allids.dtype == np.int32
        assert len(np.unique(allids)) == len(allids), "a block is used twice"
        if len(allids):
            assert allids.min() >= 0 and allids.max() < spec.num_blocks
        for r in w.requests:
            assert len(getattr(r, side)) == -(-r.num_tokens // spec.block_size)


def test_cfg1():
    w = synth.config1_tiny()
    _check_tables(w)
    r = w.requests[0]
    assert r.num_tokens == 1000 and len(r.src_blocks) == 63
    assert synth.n_runs(r.src_blocks) == 63 and synth.n_runs(r.dst_blocks) == 1
    assert w.payload_bytes == 1_024_000
    w2 = synth.config1_tiny()
    assert np.array_equal(w2.requests[0].src_blocks, r.src_blocks), "seeded => reproducible"


def test_cfg2():
    w = synth.config2_llama8b_13k()
    _check_tables(w)
    r = w.requests[0]
    assert len(r.src_blocks) == 832 and w.payload_bytes == 1_744_830_464
    assert 150 <= synth.n_runs(r.src_blocks) <= 270          # ~208 runs of mean 4
    assert r.src_blocks.max() == 16383                         # byte offsets reach the top of the 32 GiB pool
    assert w.src.bytes(w.shape) == 32 * 2 ** 30 and w.dst.bytes(w.shape) == 2 * 2 ** 30


def test_cfg3_fit_rule_and_run_lengths():
    w = synth.config3_batched(budget_bytes=int(0.85 * 178 * 2 ** 30))
    _check_tables(w)
    n = w.notes["n_requests"]
    assert 30 <= n <= 64
    assert w.src.bytes(w.shape) + w.dst.bytes(w.shape) <= 0.85 * 178 * 2 ** 30
    assert 1.9 <= w.notes["mean_src_run"] <= 2.1
    used = sum(len(r.dst_blocks) for r in w.requests)
    druns = sum(synth.n_runs(r.dst_blocks) for r in w.requests)
    assert 12 <= used / druns <= 20
    assert all(1024 <= r.num_tokens <= 32768 for r in w.requests)
    full = synth.config3_batched()
    assert len(full.requests) == 64 and full.src.num_blocks == 65536


def test_cfg4():
    w = synth.config4_hetero(n_requests=3, num_layers=2)
    _check_tables(w)
    assert w.src.block_size == 16 and w.dst.block_size == 64 and w.dst.layout == "blkhtd"
    off = 0
    for r in w.requests:                                       # contiguous dst, request after request
        assert np.array_equal(r.dst_blocks, np.arange(off, off + len(r.dst_blocks)))
        off += len(r.dst_blocks)
    assert all(4096 <= t <= 32768 for t in synth.config4_lengths())


def test_cfg5_points():
    for T in (128, 4096, 131072):
        for run in synth.SWEEP_RUNS:
            w = synth.config5_point(T, run)
            _check_tables(w)
            tab = w.requests[0].src_blocks
            nb = T // 16
            exp_runs = 1 if (run == 0 or run >= nb) else -(-nb // run)
            assert synth.n_runs(tab) == exp_runs
            assert w.src.num_blocks == max(16384, 2 * nb)


def test_table3_points():
    """The paper's Table 3 request lengths: 131,072 B per token, ragged last blocks, seeded tables."""
    assert synth.TABLE3_TOKENS == [500, 1000, 2000, 4000, 8000, 10000, 12000]
    for T in synth.TABLE3_TOKENS:
        w = synth.table3_point(T)
        _check_tables(w)
        r = w.requests[0]
        assert r.num_tokens == T and w.payload_bytes == T * 131072
        assert synth.n_runs(r.dst_blocks) == 1 and 1 <= synth.n_runs(r.src_blocks) <= len(r.src_blocks)
        assert np.array_equal(synth.table3_point(T).requests[0].src_blocks, r.src_blocks)
