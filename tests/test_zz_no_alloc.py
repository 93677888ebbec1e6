"""`-m gpu`: flowkv_transfer_static, the pool -> pool move for callers that may not allocate device memory.

Who those callers are: a serving engine that handed all of HBM to its own KV block pool at start-up (a later
cudaMalloc may simply fail, or take memory the engine already promised to requests), a decode loop that cannot take
the device-wide stall an allocation or a free can cause, a tenant with a fixed memory budget.  The ordinary path
(flowkv_plan + flowkv_transfer) allocates a device buffer per plan once the schedule has more than 512 entries; the
static entry point keeps the schedule in a fixed 1 MiB array inside the library instead and is fed by a plan from
flowkv_plan_host, which makes no CUDA call.

What is checked: on batches big enough that the ordinary path does allocate (asserted), the static path leaves the
dst pool byte for byte as the ordinary path does — three calls in a row on one stream with no synchronisation in
between, each with a shorter schedule than the one before, so the array still holds stale entries of the previous
call past the end of the current one.  Then the size limit: a schedule that does not fit is refused with a message
that names the limit, and nothing is launched.

This file sorts last on purpose (pytest -x stops at the first failure).  It needs nothing from the tests before it:
the first static call in a process does the one-time address look-up itself.
"""
import numpy as np
import pytest
import torch

from paper_2504_03775_b200 import flowkv as F
from paper_2504_03775_b200 import pools as P
from paper_2504_03775_b200 import synth

pytestmark = pytest.mark.gpu

SMALL = synth.Shape(2, 2, 64, "fp16")


def _workloads():
    # span mode, 1,438 single-block runs; rows mode (block size 16 -> 64, token-major -> head-major), 1,126 entries;
    # flat mode (both pools block-major, Eq. 5's (B,L,2,H)), 600 single-block byte ranges
    a = synth.make_workload("static_a_span", 9101, SMALL, [20000, 3001], "lkbthd", 16, ("fixed", 1), None,
                            "lkbthd", 16, ("geometric", 3.0), None, value_dist="bits")
    b = synth.make_workload("static_b_rows", 9102, SMALL, [18005], "lkbthd", 16, ("geometric", 2.0), None,
                            "blkhtd", 64, ("permutation",), None, value_dist="bits")
    c = synth.make_workload("static_c_flat", 9103, SMALL, [9600], "blkthd", 16, ("permutation",), None,
                            "blkthd", 16, ("contiguous",), None, value_dist="bits")
    return a, b, c


def _ordinary_path(dp: P.DevicePools) -> np.ndarray:
    """dst pool after flowkv_plan + flowkv_transfer; asserts that this path did allocate a device schedule."""
    st = torch.cuda.current_stream().cuda_stream
    plan = dp.plan(F.FLOWKV_CHECK_DST_ALIAS, None, st)
    assert plan.stats["plan_device_bytes"] > 0, "the batch must be large enough for the ordinary path to allocate"
    plan.transfer(st)
    torch.cuda.synchronize()
    out = P.to_numpy(dp.dst_buf)
    plan.destroy()
    P.fill_sentinel(dp.dst_buf)
    torch.cuda.synchronize()
    return out


def test_static_schedule_matches_the_allocating_path_on_calls_in_a_row():
    pools = [P.DevicePools(w) for w in _workloads()]
    expected = [_ordinary_path(dp) for dp in pools]
    st = torch.cuda.current_stream().cuda_stream
    sizes = []
    n0 = F.flowkv_launch_count()
    for dp in pools:                                   # back to back on one stream, no synchronisation in between
        plan = F.flowkv_plan_host(dp.src, dp.dst, dp.requests, F.FLOWKV_CHECK_DST_ALIAS)
        stats = plan.stats
        assert stats["plan_device_bytes"] == 0 and 512 < stats["n_chunks_transfer"] <= F.FLOWKV_STATIC_SCHEDULE_ENTRIES
        sizes.append(stats["n_chunks_transfer"])
        F.flowkv_transfer_static(plan, st)
        plan.destroy()                                 # allowed as soon as the call has returned
    assert F.flowkv_launch_count() - n0 == len(pools), "one kernel per call"
    assert sizes == sorted(sizes, reverse=True) and len(set(sizes)) == len(sizes), "each schedule shorter than the last"
    assert {p.stats["mode_transfer"] for p in (F.flowkv_plan_host(dp.src, dp.dst, dp.requests) for dp in pools)} == {1, 2, 3}
    torch.cuda.synchronize()
    for dp, exp in zip(pools, expected):
        got = P.to_numpy(dp.dst_buf)
        assert np.array_equal(got, exp), f"{dp.w.name}: {int((got != exp).sum())} bytes differ from flowkv_transfer"
    # and once more with the first (longest) schedule, over whatever the shorter ones left behind
    dp = pools[0]
    P.fill_sentinel(dp.dst_buf)
    F.flowkv_transfer_static(F.flowkv_plan_host(dp.src, dp.dst, dp.requests), st)
    torch.cuda.synchronize()
    assert np.array_equal(P.to_numpy(dp.dst_buf), expected[0])


def test_static_schedule_refuses_what_does_not_fit_or_would_need_an_allocation():
    tiny = synth.Shape(1, 1, 8, "fp16")
    n_blocks = F.FLOWKV_STATIC_SCHEDULE_ENTRIES + 40
    w = synth.make_workload("static_too_big", 9104, tiny, [16 * n_blocks], "lkbthd", 16, ("fixed", 1), None,
                            "lkbthd", 16, ("contiguous",), None, value_dist="bits")
    dp = P.DevicePools(w)
    st = torch.cuda.current_stream().cuda_stream
    plan = F.flowkv_plan_host(dp.src, dp.dst, dp.requests)
    assert plan.stats["n_chunks_transfer"] > F.FLOWKV_STATIC_SCHEDULE_ENTRIES
    n0 = F.flowkv_launch_count()
    with pytest.raises(F.FlowKVError) as ei:
        F.flowkv_transfer_static(plan, st)
    assert ei.value.status == F.FLOWKV_ERR_UNSUPPORTED and str(F.FLOWKV_STATIC_SCHEDULE_ENTRIES) in str(ei.value)
    with pytest.raises(F.FlowKVError) as ei:           # the bulk variant is not served here
        F.flowkv_transfer_static(F.flowkv_plan_host(dp.src, dp.dst, [F.Request(0, [], [])],
                                                    0, {"variant": "bulk"}), st)
    assert ei.value.status == F.FLOWKV_ERR_UNSUPPORTED
    torch.cuda.synchronize()
    assert F.flowkv_launch_count() == n0, "a refused call launches nothing"
    assert np.all(P.to_numpy(dp.dst_buf) == P.SENTINEL_BYTE), "a refused call moves nothing"
    # an empty plan is fine and enqueues nothing
    F.flowkv_transfer_static(F.flowkv_plan_host(dp.src, dp.dst, []), st)
    assert F.flowkv_launch_count() == n0
