"""cute_count_pairs_static: the pair count for callers that cannot allocate device memory.

Some users of this library have no device memory of their own to offer and no permission to ask for any: an
analysis hook running inside a simulation whose memory manager owns the whole GPU, a plug-in under a host
application's fixed memory budget, a thread that may not call cudaMalloc because that would stall the device or
because another thread is recording a stream.  They get the same count as cute_count_pairs, with the kernel's small
scratch block (work counter, status, statistics, bin edges) in a fixed 64 KiB array inside the library instead of
a buffer they would have had to allocate.

What is checked: the histograms and the evaluated-pair statistics of the new entry point equal those of the existing
path (cute_count_pairs with a torch-allocated scratch buffer) bit for bit -- they are integer counts from the same
kernel, so the tolerance is zero -- on calls made back to back.  Consecutive calls use different kinds and bin
layouts on purpose: every call finds the previous one's counter, statistics and edges in the shared array and has
to clear or replace them.  Binning too fine for the fixed array must be refused before anything runs.

This file sorts after the other test files so that, under `pytest -x`, a failure here cannot hide theirs; it builds
everything it needs itself and passes alone in a fresh process as well as after the rest of the suite.
"""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def rt():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1210_1833_b200 import api, runner, synth
    return api, runner, synth, torch


def _both_paths(api, torch, job, which):
    """(histogram, stats) of one count through the existing path and through the static-scratch entry point"""
    h_ref, st_ref = job.count(which)                       # cute_count_pairs + cute_count_status, caller's scratch
    g1, g2 = job.grids(which)
    hist = torch.full((h_ref.size,), -1, dtype=torch.int64, device="cuda")   # stale garbage: the call must overwrite it
    st = api.cute_count_pairs_static(job.kind, g1, g2, job.bins, hist, job.opts)
    return h_ref, st_ref, hist.cpu().numpy().astype(np.uint64), st


def test_static_scratch_equals_caller_scratch_on_consecutive_calls(rt):
    api, runner, synth, torch = rt
    w5 = synth.workload(5, 0.002)      # periodic box, cell list, 1-D histogram (41 edges)
    w3 = synth.workload(3, 0.02)       # r-mu, cell list, 2-D histogram (41 + 51 edges): a longer edge block
    j5 = runner.job_for_workload(w5).build()
    j3 = runner.job_for_workload(w3).build()
    # back to back, alternating layouts; the last two repeat the first two on an array that is no longer fresh
    for job, which in ((j3, "DR"), (j5, "DD"), (j5, "DR"), (j3, "DD"), (j3, "DR"), (j5, "DD")):
        h_ref, st_ref, h, st = _both_paths(api, torch, job, which)
        assert h_ref.sum() > 0
        assert np.array_equal(h, h_ref), (job.kind_name, which)
        assert st["evaluated"] == st_ref["evaluated"] > 0
        assert st["items"] == st_ref["items"]


def test_static_scratch_degenerate_and_sharded_calls(rt):
    """an empty shard counts nothing (and must not see the previous call's counts); the shards add up"""
    api, runner, synth, torch = rt
    w = synth.workload(5, 0.002)
    job = runner.job_for_workload(w).build()
    full, _ = job.count("DD")
    g1, g2 = job.grids("DD")
    n = api.cute_count_items(job.kind, g1, g2, job.counter)
    hist = torch.empty(full.size, dtype=torch.int64, device="cuda")
    acc = np.zeros(full.size, dtype=np.uint64)
    for b, e in ((0, n // 3), (n // 3, n // 3), (n // 3, n)):
        api.cute_count_pairs_static(job.kind, g1, g2, job.bins, hist, api.count_opts(item_begin=b, item_end=e, shard=1))
        part = hist.cpu().numpy().astype(np.uint64)
        if b == e:
            assert not part.any()
        acc += part
    assert np.array_equal(acc, full)


def test_static_scratch_limit_is_refused(rt):
    api, runner, synth, torch = rt
    w = synth.workload(1, 0.01)
    job = runner.job_for_workload(w).build()
    g1, g2 = job.grids("DD")
    ok = dict(w.bins, n1=8182)          # 64 + 8 * (8182 + 1) + 8 * (0 + 1) = 65536 bytes: exactly the array
    hist = torch.empty(ok["n1"], dtype=torch.int64, device="cuda")
    api.cute_count_pairs_static(job.kind, g1, g2, ok, hist)
    counter = api.Counter(ok)
    api.cute_count_pairs(job.kind, g1, g2, counter)
    api.cute_count_status(counter)
    assert torch.equal(hist, counter.hist) and int(hist.sum()) > 0
    too_many = dict(w.bins, n1=8183)
    hist = torch.full((too_many["n1"],), 7, dtype=torch.int64, device="cuda")
    with pytest.raises(api.CuteError) as err:
        api.cute_count_pairs_static(job.kind, g1, g2, too_many, hist)
    assert err.value.status == api.ERR_STATIC_SCRATCH_LIMIT
    assert "cute_count_pairs" in str(err.value)
    assert int((hist != 7).sum()) == 0            # refused before anything was enqueued
