"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot run 1e11..1e12 pairs in a test, so (i) sampled outputs it can compute one by one: blocks of
the first catalogue against the WHOLE second catalogue (same kernels, same grids, same j-side sizes as the
full run) must satisfy the parity rule, and (ii) properties that hold at any size: the full histogram equals
the exact integer sum of its blocks, totals are bounded by the pair count, and evaluated == all pairs for
brute force.  C1 is small enough to be compared in full.
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
    return api, runner, synth


def _blocks(n, size, picks):
    return [(k * size, min(n, (k + 1) * size)) for k in picks]


def test_c1_full(rt, oracle):
    api, runner, synth = rt
    w = synth.workload(1)
    job = runner.job_for_workload(w).build()
    h, st = job.count("DD")
    orc = oracle.count(w.kind, w.data, None, w.bins)
    ok, msg = oracle.parity_ok(h, orc)
    assert ok, msg
    assert st["evaluated"] == 20000 * 19999 // 2
    # analytic RR of a uniform periodic box (Eqs. 12-13): xi ~ 0 within 5 sigma
    rr = api.cute_periodic_rr(job.nd, w.bins["box_L"], w.bins)
    assert np.all(np.abs(h.astype(float) - rr) <= 5.0 * np.sqrt(rr) + 1)


def _cross_block_check(rt, oracle, w, which_full, cat1, cat2, blocks, mode, all_blocks_size=None):
    """blocks of cat1 x all of cat2 on the GPU (cross-correlation through the same grids/kernels) vs the oracle"""
    api, runner, synth = rt
    full = runner.Job(w.kind, cat1, cat2, w.bins, w.grid).build()
    hfull, stfull = full.count("DR")
    n1 = len(cat1[0])
    spec = full.spec
    for b0, b1 in blocks:
        sub = tuple(np.ascontiguousarray(c[b0:b1]) for c in cat1)
        job = runner.Job(w.kind, sub, cat2, w.bins, w.grid)
        job.spec = spec
        job.build()
        h, st = job.count("DR")
        orc = oracle.count(w.kind, sub, cat2, w.bins, mode=mode)
        ok, msg = oracle.parity_ok(h, orc)
        assert ok, f"block [{b0},{b1}): {msg}"
    if all_blocks_size:
        acc = np.zeros_like(hfull)
        for b0 in range(0, n1, all_blocks_size):
            sub = tuple(np.ascontiguousarray(c[b0:b0 + all_blocks_size]) for c in cat1)
            job = runner.Job(w.kind, sub, cat2, w.bins, w.grid)
            job.spec = spec
            job.build()
            acc += job.count("DR")[0]
        assert np.array_equal(acc, hfull), "the full histogram is not the integer sum of its blocks"
    return hfull, stfull, full


def test_c2_full_sampled(rt, oracle):
    api, runner, synth = rt
    w = synth.workload(2)
    nd, nr = len(w.data[0]), len(w.rand[0])
    h, st, job = _cross_block_check(rt, oracle, w, "DR", w.data, w.rand, _blocks(nd, 1500, (0, 66, 133)), "plain",
                                    all_blocks_size=20000)
    assert st["evaluated"] == nd * nr            # brute force: every pair evaluated
    assert 0 < h.sum() < nd * nr
    # DD and RR in the benchmarked configuration: totals bounded, low bins populated by the clustering
    hdd, sdd = job.count("DD")
    hrr, srr = job.count("RR")
    assert sdd["evaluated"] == nd * (nd - 1) // 2 and srr["evaluated"] == nr * (nr - 1) // 2
    xi, _ = api.cute_landy_szalay(hdd, h, hrr, nd, nr)
    assert xi[20:40].mean() > 0.1                # Thomas process: clustering below ~0.1 deg (xi ~ 0.4 measured)
    assert abs(xi[-4:].mean()) < 0.05            # and none at 10 deg


def test_c3_full_sampled(rt, oracle):
    api, runner, synth = rt
    w = synth.workload(3)
    nd = len(w.data[0])
    _cross_block_check(rt, oracle, w, "DR", w.data, w.rand, _blocks(nd, 1000, (0, 250, 499)), "celled")


def test_c4_full_sampled(rt, oracle):
    api, runner, synth = rt
    w = synth.workload(4)
    n = len(w.data[0])
    # cross-correlate blocks of the catalogue with the whole catalogue (self pairs at theta = 0, dz = 0 included on both sides)
    _cross_block_check(rt, oracle, w, "DR", w.data, w.data, _blocks(n, 20000, (0, 57, 99)), "celled")
    job = runner.job_for_workload(w).build()
    h, st = job.count("DD")
    assert 3e4 < h.sum() < 8e4                   # ~5e4 binned pairs expected


def test_c5_full_sampled(rt, oracle):
    api, runner, synth = rt
    w = synth.workload(5)
    nd = len(w.data[0])
    _cross_block_check(rt, oracle, w, "DR", w.data, w.rand, _blocks(nd, 500, (0, 9999, 19999)), "celled")
