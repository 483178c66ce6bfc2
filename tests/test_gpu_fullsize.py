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


def _perm_of(job, torch):
    """sorted slot -> input index of the data grid (cute_grid_info.d_perm)"""
    inf = job.g_data.info()
    ws = job.g_data.workspace
    off = inf.d_perm - ws.data_ptr()
    return ws[off:off + inf.n * 4].view(torch.int32).cpu().numpy().astype(np.int64)


@pytest.mark.parametrize("cfg,cat", [(2, "data"), (3, "data"), (4, "data"), (5, "data"), (2, "rand"), (3, "rand")])
def test_auto_path_at_full_size(rt, oracle, cfg, cat):
    """The auto-correlation path (j > i mask, own-row segments) at BASELINE.json's full sizes, tied to the oracle two ways:
    (i) the exact identity cross(A, A)[k] = 2 auto(A)[k] + N [k = 0 and lo = 0] -- the cross side is oracle-checked on
    blocks by the tests above; (ii) the auto count of ~2e4 CONSECUTIVE cell-sorted points (a dense block of the real
    catalogue, through the same grid spec, so the same cells, chunks and own-row logic) against the oracle."""
    import torch
    api, runner, synth = rt
    w = synth.workload(cfg)
    if cat == "rand":                                       # RR of C2 (400 k) and C3 (10^6): the random catalogue through the same path
        w.data = w.rand
    n = len(w.data[0])
    grid = dict(w.grid)                                     # (keeps the permutation: no_perm is not set)
    job = runner.Job(w.kind, w.data, w.data, w.bins, grid).build()   # the same catalogue twice: two grids
    h_auto, st_auto = job.count("DD")
    h_cross, st_cross = job.count("DR")
    want = 2 * h_auto.astype(np.int64)
    if w.kind == "radial":
        # the N pairs (i, i): theta = 0 (inside the aperture), zbar = z_i, dz = 0 -> cell (bin of z_i, 0)
        e1 = api.cute_bin_edges(w.bins, 0)
        k1 = np.searchsorted(e1, np.asarray(w.data[2], dtype=np.float64), side="right") - 1
        ok1 = (k1 >= 0) & (k1 < w.bins["n1"])
        assert w.bins["lo2"] == 0.0
        np.add.at(want.reshape(w.bins["n1"], w.bins["n2"])[:, 0], k1[ok1], 1)
    elif w.bins["lo1"] == 0.0 and not w.bins.get("log1", 0):
        want.reshape(-1)[0] += n                            # the N pairs (i, i) at zero separation (r = 0 => mu = 0, reading S5)
    assert np.array_equal(h_cross.astype(np.int64).reshape(want.shape), want)
    if w.grid.get("mode", "none") == "none":
        assert st_auto["evaluated"] == n * (n - 1) // 2 and st_cross["evaluated"] == n * n
    # (ii) a block of consecutive sorted points
    perm = _perm_of(job, torch)
    assert np.array_equal(np.sort(perm), np.arange(n))
    for s0 in (0, n // 2 + 12345):
        idx = perm[s0:s0 + 20000]
        sub = tuple(np.ascontiguousarray(c[idx]) for c in w.data)
        jb = runner.Job(w.kind, sub, None, w.bins, grid)
        jb.spec = job.spec
        jb.build()
        h, st = jb.count("DD")
        orc = oracle.count(w.kind, sub, None, w.bins, mode="plain" if cfg == 2 else "celled")
        ok, msg = oracle.parity_ok(h, orc)
        assert ok, f"sorted block at {s0}: {msg}"
        assert h.sum() > (1000 if cfg != 4 else 0)


def test_c5_full_in_the_benchmarked_spec(rt, oracle):
    """bench.py builds its grids with no_perm = 1 (the sort permutation is not written): the full-size C5 counts in exactly
    that spec equal the ones of the permutation-writing build, and a block against the whole random catalogue, built
    with no_perm = 1 as well, satisfies the parity rule"""
    api, runner, synth = rt
    w = synth.workload(5)
    ref = runner.job_for_workload(w).build()
    want = {k: ref.count(k)[0] for k in ("DD", "DR")}
    del ref
    w.grid = dict(w.grid, no_perm=1)
    job = runner.job_for_workload(w).build()
    assert job.spec.no_perm == 1 and not job.g_data.info().d_perm
    for k in ("DD", "DR"):
        assert np.array_equal(job.count(k)[0], want[k])
    nd = len(w.data[0])
    _cross_block_check(rt, oracle, w, "DR", w.data, w.rand, _blocks(nd, 500, (4321,)), "celled")
