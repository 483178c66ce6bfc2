"""GPU parity: the CUDA path (through the C ABI) against the float64 oracle, element by element.

Bar (BASELINE.json north_star): histograms equal the oracle's exactly, per cell and in total,
except for pairs the oracle flags as lying within relative 2^-20 of a bin edge -- oracle.parity_ok
implements |gpu[c] - oracle[c]| <= amb_cell[c] and |sum gpu - sum oracle| <= amb_out.
Integer work (cell lists, permutations) is compared bit-exactly.
"""
import math

import numpy as np
import pytest

from conftest import load_golden

pytestmark = pytest.mark.gpu

GOLDEN = ["monopole_345.txt", "monopole_periodic.txt", "monopole_cross.txt", "angular_equator.txt",
          "angular_log.txt", "rmu_345.txt", "rmu_los.txt", "radial_ladder.txt", "pisigma_los.txt"]


@pytest.fixture(scope="module")
def rt():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1210_1833_b200 import api, runner, synth
    return api, runner, synth


def _cat(pts, kind):
    a = np.array(pts, dtype=np.float64).T
    return tuple(np.ascontiguousarray(c) for c in a)


def _run(runner, kind, data, rand, bins, grid=None, opts=None, which=("DD",)):
    job = runner.Job(kind, data, rand, bins, grid, opts).build()
    return {w: job.count(w) for w in which}, job


@pytest.mark.parametrize("name", GOLDEN)
def test_golden_fixtures(rt, name):
    """the hand-enumerated catalogues of tests/golden (paper definitions, Eq. 11)"""
    api, runner, synth = rt
    kind, bins, pts, pts2, expect = load_golden(name)
    data = _cat(pts, kind)
    rand = _cat(pts2, kind) if pts2 else None
    which = "DR" if rand is not None else "DD"
    out, job = _run(runner, kind, data, rand, bins, which=(which,))
    h, st = out[which]
    want = np.zeros(h.size, dtype=np.uint64)
    for k, v in expect.items():
        want[k] = v
    assert np.array_equal(h, want), (h.nonzero(), want.nonzero())


def _parity(oracle, h, kind, c1, c2, bins, mode="plain"):
    orc = oracle.count(kind, c1, c2, bins, mode=mode)
    ok, msg = oracle.parity_ok(h, orc)
    assert ok, msg
    return orc


@pytest.mark.parametrize("scale,opts", [(0.05, None), (0.1, dict(warps=4)), (0.1, dict(hist_cols=1, flush_items=3)),
                                        (0.1, dict(force_refine=1)), (0.1, dict(tau_scale=50.0))])
def test_c1_periodic_brute(rt, oracle, scale, opts):
    api, runner, synth = rt
    w = synth.workload(1, scale)
    out, job = _run(runner, w.kind, w.data, None, w.bins, w.grid, opts)
    h, st = out["DD"]
    orc = _parity(oracle, h, w.kind, w.data, None, w.bins)
    assert st["evaluated"] == job.total_pairs("DD") == orc["npairs"]


@pytest.mark.parametrize("scale", [0.01, 0.03])
def test_c2_angular_log(rt, oracle, scale):
    api, runner, synth = rt
    w = synth.workload(2, scale)
    out, job = _run(runner, w.kind, w.data, w.rand, w.bins, w.grid, which=("DD", "DR", "RR"))
    _parity(oracle, out["DD"][0], w.kind, w.data, None, w.bins)
    _parity(oracle, out["DR"][0], w.kind, w.data, w.rand, w.bins)
    _parity(oracle, out["RR"][0], w.kind, w.rand, None, w.bins)
    assert out["DR"][1]["evaluated"] == job.nd * job.nr


def test_c2_angular_sphere_grid_equals_brute(rt, oracle):
    """V6: grid-assisted == brute force, log bins up to 2 deg on a pixel grid"""
    api, runner, synth = rt
    w = synth.workload(2, 0.03)
    bins = dict(w.bins, hi1=math.radians(2.0), n1=52)
    out_b, _ = _run(runner, w.kind, w.data, w.rand, bins, dict(mode="none"), which=("DD", "DR"))
    out_g, job = _run(runner, w.kind, w.data, w.rand, bins, dict(mode="sphere", thetamax=bins["hi1"], pix=0.5), which=("DD", "DR"))
    for k in ("DD", "DR"):
        assert np.array_equal(out_b[k][0], out_g[k][0])
        assert out_g[k][1]["evaluated"] < out_b[k][1]["evaluated"]
    _parity(oracle, out_g["DD"][0], w.kind, w.data, None, bins)


def test_sphere_grid_full_sky_poles_and_seam(rt, oracle):
    """Eq. 16 (repaired, G2) at its hard places: a full-sky catalogue (both poles, the RA = 0/360 seam) on
    a ring of pixels, and a footprint that straddles the seam; grid == brute force == oracle"""
    api, runner, synth = rt
    rng = np.random.default_rng(21)
    n = 20000
    ra = rng.random(n) * 360.0
    dec = np.degrees(np.arcsin(rng.random(n) * 2 - 1))
    dec[:40] = 90.0 - rng.random(40) * 0.5          # a knot at the north pole
    dec[40:80] = -90.0 + rng.random(40) * 0.5       # and one at the south pole
    ra[80:200] = (359.7 + rng.random(120) * 0.6) % 360.0   # and one across the seam
    bins = dict(n1=20, lo1=math.radians(0.05), hi1=math.radians(3.0), log1=1, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    for pix in (1.0, 0.4):
        out_g, job = _run(runner, "angular", (ra, dec), None, bins, dict(mode="sphere", thetamax=bins["hi1"], pix=pix))
        assert job.spec.size[0] == 360.0
        out_b, _ = _run(runner, "angular", (ra, dec), None, bins, dict(mode="none"))
        assert np.array_equal(out_g["DD"][0], out_b["DD"][0])
        assert out_g["DD"][1]["evaluated"] < out_b["DD"][1]["evaluated"]
    _parity(oracle, out_g["DD"][0], "angular", (ra, dec), None, bins)
    # a narrow footprint across RA = 0 (given as 350..360 and 0..10), cross-correlated with randoms
    m = 6000
    ra1 = (350.0 + rng.random(m) * 20.0) % 360.0
    dec1 = rng.random(m) * 10.0 - 60.0
    ra2 = (350.0 + rng.random(m) * 20.0) % 360.0
    dec2 = rng.random(m) * 10.0 - 60.0
    out_g, job = _run(runner, "angular", (ra1, dec1), (ra2, dec2), bins, dict(mode="sphere", thetamax=bins["hi1"], pix=1.0), which=("DD", "DR"))
    out_b, _ = _run(runner, "angular", (ra1, dec1), (ra2, dec2), bins, dict(mode="none"), which=("DD", "DR"))
    assert np.array_equal(out_g["DD"][0], out_b["DD"][0]) and np.array_equal(out_g["DR"][0], out_b["DR"][0])
    _parity(oracle, out_g["DR"][0], "angular", (ra1, dec1), (ra2, dec2), bins)
    # a span just short of the ring is refused (points could be neighbours through the gap)
    with pytest.raises(api.CuteError):
        spec = api.grid_spec("sphere", origin=(0.0, -0.9, 0), size=(359.0, 0.2, 0), ncell=(100, 10, 1), rmax=bins["hi1"])
        import torch
        api.cute_make_grid([torch.from_numpy(ra1).cuda(), torch.from_numpy(dec1).cuda()], api.COORD_RADEC, spec)


def test_angular_linear_wide(rt, oracle):
    """the paper's own angular binning: linear in theta up to 30 deg"""
    api, runner, synth = rt
    w = synth.workload(2, 0.02)
    bins = dict(n1=256, lo1=0.0, hi1=math.radians(30.0), log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    out, job = _run(runner, "angular", w.data, w.rand, bins, which=("DD", "DR"))
    _parity(oracle, out["DD"][0], "angular", w.data, None, bins)
    _parity(oracle, out["DR"][0], "angular", w.data, w.rand, bins)


@pytest.mark.parametrize("ncell", [(0, 0, 0), (7, 9, 11)])
def test_c3_rmu_grid(rt, oracle, ncell):
    api, runner, synth = rt
    w = synth.workload(3, 0.02)
    grid = dict(w.grid, ncell=ncell)
    out, job = _run(runner, w.kind, w.data, w.rand, w.bins, grid, which=("DD", "DR", "RR"))
    _parity(oracle, out["DD"][0], w.kind, w.data, None, w.bins, "celled")
    _parity(oracle, out["DR"][0], w.kind, w.data, w.rand, w.bins, "celled")
    _parity(oracle, out["RR"][0], w.kind, w.rand, None, w.bins, "celled")
    # and brute force gives the same integers
    out_b, _ = _run(runner, w.kind, w.data, w.rand, w.bins, dict(mode="none"), which=("DD", "DR"))
    assert np.array_equal(out_b["DD"][0], out["DD"][0])
    assert np.array_equal(out_b["DR"][0], out["DR"][0])


@pytest.mark.parametrize("grid", ["box3d", "none"])
def test_pisigma_on_c3(rt, oracle, grid):
    """xi(pi,sigma), Eq. 2 -- the variant the paper times (Table II) and plots (Fig. 6) -- on the C3 catalogues"""
    api, runner, synth = rt
    w = synth.workload(3, 0.02)
    bins = dict(n1=32, lo1=0.0, hi1=80.0, log1=0, n2=32, lo2=0.0, hi2=80.0, aperture=0.0, box_L=0.0)
    g = dict(mode="box3d", rmax=math.hypot(80.0, 80.0)) if grid == "box3d" else dict(mode="none")
    out, job = _run(runner, "pisigma", w.data, w.rand, bins, g, which=("DD", "DR", "RR"))
    _parity(oracle, out["DD"][0], "pisigma", w.data, None, bins, "celled")
    _parity(oracle, out["DR"][0], "pisigma", w.data, w.rand, bins, "celled")
    _parity(oracle, out["RR"][0], "pisigma", w.rand, None, bins, "celled")
    out2, _ = _run(runner, "pisigma", w.data, w.rand, bins, g, dict(force_refine=1), which=("DR",))
    assert np.array_equal(out2["DR"][0], out["DR"][0])
    # pairs along the line of sight (sigma -> 0) and a catalogue through the origin (|l| -> 0) go through float64
    rng = np.random.default_rng(4)
    x = rng.normal(size=(3, 300)) * 20.0
    x = np.concatenate([x, -x[:, :50], x[:, :50] * 1.01], axis=1)
    b2 = dict(bins, hi1=30.0, hi2=30.0, n1=15, n2=15)
    out3, _ = _run(runner, "pisigma", tuple(x), None, b2, dict(mode="none"))
    _parity(oracle, out3["DD"][0], "pisigma", tuple(x), None, b2)
    b3 = dict(n1=15, lo1=0.0, hi1=30.0, log1=0, n2=20, lo2=0.0, hi2=1.0, aperture=0.0, box_L=0.0)
    out4, _ = _run(runner, "rmu", tuple(x), None, b3, dict(mode="none"))
    _parity(oracle, out4["DD"][0], "rmu", tuple(x), None, b3)


@pytest.mark.parametrize("pix", [2.0, 0.7])
def test_c4_radial_sphere_grid(rt, oracle, pix):
    api, runner, synth = rt
    w = synth.workload(4, 0.05)
    grid = dict(w.grid, pix=pix)
    out, job = _run(runner, w.kind, w.data, None, w.bins, grid)
    h, st = out["DD"]
    orc = _parity(oracle, h, w.kind, w.data, None, w.bins, "celled")
    assert h.sum() > 0
    # a wider aperture on a small catalogue against the PLAIN oracle
    w2 = synth.workload(4, 0.002)
    bins = dict(w2.bins, aperture=math.radians(0.5))
    out2, _ = _run(runner, w2.kind, w2.data, None, bins, dict(mode="sphere", thetamax=bins["aperture"], pix=pix))
    _parity(oracle, out2["DD"][0], w2.kind, w2.data, None, bins, "plain")
    out3, _ = _run(runner, w2.kind, w2.data, None, bins, dict(mode="none"))
    assert np.array_equal(out2["DD"][0], out3["DD"][0])


@pytest.mark.parametrize("scale,ncell", [(0.002, (0, 0, 0)), (0.002, (5, 7, 9)), (0.0005, (0, 0, 0))])
def test_c5_periodic_grid(rt, oracle, scale, ncell):
    api, runner, synth = rt
    w = synth.workload(5, scale)
    grid = dict(w.grid, ncell=ncell)
    out, job = _run(runner, w.kind, w.data, w.rand, w.bins, grid, which=("DD", "DR"))
    _parity(oracle, out["DD"][0], w.kind, w.data, None, w.bins, "celled")
    _parity(oracle, out["DR"][0], w.kind, w.data, w.rand, w.bins, "celled")
    out_b, _ = _run(runner, w.kind, w.data, w.rand, w.bins, dict(mode="none"), which=("DD", "DR"))
    assert np.array_equal(out_b["DD"][0], out["DD"][0])
    assert np.array_equal(out_b["DR"][0], out["DR"][0])


def test_c5_grid_prunes(rt, oracle):
    """a box much larger than r_max: the cell list evaluates far fewer separations than brute force
    and still gives the same integers"""
    api, runner, synth = rt
    w = synth.workload(5, 0.01)
    bins = dict(w.bins, hi1=40.0)
    grid = dict(mode="box3d", rmax=40.0)
    out, job = _run(runner, w.kind, w.data, w.rand, bins, grid, which=("DD", "DR"))
    out_b, _ = _run(runner, w.kind, w.data, w.rand, bins, dict(mode="none"), which=("DD", "DR"))
    for k in ("DD", "DR"):
        assert np.array_equal(out_b[k][0], out[k][0])
        assert out[k][1]["evaluated"] * 4 < out_b[k][1]["evaluated"]
    _parity(oracle, out["DD"][0], w.kind, w.data, None, bins, "celled")


def test_monopole_log_bins(rt, oracle):
    """logarithmic binning of the monopole"""
    api, runner, synth = rt
    w = synth.workload(5, 0.001)
    bins = dict(w.bins, lo1=0.5, log1=1, n1=48)
    out, job = _run(runner, w.kind, w.data, w.rand, bins, w.grid, which=("DD", "DR"))
    _parity(oracle, out["DD"][0], w.kind, w.data, None, bins, "celled")
    _parity(oracle, out["DR"][0], w.kind, w.data, w.rand, bins, "celled")


def test_edge_cases(rt, oracle):
    api, runner, synth = rt
    bins = dict(n1=8, lo1=0.0, hi1=10.0, log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    rng = np.random.default_rng(5)
    for n in (0, 1, 2, 127, 128, 129, 257):
        x = tuple(rng.random((3, n)) * 8.0)
        out, job = _run(runner, "monopole", x, None, bins)
        h = out["DD"][0]
        if n > 1:
            orc = _parity(oracle, h, "monopole", x, None, bins)
            assert out["DD"][1]["evaluated"] == n * (n - 1) // 2
        else:
            assert h.sum() == 0
    # coincident points: r = 0 is a pair in bin 0 (reading S4); cross counts everything
    x = (np.array([1.0, 1.0, 5.0]), np.array([2.0, 2.0, 2.0]), np.array([3.0, 3.0, 3.0]))
    out, _ = _run(runner, "monopole", x, x, bins, which=("DD", "DR"))
    assert out["DD"][0][0] == 1 and out["DD"][0].sum() == 3
    assert out["DR"][0][0] == 5 and out["DR"][0].sum() == 9


def test_permutation_invariance_and_sharding(rt):
    """V4: the histogram is invariant under a permutation of the input (an integer race detector);
    shards of the work-item list add up exactly (the multi-GPU path of DESIGN.md)."""
    api, runner, synth = rt
    w = synth.workload(5, 0.002)
    out, job = _run(runner, w.kind, w.data, w.rand, w.bins, w.grid, which=("DD", "DR"))
    rng = np.random.default_rng(1)
    p = rng.permutation(w.data[0].size)
    data2 = tuple(c[p] for c in w.data)
    out2, _ = _run(runner, w.kind, data2, w.rand, w.bins, w.grid, which=("DD", "DR"))
    assert np.array_equal(out["DD"][0], out2["DD"][0]) and np.array_equal(out["DR"][0], out2["DR"][0])
    g1, g2 = job.grids("DR")
    n = api.cute_count_items(job.kind, g1, g2, job.counter)
    acc = np.zeros_like(out["DR"][0])
    for a, b in ((0, n // 3), (n // 3, n // 2), (n // 2, n)):
        if a == b:
            continue
        job.opts = api.count_opts(item_begin=a, item_end=b)
        acc += job.count("DR")[0]
    assert np.array_equal(acc, out["DR"][0])


@pytest.mark.parametrize("build_path", [1, 2])
def test_cell_list_is_a_permutation(rt, build_path):
    """G1-G3 bit-exact: perm is a permutation, cell_start is the exclusive scan of the cell histogram,
    and every sorted point lies in its cell -- for the one-pass counting sort (1) and for the two-level
    partition that large catalogues take (2)."""
    import torch
    api, runner, synth = rt
    w = synth.workload(5, 0.003)
    w.grid = dict(w.grid, build_path=build_path)
    job = runner.job_for_workload(w).build()
    inf = job.g_data.info()
    n, nc = inf.n, inf.ncells
    ws = job.g_data.workspace

    def view(ptr, nbytes, dtype):
        off = ptr - ws.data_ptr()
        assert 0 <= off and off + nbytes <= ws.numel()
        return ws[off:off + nbytes].view(dtype)

    perm, cs, hi = view(inf.d_perm, n * 4, torch.int32), view(inf.d_cell_start, (nc + 1) * 4, torch.int32), view(inf.d_hi, n * 16, torch.float32)
    perm, cs, hi = perm.cpu().numpy().astype(np.int64), cs.cpu().numpy().astype(np.int64), hi.cpu().numpy().reshape(n, 4)
    assert np.array_equal(np.sort(perm), np.arange(n))
    x = np.stack(w.data, axis=1)[perm]
    assert np.array_equal(hi[:, :3], x.astype(np.float32))
    ncx, ncy, ncz = inf.ncell[0], inf.ncell[1], inf.ncell[2]
    cell = np.array([inf.cell[0], inf.cell[1], inf.cell[2]])
    k = np.minimum(np.floor(x.astype(np.float64) / cell).astype(np.int64), [ncx - 1, ncy - 1, ncz - 1])
    cid = (k[:, 2] * ncy + k[:, 1]) * ncx + k[:, 0]
    assert np.all(np.diff(cid) >= 0)
    want = np.concatenate([[0], np.cumsum(np.bincount(cid, minlength=nc))])
    assert np.array_equal(cs, want)


def test_host_entry_point_and_estimators(rt, oracle):
    """cute_count_pairs_host (HOST buffers) == device path; Landy-Szalay on identical histograms
    agrees with the oracle's Eq. 15 to 1e-6 absolute (north star)."""
    api, runner, synth = rt
    w = synth.workload(2, 0.02)
    out, job = _run(runner, w.kind, w.data, w.rand, w.bins, w.grid, which=("DD", "DR", "RR"))
    spec = api.grid_spec("none")
    hh, _ = api.cute_count_pairs_host(job.kind, w.data, w.rand, job.coord, spec, w.bins)
    assert np.array_equal(hh, out["DR"][0])
    dd, dr, rr = out["DD"][0], out["DR"][0], out["RR"][0]
    xi, rc = api.cute_landy_szalay(dd, dr, rr, job.nd, job.nr)
    xo, empty = oracle.landy_szalay(dd, dr, rr, job.nd, job.nr)
    assert np.max(np.abs(xi - xo)) <= 1e-6
    assert (rc == api.WARN_EMPTY_BIN) == (empty > 0)
    w1 = synth.workload(1, 0.1)
    o1, j1 = _run(runner, w1.kind, w1.data, None, w1.bins, w1.grid)
    rr1 = api.cute_periodic_rr(j1.nd, w1.bins["box_L"], w1.bins)
    assert np.allclose(rr1, oracle.periodic_rr(j1.nd, w1.bins["box_L"], w1.bins), rtol=1e-13)


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_box_grids(rt, oracle, seed):
    """random small catalogues, boxes, cell counts, bins: periodic and open cell lists against the PLAIN oracle
    (exercises wrap segments, chunks wider than a cell, empty cells, 1..3 cells per axis, ragged tiles)"""
    api, runner, synth = rt
    rng = np.random.default_rng(1000 + seed)
    periodic = bool(seed % 2)
    n1, n2 = int(rng.integers(1, 2500)), int(rng.integers(1, 2500))
    L = float(rng.uniform(50.0, 200.0))
    if periodic:
        rmax = float(rng.uniform(0.03, 0.45)) * L
        a = tuple(rng.random((3, n1)) * L)
        b = tuple(rng.random((3, n2)) * L)
        kind = "monopole"
    else:
        rmax = float(rng.uniform(0.05, 0.8)) * L
        ext = rng.uniform(0.2, 1.0, 3) * L
        off = rng.uniform(-500.0, 500.0, 3)
        a = tuple((rng.random((3, n1)) * ext[:, None]) + off[:, None])
        b = tuple((rng.random((3, n2)) * ext[:, None] * rng.uniform(0.5, 1.2)) + off[:, None])
        kind = ("monopole", "rmu", "pisigma")[seed // 2 % 3]
    log1 = int(kind == "monopole" and rng.random() < 0.4)
    bins = dict(n1=int(rng.integers(3, 40)), lo1=(rmax * 0.01 if log1 else 0.0), hi1=rmax, log1=log1, n2=0, lo2=0.0, hi2=0.0,
                aperture=0.0, box_L=L if periodic else 0.0)
    grmax = rmax
    if kind == "rmu":
        bins.update(n2=int(rng.integers(2, 30)), hi2=1.0)
    if kind == "pisigma":
        bins.update(n2=int(rng.integers(2, 30)), hi2=rmax * float(rng.uniform(0.3, 1.0)))
        grmax = math.hypot(bins["hi1"], bins["hi2"])
    ncell = (0, 0, 0) if rng.random() < 0.4 else tuple(int(v) for v in rng.integers(1 if not periodic else 3, 14, 3))
    grid = dict(mode="box3d", rmax=grmax, ncell=ncell)
    try:
        out, job = _run(runner, kind, a, b, bins, grid, which=("DD", "DR"))
    except api.CuteError as e:
        assert periodic and e.status == -2      # too few cells for this rmax: refused, never silently wrong
        out, job = _run(runner, kind, a, b, bins, dict(mode="none"), which=("DD", "DR"))
    _parity(oracle, out["DD"][0], kind, a, None, bins)
    _parity(oracle, out["DR"][0], kind, a, b, bins)


# ------------------------------------------------------------------------------- N2: weights and pixel maps
@pytest.mark.parametrize("grid", ["none", "sphere"])
def test_weighted_angular(rt, oracle, grid):
    """pixel maps: a pair counts w_i w_j, the objects of one pixel w(w-1)/2 pairs at zero separation"""
    api, runner, synth = rt
    rng = np.random.default_rng(41)
    n1, n2 = 3000, 2500
    c1 = (rng.random(n1) * 8 + 40, rng.random(n1) * 8 - 4)
    c2 = (rng.random(n2) * 8 + 40, rng.random(n2) * 8 - 4)
    w1 = rng.integers(1, 7, n1).astype(np.uint32)
    w2 = rng.integers(1, 5, n2).astype(np.uint32)
    for bins in (dict(n1=24, lo1=0.0, hi1=math.radians(1.5), log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0),
                 dict(n1=20, lo1=math.radians(0.01), hi1=math.radians(1.5), log1=1, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)):
        g = dict(mode="none") if grid == "none" else dict(mode="sphere", thetamax=bins["hi1"], pix=1.0)
        job = runner.Job("angular", c1, c2, bins, g, None, w_data=w1, w_rand=w2).build()
        for which, a, b, wa, wb in (("DD", c1, None, w1, None), ("DR", c1, c2, w1, w2), ("RR", c2, None, w2, None)):
            h, st = job.count(which)
            orc = oracle.count("angular", a, b, bins, w1=wa, w2=wb)
            ok, msg = oracle.parity_ok(h, orc)
            assert ok, f"{which}: {msg}"
        job.opts = api.count_opts(force_refine=1)
        h2, _ = job.count("DR")
        job.opts = None
        assert np.array_equal(h2, job.count("DR")[0])
    # heavy weights: the uint32 shared-memory counters are flushed on a short epoch
    wb1 = rng.integers(1, 400, n1).astype(np.uint32)
    job = runner.Job("angular", c1, None, bins, dict(mode="none"), None, w_data=wb1).build()
    h, st = job.count("DD")
    orc = oracle.count("angular", c1, None, bins, w1=wb1)
    ok, msg = oracle.parity_ok(h, orc)
    assert ok, msg
    assert st["flushes"] > 148 * 8
    hh, _ = api.cute_count_pairs_host(api.ANGULAR, c1, None, api.COORD_RADEC, api.grid_spec("none"), bins, w1=wb1)
    assert np.array_equal(hh, h)
    with pytest.raises(api.CuteError):
        runner.Job("angular", c1, None, bins, dict(mode="none"), None, w_data=np.full(n1, 70000, dtype=np.uint32)).build()


def test_pixel_map_and_wpix(rt, oracle):
    """cute_pixelize == the oracle's pixel map (counts exact); w_pix(theta) = weighted counts of the pixel catalogues"""
    import torch
    api, runner, synth = rt
    w = synth.workload(2, 0.1)                                   # 20k clustered + 40k random points
    tm = math.radians(10.0)
    ra0, dra, u0, du, nra, nu = 155.0, 50.0, 0.17, 0.75 - 0.17, 500, 380      # ~0.1 deg pixels over the cap
    cats = {}
    for name, cat in (("d", w.data), ("r", w.rand)):
        pra, pdec, pw = oracle.pixelize(cat[0], cat[1], ra0, dra, u0, du, nra, nu)
        g = api.cute_pixelize([torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in cat[:2]], ra0, dra, u0, du, nra, nu)
        gra, gdec, gw = (t.cpu().numpy() for t in g)
        assert np.array_equal(gw.view(np.uint32), pw) and pw.sum() == len(cat[0])
        assert np.allclose(gra, pra, rtol=0, atol=1e-11) and np.allclose(gdec, pdec, rtol=0, atol=1e-11)
        cats[name] = ((pra, pdec), pw)
    assert len(cats["d"][1]) < len(w.data[0])                    # clustered data: several objects per pixel
    bins = dict(n1=16, lo1=math.radians(0.5), hi1=tm, log1=1, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    (cd, wd), (cr, wr) = cats["d"], cats["r"]
    job = runner.Job("angular", cd, cr, bins, dict(mode="none"), None, w_data=wd, w_rand=wr).build()
    out = {}
    for which, a, b, wa, wb in (("DD", cd, None, wd, None), ("DR", cd, cr, wd, wr), ("RR", cr, None, wr, None)):
        out[which], st = job.count(which)
        orc = oracle.count("angular", a, b, bins, w1=wa, w2=wb)
        ok, msg = oracle.parity_ok(out[which], orc)
        assert ok, f"{which}: {msg}"
    # and w_pix agrees with the un-pixelised w(theta) above the pixel scale
    exact, _ = _run(runner, "angular", w.data, w.rand, bins, dict(mode="none"), which=("DD", "DR", "RR"))
    xi_pix, _ = api.cute_landy_szalay(out["DD"], out["DR"], out["RR"], len(w.data[0]), len(w.rand[0]))
    xi, _ = api.cute_landy_szalay(exact["DD"][0], exact["DR"][0], exact["RR"][0], len(w.data[0]), len(w.rand[0]))
    assert np.max(np.abs(xi_pix - xi)) < 0.02


def test_monopole_log_bins_far_from_origin(rt, oracle):
    """the paper's logarithmic monopole (256 bins, 50 per decade, r < 100) on float64 coordinates of
    magnitude ~2000: the float32 error of r is far larger than the lowest edge, so tau must depend on the pair"""
    api, runner, synth = rt
    w = synth.workload(3, 0.02)
    bins = dict(n1=256, lo1=100.0 * 10 ** (-256 / 50), hi1=100.0, log1=1, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    out, job = _run(runner, "monopole", w.data, w.rand, bins, dict(mode="box3d", rmax=100.0), which=("DD", "DR"))
    _parity(oracle, out["DD"][0], "monopole", w.data, None, bins, "celled")
    _parity(oracle, out["DR"][0], "monopole", w.data, w.rand, bins, "celled")
    assert out["DD"][1]["refined"] < 0.05 * out["DD"][0].sum()      # not everything goes through float64
    # coincident points (r = 0) are dropped by log bins, exactly as in the oracle
    x = tuple(np.concatenate([c[:500], c[:500]]) for c in w.data)
    out2, _ = _run(runner, "monopole", x, None, bins, dict(mode="none"))
    _parity(oracle, out2["DD"][0], "monopole", x, None, bins)


@pytest.mark.parametrize("cfg,scale", [(2, 0.02), (3, 0.02), (4, 0.02), (5, 0.002)])
def test_partition_build_gives_the_same_histograms(rt, oracle, cfg, scale):
    """the two-level partition build (build_path 2) and the one-pass build (1) are the same cell list up to the order
    inside a cell: identical histograms for every kind, coordinate type and grid mode (float64 RA/Dec/z and xyz, float32
    xyz; brute-force ordering cells, pixels, periodic and bounding-box cells)"""
    api, runner, synth = rt
    w = synth.workload(cfg, scale)
    outs = []
    for bp in (1, 2):
        out, job = _run(runner, w.kind, w.data, w.rand, w.bins, dict(w.grid, build_path=bp), which=tuple(w.pairs))
        outs.append(out)
    for k in w.pairs:
        assert np.array_equal(outs[0][k][0], outs[1][k][0])
    c2 = w.rand if "DR" in w.pairs else None
    which = "DR" if c2 is not None else "DD"
    _parity(oracle, outs[1][which][0], w.kind, w.data, c2, w.bins, mode="celled" if w.grid.get("mode", "none") != "none" else "plain")


@pytest.mark.parametrize("n,theta_deg,pix", [(20000, 10.0, 0.1), (3000, 20.0, 0.05), (9000, 3.0, 0.2)])
def test_sphere_ring_rows_with_mixed_chunks(rt, n, theta_deg, pix):
    """Regression (round-1 advisor): on a full ring, rows holding a little more than a multiple of 128 points mix a chunk
    whose window covers the whole ring with one whose window does not; seam pairs of the row's own points were then
    counted twice or dropped.  Full sky, fine pixels, 130-260 points per row, wide windows at high declination:
    the pixel grid must equal brute force exactly."""
    api, runner, synth = rt
    rng = np.random.default_rng(77 + n)
    ra = rng.random(n) * 360.0
    dec = np.degrees(np.arcsin(rng.random(n) * 2 - 1))
    th = math.radians(theta_deg)
    bins = dict(n1=24, lo1=0.0, hi1=th, log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    out_g, job = _run(runner, "angular", (ra, dec), None, bins, dict(mode="sphere", thetamax=th, pix=pix))
    assert job.spec.size[0] == 360.0
    per_row = n / job.spec.ncell[1]
    assert 10 < per_row < 400, per_row
    out_b, _ = _run(runner, "angular", (ra, dec), None, bins, dict(mode="none"))
    assert np.array_equal(out_g["DD"][0], out_b["DD"][0])
    # and a second catalogue through the same grid (cross: every row window is met exactly once)
    m = n // 2
    ra2, dec2 = rng.random(m) * 360.0, np.degrees(np.arcsin(rng.random(m) * 2 - 1))
    out_g, _ = _run(runner, "angular", (ra, dec), (ra2, dec2), bins, dict(mode="sphere", thetamax=th, pix=pix), which=("DR",))
    out_b, _ = _run(runner, "angular", (ra, dec), (ra2, dec2), bins, dict(mode="none"), which=("DR",))
    assert np.array_equal(out_g["DR"][0], out_b["DR"][0])


def test_refine_path_against_enumeration_and_eq9(rt):
    """The float64 refine path decides EVERY pair under force_refine.  It is compared here with counts that do not come
    from the oracle: (i) the torus-lattice enumeration of integer vectors (Eq. 11 PAPER.md:85 with the periodic wrap of
    PAPER.md:94) and (ii) r, mu from Eq. 9 for pairs built from (chi_1, chi_2, theta)."""
    import itertools
    api, runner, synth = rt
    n, h = 6, 1.5
    L = n * h
    g = np.arange(n) * h + 0.25
    x = np.array(list(itertools.product(g, g, g))).T
    x = x[:, np.random.default_rng(5).permutation(x.shape[1])]
    bins = dict(n1=29, lo1=0.05 * h, hi1=2.95 * h, log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=L)
    edges = bins["lo1"] + (bins["hi1"] - bins["lo1"]) * np.arange(30) / 29
    want = np.zeros(29, dtype=np.int64)
    rep = range(-n // 2, n // 2)
    for v in itertools.product(rep, rep, rep):
        m = v[0] ** 2 + v[1] ** 2 + v[2] ** 2
        if m == 0:
            continue
        r = h * math.sqrt(m)
        k = np.searchsorted(edges, r, side="right") - 1
        if 0 <= k < 29 and r < edges[-1]:
            want[k] += 1
    want = want * n ** 3 // 2
    for opts in (dict(force_refine=1), None):
        out, _ = _run(runner, "monopole", tuple(x), None, bins, dict(mode="none"), opts)
        assert np.array_equal(out["DD"][0].astype(np.int64), want)
    # Eq. 9: one pair per catalogue, (r, mu) cell from the closed form
    rng = np.random.default_rng(41)
    nr, nm = 64, 64
    b2 = dict(n1=nr, lo1=0.0, hi1=400.0, log1=0, n2=nm, lo2=0.0, hi2=1.0, aperture=0.0, box_L=0.0)
    checked = 0
    for _ in range(60):
        c1, c2 = 1000.0 + 600.0 * rng.random(2)
        th = 0.15 * rng.random()
        r9 = math.sqrt(c1 * c1 + c2 * c2 - 2 * c1 * c2 * math.cos(th))
        mu9 = abs(c1 * c1 - c2 * c2) / math.sqrt((c1 * c1 + c2 * c2) ** 2 - 4 * c1 * c1 * c2 * c2 * math.cos(th) ** 2)
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        v = rng.normal(size=3); v -= v.dot(u) * u; v /= np.linalg.norm(v)
        x1, x2 = c1 * u, c2 * (math.cos(th) * u + math.sin(th) * v)
        tr, tm = r9 / 400.0 * nr, mu9 * nm
        if r9 >= 399.0 or min(tr % 1, 1 - tr % 1, tm % 1, 1 - tm % 1) < 1e-6:
            continue
        cell = int(tr) * nm + min(int(tm), nm - 1)
        for opts in (dict(force_refine=1), None):
            out, _ = _run(runner, "rmu", tuple(np.array([x1, x2]).T), None, b2, dict(mode="none"), opts)
            hh = out["DD"][0]
            assert hh.sum() == 1 and hh[cell] == 1, (r9, mu9, opts)
        checked += 1
    assert checked > 40


@pytest.mark.parametrize("grid", ["none", "box3d"])
def test_weighted_3d_kinds(rt, oracle, grid):
    """integer weights per object for the 3-D kinds (PAPER.md:233 generalised): a pair counts w_i w_j,
    the w objects of one point w(w-1)/2 pairs at zero separation -- weighted C5-like DD/DR (periodic box, float32), weighted
    (r,mu) and (pi,sigma) on comoving float64 coordinates, brute force and cell lists, heavy weights, force_refine"""
    api, runner, synth = rt
    rng = np.random.default_rng(43)
    w5 = synth.workload(5, 0.0008)
    nd, nr = len(w5.data[0]), len(w5.rand[0])
    wd, wr = rng.integers(1, 9, nd).astype(np.uint32), rng.integers(1, 4, nr).astype(np.uint32)
    g5 = dict(mode="none") if grid == "none" else w5.grid
    job = runner.Job("monopole", w5.data, w5.rand, w5.bins, g5, None, w_data=wd, w_rand=wr).build()
    for which, a, b, wa, wb in (("DD", w5.data, None, wd, None), ("DR", w5.data, w5.rand, wd, wr)):
        h, st = job.count(which)
        orc = oracle.count("monopole", a, b, w5.bins, mode="celled", w1=wa, w2=wb)
        ok, msg = oracle.parity_ok(h, orc)
        assert ok, f"monopole {which}: {msg}"
    job.opts = api.count_opts(force_refine=1)
    h2, _ = job.count("DR")
    job.opts = None
    assert np.array_equal(h2, job.count("DR")[0])
    # the weighted count of unit weights is the unweighted count
    one = runner.Job("monopole", w5.data, None, w5.bins, g5, None, w_data=np.ones(nd, dtype=np.uint32)).build()
    plain = runner.Job("monopole", w5.data, None, w5.bins, g5).build()
    assert np.array_equal(one.count("DD")[0], plain.count("DD")[0])
    # heavy weights: short uint32 epochs
    wh = rng.integers(1, 300, nd).astype(np.uint32)
    job = runner.Job("monopole", w5.data, None, w5.bins, g5, None, w_data=wh).build()
    h, st = job.count("DD")
    ok, msg = oracle.parity_ok(h, oracle.count("monopole", w5.data, None, w5.bins, mode="celled", w1=wh))
    assert ok, msg
    h_heavy = h
    # (r, mu) and (pi, sigma) on C3-like comoving coordinates
    w3 = synth.workload(3, 0.012)
    n3d, n3r = len(w3.data[0]), len(w3.rand[0])
    v1, v2 = rng.integers(1, 6, n3d).astype(np.uint32), rng.integers(1, 3, n3r).astype(np.uint32)
    g3 = dict(mode="none") if grid == "none" else w3.grid
    for kind, bins in (("rmu", w3.bins), ("pisigma", dict(w3.bins, n1=24, hi1=120.0, n2=24, lo2=0.0, hi2=120.0))):
        g = dict(g3, rmax=math.hypot(bins["hi1"], bins["hi2"])) if (kind == "pisigma" and grid != "none") else g3
        job = runner.Job(kind, w3.data, w3.rand, bins, g, None, w_data=v1, w_rand=v2).build()
        for which, a, b, wa, wb in (("DD", w3.data, None, v1, None), ("DR", w3.data, w3.rand, v1, v2)):
            h, st = job.count(which)
            orc = oracle.count(kind, a, b, bins, mode="celled", w1=wa, w2=wb)
            ok, msg = oracle.parity_ok(h, orc)
            assert ok, f"{kind} {which}: {msg}"
    # the end-to-end host entry point carries the weights too
    hh, _ = api.cute_count_pairs_host(api.MONOPOLE, w5.data, None, api.COORD_XYZ, job_spec_for(api, w5, g5), w5.bins, w1=wh)
    assert np.array_equal(hh, h_heavy)


def job_spec_for(api, w, grid):
    if grid.get("mode", "none") == "none":
        return api.grid_spec("none")
    L = w.bins["box_L"]
    return api.grid_spec("box3d", periodic=True, size=(L, L, L), rmax=grid["rmax"])


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_density_grid_monopole(rt, oracle, dtype):
    """N4 (Eq. 17): TSC overdensity field and grid-point correlation against the float64 oracle.
    Float64 on both sides, so the tolerance is the order of the additions: 1e-12 on delta, 1e-10 (absolute, in units of
    <delta^2>) on xi; the numbers of grid-point pairs per bin are integers and must be equal."""
    import torch
    api, runner, synth = rt
    L, n, ng = 200.0, 30000, 48
    x = synth.thomas_box(n, L, 3.0, 10.0, 99, dtype)
    cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in x]
    for bins in (dict(n1=12, lo1=0.0, hi1=60.0), dict(n1=9, lo1=3.0, hi1=80.0, log1=1), dict(n1=40, lo1=0.0, hi1=10.0)):
        out = api.cute_density_grid_xi(cols, L, ng, bins, want_delta=True)
        orc = oracle.density_grid_xi(tuple(np.asarray(c, dtype=np.float64) for c in x), L, ng, bins)
        d = out["delta"].cpu().numpy()
        assert np.max(np.abs(d - orc["delta"])) < 1e-12 * max(1.0, np.abs(orc["delta"]).max())
        assert np.array_equal(out["npairs"], orc["npairs"])
        var = float((orc["delta"] ** 2).mean())
        assert np.max(np.abs(out["xi"] - orc["xi"])) < 1e-10 * max(1.0, var)
        assert (out["status"] == api.WARN_EMPTY_BIN) == (orc["empty"] > 0)
    # mass conservation on the device: <delta> = 0
    assert abs(float(out["delta"].mean())) < 1e-12
    # grids whose rows are whole 8-point lane segments take the register-tiled stencil (16, 8 and 4 lanes per row)
    for ng2, hi in ((64, 30.0), (32, 40.0), (128, 10.0)):
        bins = dict(n1=10, lo1=0.0, hi1=hi)
        out = api.cute_density_grid_xi(cols, L, ng2, bins)
        orc = oracle.density_grid_xi(tuple(np.asarray(c, dtype=np.float64) for c in x), L, ng2, bins)
        assert np.array_equal(out["npairs"], orc["npairs"])
        var = float((orc["delta"] ** 2).mean())
        assert np.max(np.abs(out["xi"] - orc["xi"])) < 1e-10 * max(1.0, var)
    # validation: r_max beyond L/2, a non-xyz catalogue
    with pytest.raises(api.CuteError):
        api.cute_density_grid_xi(cols, L, ng, dict(n1=4, lo1=0.0, hi1=120.0))


def test_periodic_point_one_ulp_below_the_upper_face(rt):
    """a float64 coordinate just below L whose product with 1/cell rounds up to nc is a legal point of the periodic
    box [0, L): it joins the last cell; x = L itself is refused"""
    import torch
    api, runner, synth = rt
    L = 1000.0
    x_top = np.nextafter(L, 0.0)
    nc = next(n for n in range(3, 400) if x_top * (n / L) >= n)      # the rounding the fast path trips over
    rng = np.random.default_rng(5)
    pts = rng.uniform(0.0, L, size=(3, 500))
    pts[0, 0] = pts[1, 1] = pts[2, 2] = x_top
    cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in pts]
    spec = api.grid_spec("box3d", periodic=True, size=(L, L, L), ncell=(nc, nc, nc), rmax=0.9 * L / nc)
    g = api.cute_make_grid(cols, api.COORD_XYZ, spec)
    inf = g.info()
    ws = g.workspace
    off = inf.d_cell_start - ws.data_ptr()
    cs = ws[off:off + (inf.ncells + 1) * 4].view(torch.int32).cpu().numpy().astype(np.int64)
    k = np.minimum(np.floor(pts / (L / nc)).astype(np.int64), nc - 1)
    cid = (k[2] * nc + k[1]) * nc + k[0]
    assert np.array_equal(cs, np.concatenate([[0], np.cumsum(np.bincount(cid, minlength=nc ** 3))]))
    pts[0, 0] = L
    cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in pts]
    with pytest.raises(api.CuteError) as err:
        api.cute_make_grid(cols, api.COORD_XYZ, spec)
    assert err.value.status == -6


@pytest.mark.parametrize("bad", [float("nan"), float("inf"), -float("inf"), 1.0e30, -1.0, 2000.0])
@pytest.mark.parametrize("mode,build_path", [("box3d", 1), ("box3d", 2), ("none", 1)])
def test_bad_coordinates_are_refused(rt, bad, mode, build_path):
    """NaN / Inf / out-of-box coordinates give CUTE_ERR_POINT_OUT_OF_BOX and write nothing outside the
    workspace (the bytes after it keep their pattern); the box of PAPER.md:206 here is given explicitly, [0, 1000)^3"""
    import torch
    api, runner, synth = rt
    if mode == "none" and np.isfinite(bad):
        pytest.skip("brute force has no box: every finite point is legal")
    rng = np.random.default_rng(11)
    pts = rng.uniform(0.0, 1000.0, size=(3, 3000))
    pts[1, 1234] = bad
    cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in pts]
    spec = api.grid_spec(mode, size=(1000.0,) * 3 if mode == "box3d" else (0, 0, 0), ncell=(8, 8, 8) if mode == "box3d" else (0, 0, 0),
                         rmax=100.0 if mode == "box3d" else 0.0, build_path=build_path)
    cat, keep = api._catalog(cols, api.COORD_XYZ, True)
    nbytes = api.cute_grid_workspace_bytes(cat, spec)
    guard = 4096
    ws = torch.full((nbytes + 256 + guard,), 0x5A, dtype=torch.uint8, device="cuda")
    off = (-ws.data_ptr()) % 256
    # hand the library exactly nbytes: whatever lies behind must survive
    sub = ws[off:off + nbytes]
    with pytest.raises(api.CuteError) as err:
        api.cute_make_grid(cols, api.COORD_XYZ, spec, workspace=sub)
    assert err.value.status == -6
    torch.cuda.synchronize()
    assert bool((ws[off + nbytes:] == 0x5A).all()) and bool((ws[:off] == 0x5A).all())


_SHARD_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_1210_1833_b200 import api, runner, synth
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
r, world = dist.get_rank(), dist.get_world_size()
out = {}
cats = np.load(sys.argv[3])
for cfg, scale in ((5, 0.003), (2, 0.02)):
    w = synth.workload(cfg, scale)
    # the parent's catalogues, bit for bit (the generators use BLAS, whose rounding may depend on the threads a process gets)
    w.data = tuple(cats[f"C{cfg}_d{k}"] for k in range(len(w.data)))
    w.rand = tuple(cats[f"C{cfg}_r{k}"] for k in range(len(w.rand)))
    def share(t):                                     # rank 0's cell-sorted arrays to every rank (gloo: through the host)
        c = t.cpu()
        dist.broadcast(c, src=0)
        t.copy_(c)
    job = runner.job_for_workload(w).build(share=share)   # catalogues replicated, grids identical on every rank
    for which in w.pairs:
        g1, g2 = job.grids(which)
        n = api.cute_count_items(job.kind, g1, g2, job.counter)
        b, e = api.cute_shard_items(n, g1.info().nchunks, r, world, w.grid.get("mode", "none") == "none" and g2 is None)
        job.opts = api.count_opts(item_begin=b, item_end=e, shard=1)
        h, st = job.count(which)                      # the real pair kernel on this rank's share of the items
        t = torch.from_numpy(h.astype(np.int64))
        dist.all_reduce(t)                            # the one exchange step: sum of the partial histograms
        out[f"C{cfg}_{which}"] = t.numpy()
        out[f"C{cfg}_{which}_items"] = np.array([b, e, n])
if r == 0:
    np.savez(sys.argv[2], **out)
dist.destroy_process_group()
"""


def test_two_processes_count_their_shards_with_the_real_kernel(rt, tmp_path):
    """two processes on the one GPU, each counting its cute_shard_items share with the real pair kernel (no
    kernel waits on another process), partial uint64 histograms summed with a gloo all-reduce (the sum
    of private histograms) == the single-process histogram, for a cell-list cross/auto count and a brute-force triangle"""
    import os
    import subprocess
    import sys
    api, runner, synth = rt
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    script = tmp_path / "shard_worker.py"
    script.write_text(_SHARD_WORKER)
    res, cats = tmp_path / "res.npz", tmp_path / "cats.npz"
    ws = {cfg: synth.workload(cfg, scale) for cfg, scale in ((5, 0.003), (2, 0.02))}
    np.savez(cats, **{f"C{cfg}_{t}{k}": c for cfg, w in ws.items() for t, cat in (("d", w.data), ("r", w.rand)) for k, c in enumerate(cat)})
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29573", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script), root, str(res), str(cats)], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT) for r in range(2)]
    outs = [p.communicate(timeout=600)[0].decode() for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o
    got = np.load(res)
    for cfg, w in ws.items():
        job = runner.job_for_workload(w).build()
        for which in w.pairs:
            h, st = job.count(which)
            assert np.array_equal(got[f"C{cfg}_{which}"].astype(np.uint64), h), (cfg, which)
            b, e, n = got[f"C{cfg}_{which}_items"]
            assert 0 < e <= n and b == 0                  # rank 0's share is a proper, non-empty prefix
            assert e < n
