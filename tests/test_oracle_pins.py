"""Pins of the oracle: closed forms, exact enumerations, invariants.

None of these re-types the oracle's formula or calls it twice: each compares it with something
the paper or the mathematics fixes independently.  CPU only.
"""
import itertools
import math

import numpy as np
import pytest

from conftest import load_golden
from paper_1210_1833_b200 import synth

GOLDEN = ["monopole_345.txt", "monopole_periodic.txt", "monopole_cross.txt", "angular_equator.txt",
          "angular_log.txt", "rmu_345.txt", "rmu_los.txt", "radial_ladder.txt"]


def _cat(pts):
    a = np.array(pts, dtype=np.float64).T
    return tuple(a) if a.shape[0] == 3 else (a[0], a[1], np.zeros_like(a[0]))


# ---------------------------------------------------------------- V3 hand-enumerated catalogues
@pytest.mark.parametrize("name", GOLDEN)
@pytest.mark.parametrize("mode", ["plain", "celled"])
def test_golden_hand_enumerated(oracle, name, mode):
    kind, bins, pts, pts2, expect = load_golden(name)
    res = oracle.count(kind, _cat(pts), _cat(pts2) if pts2 else None, bins, mode=mode)
    want = np.zeros_like(res["hist"])
    for k, v in expect.items():
        want[k] = v
    assert np.array_equal(res["hist"], want), (name, res["hist"].nonzero(), res["hist"][res["hist"] > 0])
    # hand fixtures keep every separation away from the edges except r = 0 / mu = 0,1 on outer edges
    assert res["amb_cell"][:-1].sum() <= 2 * 2


# ---------------------------------------------------------------- V2 exact lattice counts
def test_lattice_periodic_exact(oracle):
    """Points on an n^3 lattice in a periodic box: DD_k = N/2 * #{integer vectors v in the torus with
    h|v| in bin k}; the vectors are enumerated here, independently of the oracle (Eq. 11, PAPER.md:85;
    periodic wrap PAPER.md:94)."""
    n, h = 6, 1.5
    L = n * h
    g = np.arange(n) * h + 0.25  # offset: the lattice need not sit on the box corner
    x = np.array(list(itertools.product(g, g, g))).T
    rng = np.random.default_rng(5)
    x = x[:, rng.permutation(x.shape[1])]
    bins = dict(n1=29, lo1=0.05 * h, hi1=2.95 * h, box_L=L)
    edges = bins["lo1"] + (bins["hi1"] - bins["lo1"]) * np.arange(30) / 29
    want = np.zeros(29, dtype=np.int64)
    rep = range(-n // 2, n // 2)  # torus representatives [-n/2, n/2)
    for v in itertools.product(rep, rep, rep):
        m = v[0] ** 2 + v[1] ** 2 + v[2] ** 2
        if m == 0:
            continue
        # minimum image of component -n/2 has the same |.|, so |v| is the minimum-image distance
        r = h * math.sqrt(m)
        k = np.searchsorted(edges, r, side="right") - 1
        if 0 <= k < 29 and r < edges[-1]:
            want[k] += 1
    N = n ** 3
    assert np.all((want * N) % 2 == 0)
    want = want * N // 2
    for mode in ("plain", "celled"):
        res = oracle.count("monopole", tuple(x), None, bins, mode=mode)
        assert np.array_equal(res["hist"].astype(np.int64), want)
        assert res["amb_cell"].sum() == 0  # lattice distances sit far from the edges


# ---------------------------------------------------------------- V1 analytic RR (statistical)
def test_analytic_rr_uniform_periodic_box(oracle):
    """C1 itself: uniform N=20000 in [0,1000)^3, E[DD_k] = N(N-1)/2 * 4pi/3 (e_{k+1}^3-e_k^3)/L^3
    (north star (a); Eqs. 12-13)."""
    w = synth.workload(1)
    N = w.data[0].size
    res = oracle.count("monopole", w.data, None, w.bins, mode="plain")
    e = np.linspace(0.0, 150.0, 51)
    rr = N * (N - 1) / 2 * 4 * math.pi / 3 * (e[1:] ** 3 - e[:-1] ** 3) / 1000.0 ** 3
    dd = res["hist"].astype(np.float64)
    pull = (dd - rr) / np.sqrt(rr)
    assert np.all(np.abs(pull) < 5.0), pull
    chi2 = float((pull ** 2).mean())
    assert 0.4 < chi2 < 1.8, chi2
    assert res["npairs"] == N * (N - 1) // 2
    # the oracle's own periodic_rr is the same closed form
    assert np.allclose(oracle.periodic_rr(N, 1000.0, w.bins), rr, rtol=1e-13)
    # and celled mode (27 cells, wrap) agrees exactly on the same catalogue
    res2 = oracle.count("monopole", w.data, None, w.bins, mode="celled")
    assert np.array_equal(res2["hist"], res["hist"])


# ---------------------------------------------------------------- V4 totals, symmetry, permutation
def test_totals_and_symmetries(oracle):
    rng = np.random.default_rng(11)
    a = tuple(rng.random((3, 700)) * 50.0)
    b = tuple(rng.random((3, 450)) * 50.0 + 10.0)
    wide = dict(n1=37, lo1=0.0, hi1=200.0)
    assert oracle.count("monopole", a, None, wide)["hist"].sum() == 700 * 699 // 2
    hab = oracle.count("monopole", a, b, wide)["hist"]
    hba = oracle.count("monopole", b, a, wide)["hist"]
    assert hab.sum() == 700 * 450
    assert np.array_equal(hab, hba)
    p = rng.permutation(700)
    ap = tuple(c[p] for c in a)
    fine = dict(n1=64, lo1=0.0, hi1=30.0)
    assert np.array_equal(oracle.count("monopole", a, None, fine)["hist"],
                          oracle.count("monopole", ap, None, fine)["hist"])
    # rmu: totals with bins covering everything (mu in [0,1] closed top)
    shift = tuple(c + 1000.0 for c in a)
    rm = dict(n1=7, lo1=0.0, hi1=200.0, n2=9, lo2=0.0, hi2=1.0)
    assert oracle.count("rmu", shift, None, rm)["hist"].sum() == 700 * 699 // 2
    # angular: theta in [0, pi] covers every pair
    ra, dec = synth.uniform_cap(600, 30000.0, 3)
    ang = dict(n1=50, lo1=0.0, hi1=3.2)
    assert oracle.count("angular", (ra, dec), None, ang)["hist"].sum() == 600 * 599 // 2
    # periodic translation invariance (up to the flagged pairs)
    L = 50.0
    per = dict(n1=20, lo1=0.0, hi1=25.0, box_L=L)
    h0 = oracle.count("monopole", a, None, per)
    a2 = tuple(np.mod(c + 17.3, L) for c in a)
    h1 = oracle.count("monopole", a2, None, per)
    ok, msg = oracle.parity_ok(h1["hist"], h0)
    assert ok, msg


# ---------------------------------------------------------------- V5 additivity
@pytest.mark.parametrize("kind", ["monopole", "angular", "rmu", "radial"])
def test_additivity_auto_cross(oracle, kind):
    """auto(A u B) = auto(A) + auto(B) + cross(A, B) per bin (follows from Eq. 11)."""
    rng = np.random.default_rng(21)
    if kind in ("monopole", "rmu"):
        pts = rng.random((3, 900)) * 60.0 + (500.0 if kind == "rmu" else 0.0)
        bins = dict(n1=12, lo1=0.0, hi1=30.0)
        if kind == "rmu":
            bins.update(n2=5, lo2=0.0, hi2=1.0)
    else:
        ra, dec = synth.uniform_cap(900, 4.0, 8)
        z = 0.2 + rng.random(900)
        pts = np.stack([ra, dec, z])
        if kind == "angular":
            bins = dict(n1=16, lo1=math.radians(0.01), hi1=math.radians(1.5), log1=1)
        else:
            bins = dict(n1=5, lo1=0.2, hi1=1.2, n2=8, lo2=0.0, hi2=0.4, aperture=math.radians(0.1))
    A, B = tuple(pts[:, :500]), tuple(pts[:, 500:])
    full = oracle.count(kind, tuple(pts), None, bins)["hist"]
    parts = (oracle.count(kind, A, None, bins)["hist"] + oracle.count(kind, B, None, bins)["hist"]
             + oracle.count(kind, A, B, bins)["hist"])
    assert full.sum() > 100
    assert np.array_equal(full, parts)


# ---------------------------------------------------------------- V6 celled == plain
def test_celled_equals_plain_all_kinds(oracle):
    rng = np.random.default_rng(31)
    # periodic monopole, clustered
    x = synth.thomas_box(3000, 120.0, 2.0, 8.0, 77)
    y = synth.uniform_box(2500, 120.0, 78)
    b = dict(n1=25, lo1=0.0, hi1=17.0, box_L=120.0)
    for c2 in (None, tuple(y)):
        p = oracle.count("monopole", tuple(x), c2, b, mode="plain")
        c = oracle.count("monopole", tuple(x), c2, b, mode="celled")
        assert np.array_equal(p["hist"], c["hist"]) and np.array_equal(p["amb_cell"], c["amb_cell"])
        assert c["npairs"] < p["npairs"]
    # non-periodic rmu with different bounding boxes for the two catalogues
    a = tuple(rng.random((3, 2000)) * 80.0 + 900.0)
    bb = tuple(rng.random((3, 1500)) * 100.0 + 880.0)
    rb = dict(n1=10, lo1=0.0, hi1=12.0, n2=6, lo2=0.0, hi2=1.0)
    for c2 in (None, bb):
        p = oracle.count("rmu", a, c2, rb, mode="plain")
        c = oracle.count("rmu", a, c2, rb, mode="celled")
        assert np.array_equal(p["hist"], c["hist"])
    # angular: footprint straddling RA = 0/360 and one containing the pole
    for center in ((0.5, 10.0), (120.0, 89.2), (200.0, -89.5)):
        ra, dec = synth.uniform_cap(2500, 40.0, 5, center=center)
        ra2, dec2 = synth.thomas_cap(2000, 40.0, 0.05, 6.0, 6, center=center)
        ab = dict(n1=20, lo1=math.radians(0.003), hi1=math.radians(0.8), log1=1)
        for c2 in (None, (ra2, dec2)):
            p = oracle.count("angular", (ra, dec), c2, ab, mode="plain")
            c = oracle.count("angular", (ra, dec), c2, ab, mode="celled")
            assert p["hist"].sum() > 1000
            assert np.array_equal(p["hist"], c["hist"]), center
    # radial
    ra, dec, z = synth.gaussian_nz_cap(6000, 3.0, 0.7, 0.2, 0.2, 1.2, 9)
    rb = dict(n1=6, lo1=0.2, hi1=1.2, n2=10, lo2=0.0, hi2=0.3, aperture=math.radians(2.0 / 60))
    p = oracle.count("radial", (ra, dec, z), None, rb, mode="plain")
    c = oracle.count("radial", (ra, dec, z), None, rb, mode="celled")
    assert p["hist"].sum() > 50
    assert np.array_equal(p["hist"], c["hist"])


def test_islice_partitions_the_count(oracle):
    """i-slices (used by the timed CPU baseline and the sharding test) add up to the whole."""
    x = tuple(synth.uniform_box(1500, 100.0, 3))
    b = dict(n1=10, lo1=0.0, hi1=40.0, box_L=100.0)
    full = oracle.count("monopole", x, None, b)["hist"]
    parts = sum(oracle.count("monopole", x, None, b, i_range=r, mode=m)["hist"]
                for r, m in (((0, 400), "plain"), ((400, 1100), "celled"), ((1100, 1500), "plain")))
    assert np.array_equal(full, parts)


# ---------------------------------------------------------------- V7 theta: chord route == arccos route, paper's series
def test_theta_equals_arccos_of_dot(oracle):
    """theta = arccos(n1.n2) (Eq. 7) computed independently with numpy for theta > 1 deg,
    where arccos is well conditioned, must land in the oracle's bins."""
    ra, dec = synth.uniform_cap(900, 8000.0, 13, center=(40.0, -20.0))
    bins = dict(n1=59, lo1=math.radians(1.0), hi1=math.radians(60.0))
    res = oracle.count("angular", (ra, dec), None, bins)
    a, d = np.radians(ra), np.radians(dec)
    n = np.stack([np.cos(d) * np.cos(a), np.cos(d) * np.sin(a), np.sin(d)])
    dot = np.clip(n.T @ n, -1.0, 1.0)
    iu = np.triu_indices(ra.size, 1)
    th = np.arccos(dot[iu])
    want, _ = np.histogram(th, bins=np.linspace(bins["lo1"], bins["hi1"], 60))
    ok, msg = oracle.parity_ok(want, res)  # arccos is only good to ~1e-15/sin(theta): allow flagged pairs
    assert ok, msg
    assert want.sum() > 50000


def test_paper_arccos_series_pins_chord_mapping():
    """arccos(1-x) ~ sqrt(2x + x^2/3 + 4x^3/45), '1 part in 10^4 below 40 deg'.
    With x = chord^2/2 this pins theta = 2 asin(chord/2) <-> chord^2 = 4 sin^2(theta/2)."""
    for deg, tol in ((0.5, 1e-12), (10.0, 1e-7), (40.0, 2e-4)):
        th = math.radians(deg)
        chord2 = 4.0 * math.sin(th / 2) ** 2
        x = chord2 / 2.0
        assert abs(x - (1.0 - math.cos(th))) < 1e-15
        series = math.sqrt(2 * x + x * x / 3 + 4 * x ** 3 / 45)
        assert abs(series / th - 1.0) < tol
        assert abs(2.0 * math.asin(math.sqrt(chord2) / 2.0) / th - 1.0) < 1e-14


# ---------------------------------------------------------------- V8 Eq. 9 identity
def test_rmu_matches_eq9(oracle):
    """r(z1,z2,theta), mu(z1,z2,theta) of Eq. 9 fix the mid-point line of sight."""
    rng = np.random.default_rng(41)
    nr, nm = 64, 64
    bins = dict(n1=nr, lo1=0.0, hi1=400.0, n2=nm, lo2=0.0, hi2=1.0)
    checked = 0
    for _ in range(300):
        c1, c2 = 1000.0 + 600.0 * rng.random(2)
        th = 0.15 * rng.random()
        r9 = math.sqrt(c1 * c1 + c2 * c2 - 2 * c1 * c2 * math.cos(th))
        mu9 = abs(c1 * c1 - c2 * c2) / math.sqrt((c1 * c1 + c2 * c2) ** 2 - 4 * c1 * c1 * c2 * c2 * math.cos(th) ** 2)
        # two directions separated by theta, randomly oriented
        u = rng.normal(size=3); u /= np.linalg.norm(u)
        v = rng.normal(size=3); v -= v.dot(u) * u; v /= np.linalg.norm(v)
        x1 = c1 * u
        x2 = c2 * (math.cos(th) * u + math.sin(th) * v)
        res = oracle.count("rmu", tuple(np.array([x1, x2]).T), None, bins)
        if r9 >= 400.0:
            assert res["hist"].sum() == 0
            continue
        tr, tm = r9 / 400.0 * nr, mu9 * nm
        if min(tr % 1, 1 - tr % 1, tm % 1, 1 - tm % 1) < 1e-6:
            continue
        cell = int(tr) * nm + min(int(tm), nm - 1)
        assert res["hist"][cell] == 1, (r9, mu9)
        checked += 1
    assert checked > 200


# ---------------------------------------------------------------- V9 / V10 estimators
def test_landy_szalay_algebra_and_poisson(oracle):
    rng = np.random.default_rng(51)
    dd = rng.integers(1, 10 ** 6, 40).astype(np.uint64)
    dr = rng.integers(1, 10 ** 6, 40).astype(np.uint64)
    rr = rng.integers(1, 10 ** 6, 40).astype(np.uint64)
    nd, nr = 12345, 67890
    xi, empty = oracle.landy_szalay(dd, dr, rr, nd, nr)
    ndd, ndr, nrr = nd * (nd - 1) / 2, nd * nr, nr * (nr - 1) / 2
    ref = (dd / ndd - 2 * dr / ndr + rr / nrr) / (rr / nrr)  # normalised-counts form (derived from Eq. 15)
    assert empty == 0 and np.allclose(xi, ref, rtol=1e-12, atol=1e-12)
    xin, _ = oracle.natural(dd, rr, nd, nr)
    assert np.allclose(xin, (dd / ndd) / (rr / nrr) - 1, rtol=1e-12)
    rr0 = rr.copy(); rr0[3] = 0
    xi0, empty0 = oracle.landy_szalay(dd, dr, rr0, nd, nr)
    assert empty0 == 1 and xi0[3] == 0.0
    # Poisson data and randoms on the same footprint: xi ~ 0 (north star (d))
    d = tuple(rng.random((3, 3000)) * 100.0)
    r = tuple(rng.random((3, 6000)) * 100.0)
    b = dict(n1=10, lo1=2.0, hi1=30.0)
    DD = oracle.count("monopole", d, None, b)["hist"]
    DR = oracle.count("monopole", d, r, b)["hist"]
    RR = oracle.count("monopole", r, None, b)["hist"]
    xi, _ = oracle.landy_szalay(DD, DR, RR, 3000, 6000)
    assert np.all(np.abs(xi) < 5.0 * (1.0 + np.abs(xi)) / np.sqrt(DD.astype(float))), xi


# ---------------------------------------------------------------- edges, half-open bins, ambiguity flags
def test_edges_and_halfopen_bins(oracle):
    b = dict(n1=8, lo1=1e-3, hi1=10.0, log1=1)
    e = oracle.edges(b)
    assert e[0] == 1e-3 and e[-1] == 10.0
    assert np.allclose(e, 1e-3 * (10.0 / 1e-3) ** (np.arange(9) / 8), rtol=1e-14)
    bl = dict(n1=5, lo1=1.0, hi1=6.0)
    assert np.array_equal(oracle.edges(bl), [1, 2, 3, 4, 5, 6])
    # a pair exactly on an edge belongs to the upper bin; r = hi is out; r = lo is in
    def one(r):
        return oracle.count("monopole", (np.array([0.0, r]), np.zeros(2), np.zeros(2)), None, bl)
    assert one(3.0)["hist"].tolist() == [0, 0, 1, 0, 0]
    assert one(6.0)["hist"].sum() == 0
    assert one(1.0)["hist"].tolist() == [1, 0, 0, 0, 0]
    assert one(0.999)["hist"].sum() == 0
    # flags: within relative 2^-20 of an edge -> both neighbouring cells (or the virtual out cell)
    r = one(3.0 * (1 + 2.0 ** -21))
    assert r["amb_cell"].tolist() == [0, 1, 1, 0, 0, 0] and r["amb_e1"].tolist() == [0, 0, 1, 0, 0, 0]
    r = one(3.0 * (1 + 2.0 ** -19))
    assert r["amb_cell"].sum() == 0
    r = one(6.0 * (1 - 2.0 ** -21))
    assert r["hist"][4] == 1 and r["amb_cell"].tolist() == [0, 0, 0, 0, 1, 1]
    r = one(1.0 * (1 - 2.0 ** -21))
    assert r["hist"].sum() == 0 and r["amb_cell"].tolist() == [1, 0, 0, 0, 0, 1]
    # parity rule helper
    ok, _ = oracle.parity_ok(np.array([1, 0, 0, 0, 0]), r)
    assert ok
    ok, _ = oracle.parity_ok(np.array([0, 1, 0, 0, 0]), r)
    assert not ok


def test_radial_aperture_is_strict_and_flagged(oracle):
    ap = math.radians(1.0 / 60)
    b = dict(n1=2, lo1=0.0, hi1=2.0, n2=2, lo2=0.0, hi2=1.0, aperture=ap)
    def pair(sep_rad):
        return oracle.count("radial", (np.array([10.0, 10.0]), np.array([0.0, math.degrees(sep_rad)]),
                                       np.array([0.5, 0.8])), None, b)
    assert pair(ap * 0.999)["hist"].tolist() == [1, 0, 0, 0]
    assert pair(ap * 1.001)["hist"].sum() == 0
    r = pair(ap * (1 + 2.0 ** -22))
    assert r["amb_cell"][0] == 1 and r["amb_cell"][-1] == 1 and r["amb_e2"][-1] == 1


# ------------------------------------------------------------------------------- N1: (pi, sigma) and multipoles
def test_pisigma_fixture(oracle):
    kind, bins, pts, pts2, expect = load_golden("pisigma_los.txt")
    cat = tuple(np.array(c) for c in zip(*pts))
    r = oracle.count(kind, cat, None, bins)
    want = np.zeros(r["hist"].size, dtype=np.uint64)
    for k, v in expect.items():
        want[k] = v
    assert np.array_equal(r["hist"], want)


def test_pisigma_is_the_geometric_decomposition(oracle):
    """V11: Eq. 2, pi = r mu and sigma = sqrt(r^2 - pi^2), must equal the geometric definition:
    pi = |s . l^| (component of the separation along the unit mid-point vector) and sigma = |s - (s.l^) l^|
    (the perpendicular component), computed here with numpy from scratch."""
    rng = np.random.default_rng(11)
    n = 400
    x = rng.normal(size=(n, 3)) * 30.0 + np.array([0.0, 200.0, 900.0])
    bins = dict(n1=13, lo1=0.0, hi1=60.0, n2=11, lo2=0.0, hi2=70.0)
    r = oracle.count("pisigma", tuple(x.T.copy()), None, bins)
    i, j = np.triu_indices(n, 1)
    s = x[i] - x[j]
    lv = x[i] + x[j]
    lhat = lv / np.linalg.norm(lv, axis=1)[:, None]
    par = np.einsum("ij,ij->i", s, lhat)
    perp = np.linalg.norm(s - par[:, None] * lhat, axis=1)
    h, _, _ = np.histogram2d(np.abs(par), perp, bins=[oracle.edges(bins, 0), oracle.edges(bins, 1)])
    ok, msg = oracle.parity_ok(h.astype(np.int64).ravel(), r)
    assert ok, msg
    assert r["hist"].sum() > 1000
    # bins that cover every separation: total = N(N-1)/2 (V4)
    big = dict(n1=3, lo1=0.0, hi1=1e4, n2=3, lo2=0.0, hi2=1e4)
    assert oracle.count("pisigma", tuple(x.T.copy()), None, big)["hist"].sum() == n * (n - 1) // 2


def test_pisigma_celled_equals_plain(oracle):
    rng = np.random.default_rng(12)
    x = rng.random((3, 3000)) * 300.0 + 500.0
    y = rng.random((3, 2000)) * 300.0 + 500.0
    bins = dict(n1=8, lo1=0.0, hi1=40.0, n2=8, lo2=0.0, hi2=30.0)
    for c2 in (None, tuple(y)):
        a = oracle.count("pisigma", tuple(x), c2, bins, mode="plain")
        b = oracle.count("pisigma", tuple(x), c2, bins, mode="celled")
        assert np.array_equal(a["hist"], b["hist"]) and b["npairs"] < a["npairs"]


def test_multipoles_closed_form(oracle):
    """Eq. 3-4: xi(r,mu) = xi_0 + xi_2 P_2(mu) + xi_4 P_4(mu) must give back xi_0, xi_2, xi_4
    (mid-point rule over 50 mu bins: error O(1/n_mu^2)); a mu-independent xi has only a monopole, exactly."""
    n_r, n_mu = 7, 50
    mu = (np.arange(n_mu) + 0.5) / n_mu
    p2, p4 = 0.5 * (3 * mu**2 - 1), (35 * mu**4 - 30 * mu**2 + 3) / 8
    a, b, c = np.linspace(1, 2, n_r), np.linspace(-0.5, 0.5, n_r), np.linspace(0.1, 0.3, n_r)
    xi = a[:, None] + b[:, None] * p2[None, :] + c[:, None] * p4[None, :]
    m = oracle.multipoles(xi, n_r, n_mu)
    assert np.allclose(m[0], a, atol=2e-3) and np.allclose(m[1], b, atol=5e-3) and np.allclose(m[2], c, atol=1e-2)
    m = oracle.multipoles(np.full((n_r, n_mu), 0.7), n_r, n_mu)
    assert np.allclose(m[0], 0.7, atol=1e-14) and np.allclose(m[1], 0, atol=2e-3) and np.allclose(m[2], 0, atol=2e-3)


# ------------------------------------------------------------------------------- N2: weights and pixel maps
@pytest.mark.parametrize("kind", ["angular", "monopole", "rmu"])
def test_weights_are_repeated_objects(oracle, kind):
    """reading P2: a catalogue with integer weights gives exactly the counts of the catalogue in which object i is
    repeated w_i times (the copies of one object being w(w-1)/2 pairs at zero separation), auto and cross, plain and celled"""
    rng = np.random.default_rng(31)
    n1, n2 = 300, 200
    if kind == "angular":
        c1 = (rng.random(n1) * 6 + 10, rng.random(n1) * 6 - 3)
        c2 = (rng.random(n2) * 6 + 10, rng.random(n2) * 6 - 3)
        bins = dict(n1=12, lo1=0.0, hi1=math.radians(2.0))
    else:
        c1 = tuple(rng.random((3, n1)) * 100 + 300)
        c2 = tuple(rng.random((3, n2)) * 100 + 300)
        bins = dict(n1=10, lo1=0.0, hi1=40.0)
        if kind == "rmu":
            bins.update(n2=5, lo2=0.0, hi2=1.0)
        else:
            bins.update(box_L=0.0)
    w1, w2 = rng.integers(1, 5, n1), rng.integers(1, 4, n2)
    e1 = tuple(np.repeat(c, w1) for c in c1)
    e2 = tuple(np.repeat(c, w2) for c in c2)
    for mode in ("plain", "celled"):
        a = oracle.count(kind, c1, None, bins, mode=mode, w1=w1)
        b = oracle.count(kind, e1, None, bins, mode=mode)
        assert np.array_equal(a["hist"], b["hist"]) and a["hist"][0] >= (w1 * (w1 - 1) // 2).sum()
        a = oracle.count(kind, c1, c2, bins, mode=mode, w1=w1, w2=w2)
        b = oracle.count(kind, e1, e2, bins, mode=mode)
        assert np.array_equal(a["hist"], b["hist"])
    ones = oracle.count(kind, c1, c2, bins, w1=np.ones(n1, dtype=np.uint32), w2=np.ones(n2, dtype=np.uint32))
    assert np.array_equal(ones["hist"], oracle.count(kind, c1, c2, bins)["hist"])


def test_pixel_map(oracle):
    """reading P1: pixels with constant limits in (RA, sin dec), represented by their centres"""
    # 2 x 2 pixels over RA [0,20) x sin(dec) [0,0.5): centres RA 5, 15; sin(dec) 0.125, 0.375 -> dec 7.18076, 22.02431 deg
    ra = np.array([1.0, 2.0, 19.0, 11.0, 3.0])
    dec = np.array([1.0, 14.0, 16.0, 29.0, 2.0])       # sin: 0.0175, 0.2419, 0.2756, 0.4848, 0.0349
    pra, pdec, pw = oracle.pixelize(ra, dec, 0.0, 20.0, 0.0, 0.5, 2, 2)
    assert np.allclose(pra, [5.0, 15.0]) and np.allclose(pdec, [7.18076, 22.02431], atol=1e-5)
    assert list(pw) == [3, 2]                          # (1,1) (2,14) (3,2) below sin = 0.25 at RA < 10; (19,16) (11,29) above, RA > 10
    rng = np.random.default_rng(5)
    n = 5000
    ra = (355.0 + rng.random(n) * 12.0) % 360.0        # across the RA = 0 seam
    dec = np.degrees(np.arcsin(rng.random(n) * 0.4 - 0.2))
    nra, nu = 24, 20
    pra, pdec, pw = oracle.pixelize(ra, dec, 355.0, 12.0, -0.2, 0.4, nra, nu)
    assert pw.sum() == n and len(pw) <= nra * nu
    # every object lies inside the pixel that counts it: rebuild the counts from the centres
    kx = np.floor(((ra - 355.0) % 360.0) / (12.0 / nra)).astype(int)
    ky = np.floor((np.sin(np.radians(dec)) + 0.2) / (0.4 / nu)).astype(int)
    cx = np.floor(((pra - 355.0) % 360.0) / (12.0 / nra)).astype(int)
    cy = np.floor((np.sin(np.radians(pdec)) + 0.2) / (0.4 / nu)).astype(int)
    want = np.bincount(ky * nra + kx, minlength=nra * nu)
    assert np.array_equal(want[cy * nra + cx], pw) and want.sum() == pw.sum()
    with pytest.raises(ValueError):
        oracle.pixelize(np.array([30.0]), np.array([0.0]), 0.0, 20.0, -0.5, 1.0, 4, 4)   # outside the map


def test_pixelised_counts_approach_the_exact_ones_above_the_pixel_scale(oracle):
    """"if one is not interested in extremely small angular scales": w_pix pair counts agree with the
    object counts at separations well above the pixel size, and differ below it"""
    rng = np.random.default_rng(9)
    n = 6000
    ra = rng.random(n) * 20.0 + 100.0
    dec = np.degrees(np.arcsin(rng.random(n) * 0.3))
    pra, pdec, pw = oracle.pixelize(ra, dec, 100.0, 20.0, 0.0, 0.3, 100, 86)       # ~0.2 deg pixels
    bins = dict(n1=8, lo1=math.radians(1.0), hi1=math.radians(5.0))
    exact = oracle.count("angular", (ra, dec), None, bins)["hist"].astype(float)
    pix = oracle.count("angular", (pra, pdec), None, bins, w1=pw)["hist"].astype(float)
    assert np.all(np.abs(pix / exact - 1.0) < 0.04) and np.abs(pix.sum() / exact.sum() - 1.0) < 0.005
    small = dict(n1=4, lo1=0.0, hi1=math.radians(0.1))
    a = oracle.count("angular", (ra, dec), None, small)["hist"]
    b = oracle.count("angular", (pra, pdec), None, small, w1=pw)["hist"]
    assert b[0] == (pw.astype(np.int64) * (pw.astype(np.int64) - 1) // 2).sum() and b[1:].sum() == 0 and a[1:].sum() > 0


# ---------------------------------------------------------------- 2-D ambiguity cells (parity rule)
def _rmu_pair(r, mu, chi=1000.0):
    """two points whose mid-point line of sight is the z axis exactly: s = r (sqrt(1-mu^2), 0, mu), l = 2 chi z"""
    t = math.sqrt(max(0.0, 1.0 - mu * mu))
    return (np.array([0.5 * r * t, -0.5 * r * t]), np.zeros(2), np.array([chi + 0.5 * r * mu, chi - 0.5 * r * mu]))


def test_amb_cell_composition_two_axes(oracle):
    """`amb_cell` of a 2-D histogram: every cell a flagged pair could land in when the flagged variable(s) cross their
    edge -- the product of the candidate bins of both axes, out-of-range candidates going to the virtual cell.  Hand
    cases on 10 x 10 bins of width 1 in r and 0.1 in mu (cell = 10 k_r + k_mu)."""
    b = dict(n1=10, lo1=0.0, hi1=10.0, n2=10, lo2=0.0, hi2=1.0)
    eps = 2.0 ** -21
    # (a) only mu on an edge: mu = 0.4 (1 + 2^-21) is in mu-bin 4 and could be in 3; r = 2.5 is unflagged
    res = oracle.count("rmu", _rmu_pair(2.5, 0.4 * (1 + eps)), None, b)
    assert res["hist"][24] == 1 and res["hist"].sum() == 1
    amb = res["amb_cell"]
    assert amb[24] == 1 and amb[23] == 1 and amb.sum() == 2
    assert res["amb_e2"][4] == 1 and res["amb_e1"].sum() == 0
    # (b) r and mu both on an edge: r = 3 (1 - 2^-21) in r-bin 2 (could be 3), mu as above: four cells
    res = oracle.count("rmu", _rmu_pair(3.0 * (1 - eps), 0.4 * (1 + eps)), None, b)
    assert res["hist"][24] == 1
    amb = res["amb_cell"]
    assert sorted(np.nonzero(amb)[0].tolist()) == [23, 24, 33, 34] and amb.sum() == 4
    assert res["amb_e1"][3] == 1 and res["amb_e2"][4] == 1
    # (c) the outermost r edge: r = 10 (1 - 2^-21) is counted in r-bin 9 and could be out of range (virtual cell 100)
    res = oracle.count("rmu", _rmu_pair(10.0 * (1 - eps), 0.55), None, b)
    assert res["hist"][95] == 1
    amb = res["amb_cell"]
    assert amb[95] == 1 and amb[100] == 1 and amb.sum() == 2
    # ... and from the other side: not counted, could be in cell 95
    res = oracle.count("rmu", _rmu_pair(10.0 * (1 + eps), 0.55), None, b)
    assert res["hist"].sum() == 0
    amb = res["amb_cell"]
    assert amb[95] == 1 and amb[100] == 1 and amb.sum() == 2
    # (d) the parity rule accepts each allowed placement and nothing else
    res = oracle.count("rmu", _rmu_pair(3.0 * (1 - eps), 0.4 * (1 + eps)), None, b)
    for cell in (23, 24, 33, 34):
        g = np.zeros(100, dtype=np.int64); g[cell] = 1
        assert oracle.parity_ok(g, res)[0]
    g = np.zeros(100, dtype=np.int64); g[25] = 1
    assert not oracle.parity_ok(g, res)[0]


def test_amb_cell_aperture_times_dz(oracle):
    """RADIAL: the aperture is an edge in theta; a pair within 2^-20 of it AND of a dz edge could be in either dz cell or
    not counted at all (virtual cell)."""
    ap = math.radians(1.0 / 60)
    b = dict(n1=2, lo1=0.0, hi1=2.0, n2=2, lo2=0.0, hi2=1.0, aperture=ap)
    dz = 0.5 * (1 - 2.0 ** -21)                     # dz-bin 0, could be 1
    def pair(sep_rad):
        return oracle.count("radial", (np.array([10.0, 10.0]), np.array([0.0, math.degrees(sep_rad)]),
                                       np.array([0.3, 0.3 + dz])), None, b)
    out = pair(ap * (1 + 2.0 ** -22))               # just outside the aperture: not counted
    assert out["hist"].sum() == 0
    assert out["amb_cell"].tolist() == [1, 1, 0, 0, 1]
    assert out["amb_e2"][1] == 1 and out["amb_e2"][3] == 1 and out["amb_e1"].sum() == 0
    inn = pair(ap * (1 - 2.0 ** -22))               # just inside: counted in (zbar-bin 0, dz-bin 0)
    assert inn["hist"].tolist() == [1, 0, 0, 0]
    assert inn["amb_cell"].tolist() == [1, 1, 0, 0, 1]


# ---------------------------------------------------------------- N4 density-grid monopole (Eq. 17)
def test_tsc_weights_closed_forms(oracle):
    """TSC (reading D2): a particle at a cell centre feeds (1/8, 3/4, 1/8) per axis; one on a cell face (1/2, 1/2, 0);
    the weights of any particle sum to 1 (mass conservation); a particle per cell centre gives rho = 1, delta = 0."""
    L, ng = 8.0, 8
    rho = oracle.tsc_assign((np.array([3.5]), np.array([3.5]), np.array([3.5])), L, ng)      # centre of cell (3,3,3)
    w = np.array([0.125, 0.75, 0.125])
    want = np.zeros((ng, ng, ng))
    want[2:5, 2:5, 2:5] = w[:, None, None] * w[None, :, None] * w[None, None, :]
    assert np.allclose(rho, want, atol=1e-15)
    rho = oracle.tsc_assign((np.array([4.0]), np.array([3.5]), np.array([3.5])), L, ng)      # on the face between x-cells 3 and 4
    assert np.allclose(rho[3, 3, 2:6], 0.75 * 0.75 * np.array([0.0, 0.5, 0.5, 0.0]), atol=1e-15)
    # periodic wrap: a particle in cell 0 reaches cell ng - 1
    rho = oracle.tsc_assign((np.array([0.5]), np.array([0.5]), np.array([0.5])), L, ng)
    assert abs(rho[0, 0, ng - 1] - 0.125 * 0.75 * 0.75) < 1e-15 and abs(rho.sum() - 1.0) < 1e-14
    rng = np.random.default_rng(7)
    x = rng.random((3, 5000)) * L
    rho = oracle.tsc_assign(tuple(x), L, ng)
    assert abs(rho.sum() - 5000.0) < 1e-9 and rho.min() >= 0.0
    g = (np.arange(ng) + 0.5) * (L / ng)
    lat = np.array(list(itertools.product(g, g, g))).T
    rho = oracle.tsc_assign(tuple(lat), L, ng)
    assert np.allclose(rho, 1.0, atol=1e-14)
    assert np.allclose(oracle.overdensity(rho, ng ** 3), 0.0, atol=1e-14)
    assert np.allclose(oracle.overdensity(2.0 * np.ones((4, 4, 4)), 128), 0.0)            # rho_bar = N / ng^3


def test_grid_correlation_of_a_plane_wave(oracle):
    """Eq. 17 on delta = A cos(k.x): (1/N) sum_g delta_g delta_{g+v} = A^2/2 cos(k.v) for a grid wave vector, so
    xi_k = A^2/2 * mean over the offsets of the shell of cos(k.v) -- the offsets are enumerated here, not by the oracle."""
    ng, L, A = 16, 32.0, 0.3
    h = L / ng
    kv = np.array([2, 1, 3])                                   # wave vector in units of 2 pi / L
    gz, gy, gx = np.meshgrid(np.arange(ng), np.arange(ng), np.arange(ng), indexing="ij")
    delta = A * np.cos(2 * np.pi * (kv[0] * gx + kv[1] * gy + kv[2] * gz) / ng)
    bins = dict(n1=6, lo1=0.0, hi1=12.0)
    e = np.linspace(0.0, 12.0, 7)
    want_s, want_n = np.zeros(6), np.zeros(6)
    m = int(12.0 // h)
    for dz, dy, dx in itertools.product(range(-m, m + 1), repeat=3):
        if dx == dy == dz == 0:
            continue
        r = h * math.sqrt(dx * dx + dy * dy + dz * dz)
        k = np.searchsorted(e, r, side="right") - 1
        if 0 <= k < 6 and r < e[-1]:
            want_s[k] += 0.5 * A * A * math.cos(2 * np.pi * (kv[0] * dx + kv[1] * dy + kv[2] * dz) / ng)
            want_n[k] += 1
    out = oracle.grid_correlation(delta, L, bins)
    assert np.array_equal(out["npairs"], (want_n * ng ** 3).astype(np.uint64))
    ok = want_n > 0
    assert ok.sum() == 5 and out["empty"] == 1 and out["xi"][0] == 0.0          # no offset is shorter than h = 2
    assert np.allclose(out["xi"][ok], want_s[ok] / want_n[ok], atol=1e-13)
    assert np.allclose(out["sum_dd"], want_s * ng ** 3, atol=1e-9)
    # a constant field correlates with itself everywhere; bins no offset reaches are reported empty
    out = oracle.grid_correlation(np.full((ng, ng, ng), 0.5), L, dict(n1=40, lo1=0.0, hi1=4.0))
    assert out["empty"] > 0 and np.all(out["xi"][out["npairs"] > 0] == 0.25) and np.all(out["xi"][out["npairs"] == 0] == 0.0)


def test_density_grid_agrees_with_pair_counts_above_the_grid_scale(oracle):
    """"it will only yield reliable results down to the scale of the grid": on a clustered periodic box
    (Thomas process, sigma = 3) the density-grid xi equals the pair-count xi of Eq. 13 at r >> h and is smoothed (lower)
    at r ~ h."""
    L, n, ng = 200.0, 30000, 64                                  # h = 3.125
    x = synth.thomas_box(n, L, 3.0, 10.0, 99)
    bins = dict(n1=10, lo1=0.0, hi1=50.0, box_L=L)
    dd = oracle.count("monopole", tuple(x), None, bins, mode="celled")["hist"].astype(float)
    xi_pairs = dd / oracle.periodic_rr(n, L, bins) - 1.0
    xi_grid = oracle.density_grid_xi(tuple(x), L, ng, dict(n1=10, lo1=0.0, hi1=50.0))["xi"]
    assert np.all(np.abs(xi_grid[3:] - xi_pairs[3:]) < 2e-3)                       # r > 15 = 5 h: the same function
    assert xi_pairs[0] > 1.0 and 0.9 * xi_pairs[0] < xi_grid[0] < xi_pairs[0]      # r < 5: the signal, a little smoothed
    assert 0.85 * xi_pairs[1] < xi_grid[1] < xi_pairs[1]
