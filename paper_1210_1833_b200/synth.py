"""Seeded synthetic catalogues for the five BASELINE.json workloads (C1..C5).

This module is the ONLY code shared by the CUDA path and the oracle: it produces inputs and
nothing else.  It holds none of the method's arithmetic (no separations, no bins, no cell
lists, no estimators) and imports neither `oracle/` nor the CUDA binding.

The paper's own workloads are a MICE mock subset, the PTHalos mocks
 and a log-normal mock; none of them is available here, so
BASELINE.json's five synthetic configurations stand in for them.  The recipe (SURVEY.md
section 8(d) D0, restated in DESIGN.md "Input recipe"):

* generator: ``numpy.random.default_rng(seed)`` (PCG64),
  ``seed = 12101833*100 + 10*config + {0: data, 1: randoms}``;
* C1  N=20 000 uniform in [0,1000)^3 Mpc/h, float64, periodic;
* C2  data 200 000 Thomas process (Poisson(10) children, Gaussian sigma=0.1 deg per
      tangent-plane axis) on a 1000 sq-deg cap centred (RA 180, Dec +30); randoms 400 000
      uniform on the same cap; RA/Dec in degrees, float64;
* C3  data 500 000 3-D Thomas process (sigma=5 Mpc/h per axis, Poisson(10) children) in the
      comoving volume of a 5000 sq-deg cap, 0.4<z<0.7, flat LCDM Om=0.3; randoms 1 000 000
      uniform in the same volume; RA/Dec/z float64 -> comoving xyz float64 on the host;
* C4  N=2 000 000, RA/Dec uniform on the 5000 sq-deg cap, z ~ N(0.7, 0.2^2) truncated to
      [0.2, 1.2];
* C5  data 10 000 000 Thomas process (sigma=5 Mpc/h) in the periodic box [0,2000)^3,
      float32 (cast, then re-wrapped so that no coordinate equals L); randoms 10 000 000
      uniform, float32.

Every function takes explicit sizes so that the tests can run the same recipes at sizes the
oracle finishes in seconds.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 12101833 * 100
C_OVER_H0 = 2997.92458  # Mpc/h
DEFAULT_CENTER = (180.0, 30.0)  # RA, Dec of the cap centre, degrees


def seed_for(config: int, which: int) -> int:
    """seed = 12101833*100 + 10*config + which (0 data, 1 randoms)."""
    return SEED_BASE + 10 * int(config) + int(which)


def cap_radius_deg(area_sqdeg: float) -> float:
    """Opening angle of a spherical cap of the given area (1000 -> 17.9141, 5000 -> 40.7475)."""
    return math.degrees(math.acos(1.0 - area_sqdeg * (math.pi / 180.0) ** 2 / (2.0 * math.pi)))


# ----------------------------------------------------------------------------- boxes
def uniform_box(n: int, L: float, seed: int, dtype=np.float64) -> np.ndarray:
    """n points uniform in [0,L)^3; returns an array of shape (3, n) (SoA)."""
    rng = np.random.default_rng(seed)
    x = rng.random((3, n)) * L
    return _finish_box(x, L, dtype)


def _finish_box(x: np.ndarray, L: float, dtype) -> np.ndarray:
    x = np.mod(x, L)
    x = x.astype(dtype)
    # casting to float32 may round up to exactly L: re-wrap
    x[x >= dtype(L)] = dtype(0.0)
    return np.ascontiguousarray(x)


def thomas_box(n: int, L: float, sigma: float, mean_children: float, seed: int,
               dtype=np.float64) -> np.ndarray:
    """Thomas cluster process in a periodic box: Poisson parents, Poisson(mean_children)
    children each, isotropic Gaussian offsets (sigma per axis), wrapped; first n kept."""
    rng = np.random.default_rng(seed)
    out = []
    have = 0
    while have < n:
        npar = int((n - have) / mean_children * 1.05) + 16
        par = rng.random((3, npar)) * L
        nch = rng.poisson(mean_children, npar)
        idx = np.repeat(np.arange(npar), nch)
        ch = par[:, idx] + rng.normal(0.0, sigma, (3, idx.size))
        out.append(ch)
        have += ch.shape[1]
    x = np.concatenate(out, axis=1)[:, :n]
    return _finish_box(x, L, dtype)


# ----------------------------------------------------------------------------- sphere
def _rot_to_center(v: np.ndarray, center) -> np.ndarray:
    """Rotate vectors given relative to the north pole so that the pole goes to `center`."""
    ra0, dec0 = math.radians(center[0]), math.radians(center[1])
    colat = math.pi / 2 - dec0
    cy, sy = math.cos(colat), math.sin(colat)
    cz, sz = math.cos(ra0), math.sin(ra0)
    x, y, z = v
    x1 = cy * x + sy * z
    z1 = -sy * x + cy * z
    x2 = cz * x1 - sz * y
    y2 = sz * x1 + cz * y
    return np.stack([x2, y2, z1])


def _vec_to_radec(v: np.ndarray):
    x, y, z = v
    r = np.sqrt(x * x + y * y + z * z)
    dec = np.degrees(np.arcsin(np.clip(z / r, -1.0, 1.0)))
    ra = np.mod(np.degrees(np.arctan2(y, x)), 360.0)
    ra[ra >= 360.0] = 0.0
    return ra, dec


def _radec_to_vec(ra, dec) -> np.ndarray:
    a, d = np.radians(ra), np.radians(dec)
    cd = np.cos(d)
    return np.stack([cd * np.cos(a), cd * np.sin(a), np.sin(d)])


def _uniform_cap_vec(rng, n: int, radius_deg: float) -> np.ndarray:
    """Unit vectors uniform on a cap of the given radius about the north pole."""
    cmin = math.cos(math.radians(radius_deg))
    ct = cmin + (1.0 - cmin) * rng.random(n)
    st = np.sqrt(np.maximum(0.0, 1.0 - ct * ct))
    ph = 2.0 * math.pi * rng.random(n)
    return np.stack([st * np.cos(ph), st * np.sin(ph), ct])


def uniform_cap(n: int, area_sqdeg: float, seed: int, center=DEFAULT_CENTER):
    """(ra, dec) in degrees, uniform on a cap of the given area."""
    rng = np.random.default_rng(seed)
    v = _rot_to_center(_uniform_cap_vec(rng, n, cap_radius_deg(area_sqdeg)), center)
    return _vec_to_radec(v)


def thomas_cap(n: int, area_sqdeg: float, sigma_deg: float, mean_children: float, seed: int,
               center=DEFAULT_CENTER):
    """Thomas process on a cap: parents uniform on the cap, Poisson children, Gaussian offsets
    of sigma_deg per tangent-plane axis, children outside the cap dropped, first n kept."""
    rng = np.random.default_rng(seed)
    rad = cap_radius_deg(area_sqdeg)
    cmin = math.cos(math.radians(rad))
    sig = math.radians(sigma_deg)
    out = []
    have = 0
    while have < n:
        npar = int((n - have) / mean_children * 1.1) + 16
        p = _uniform_cap_vec(rng, npar, rad)
        nch = rng.poisson(mean_children, npar)
        idx = np.repeat(np.arange(npar), nch)
        pp = p[:, idx]
        # tangent basis at each parent
        e1 = np.stack([-pp[1], pp[0], np.zeros_like(pp[0])])
        nrm = np.sqrt((e1 * e1).sum(0))
        bad = nrm < 1e-12
        e1[:, bad] = np.array([[1.0], [0.0], [0.0]])
        nrm[bad] = 1.0
        e1 /= nrm
        e2 = np.cross(pp.T, e1.T).T
        off = rng.normal(0.0, sig, (2, idx.size))
        c = pp + off[0] * e1 + off[1] * e2
        c /= np.sqrt((c * c).sum(0))
        c = c[:, c[2] >= cmin]
        out.append(c)
        have += c.shape[1]
    v = np.concatenate(out, axis=1)[:, :n]
    return _vec_to_radec(_rot_to_center(v, center))


# ----------------------------------------------------------------------------- cosmology (host side, A20)
def _chi_table(om: float, zmax: float, nstep: int = 1 << 15):
    z = np.linspace(0.0, zmax, nstep + 1)
    inv_e = 1.0 / np.sqrt(om * (1.0 + z) ** 3 + (1.0 - om))
    h = z[1] - z[0]
    # composite Simpson on successive pairs, cumulative
    mid = 1.0 / np.sqrt(om * (1.0 + (z[:-1] + 0.5 * h)) ** 3 + (1.0 - om))
    seg = h / 6.0 * (inv_e[:-1] + 4.0 * mid + inv_e[1:])
    chi = np.concatenate([[0.0], np.cumsum(seg)]) * C_OVER_H0
    return z, chi


def lcdm_chi(z, om: float = 0.3):
    """Comoving distance in Mpc/h for flat LCDM (h drops out in Mpc/h units).
    chi(0.4) = 1086.08, chi(0.7) = 1753.99 for om = 0.3."""
    z = np.asarray(z, dtype=np.float64)
    zt, ct = _chi_table(om, max(float(z.max(initial=0.0)) * 1.0001, 1e-3))
    return np.interp(z, zt, ct)


def lcdm_z_of_chi(chi, om: float = 0.3, zmax: float = 3.0):
    zt, ct = _chi_table(om, zmax)
    return np.interp(np.asarray(chi, dtype=np.float64), ct, zt)


def radecz_to_xyz(ra, dec, z, om: float = 0.3) -> np.ndarray:
    """Host-side z -> chi(z) and projection; shape (3, n) float64."""
    return _radec_to_vec(ra, dec) * lcdm_chi(z, om)


def uniform_cap_shell(n: int, area_sqdeg: float, zmin: float, zmax: float, seed: int,
                      om: float = 0.3, center=DEFAULT_CENTER):
    """Uniform in the comoving volume of cap x [zmin, zmax]; returns ra, dec, z, xyz."""
    rng = np.random.default_rng(seed)
    c0, c1 = lcdm_chi(np.array([zmin, zmax]), om)
    chi = np.cbrt(c0 ** 3 + (c1 ** 3 - c0 ** 3) * rng.random(n))
    v = _rot_to_center(_uniform_cap_vec(rng, n, cap_radius_deg(area_sqdeg)), center)
    ra, dec = _vec_to_radec(v)
    z = lcdm_z_of_chi(chi, om)
    return ra, dec, z, radecz_to_xyz(ra, dec, z, om)


def thomas_cap_shell(n: int, area_sqdeg: float, zmin: float, zmax: float, sigma: float,
                     mean_children: float, seed: int, om: float = 0.3, center=DEFAULT_CENTER):
    """3-D Thomas process in the comoving volume of cap x [zmin, zmax] (children outside the
    footprint dropped); returns ra, dec, z, xyz."""
    rng = np.random.default_rng(seed)
    rad = cap_radius_deg(area_sqdeg)
    cmin = math.cos(math.radians(rad))
    c0, c1 = lcdm_chi(np.array([zmin, zmax]), om)
    out = []
    have = 0
    while have < n:
        npar = int((n - have) / mean_children * 1.15) + 16
        chi = np.cbrt(c0 ** 3 + (c1 ** 3 - c0 ** 3) * rng.random(npar))
        p = _uniform_cap_vec(rng, npar, rad) * chi
        nch = rng.poisson(mean_children, npar)
        idx = np.repeat(np.arange(npar), nch)
        c = p[:, idx] + rng.normal(0.0, sigma, (3, idx.size))
        r = np.sqrt((c * c).sum(0))
        keep = (r >= c0) & (r < c1) & (c[2] >= cmin * r)
        out.append(c[:, keep])
        have += int(keep.sum())
    x = np.concatenate(out, axis=1)[:, :n]
    x = _rot_to_center(x, center)
    ra, dec = _vec_to_radec(x)
    z = lcdm_z_of_chi(np.sqrt((x * x).sum(0)), om)
    return ra, dec, z, radecz_to_xyz(ra, dec, z, om)


def gaussian_nz_cap(n: int, area_sqdeg: float, zmean: float, zsig: float, zmin: float,
                    zmax: float, seed: int, center=DEFAULT_CENTER):
    """RA/Dec uniform on the cap, z ~ N(zmean, zsig^2) truncated to [zmin, zmax] by rejection."""
    rng = np.random.default_rng(seed)
    v = _rot_to_center(_uniform_cap_vec(rng, n, cap_radius_deg(area_sqdeg)), center)
    ra, dec = _vec_to_radec(v)
    z = np.empty(0)
    while z.size < n:
        t = rng.normal(zmean, zsig, int((n - z.size) * 1.2) + 16)
        z = np.concatenate([z, t[(t >= zmin) & (t < zmax)]])
    return ra, dec, np.ascontiguousarray(z[:n])


# ----------------------------------------------------------------------------- the five workloads
def uniform_wedge(n: int, ra_max: float, dec_max: float, zmin: float, zmax: float, seed: int, om: float = 0.3):
    """Uniform in the comoving volume of the wedge 0 < RA < ra_max, 0 < Dec < dec_max, zmin < z < zmax: the footprint of
    the MICE subset the paper times in Table II (the mock itself is not available).  Returns ra, dec, z, xyz."""
    rng = np.random.default_rng(seed)
    ra = ra_max * rng.random(n)
    dec = np.degrees(np.arcsin(math.sin(math.radians(dec_max)) * rng.random(n)))
    c0, c1 = lcdm_chi(np.array([zmin, zmax]), om)
    chi = np.cbrt(c0 ** 3 + (c1 ** 3 - c0 ** 3) * rng.random(n))
    z = lcdm_z_of_chi(chi, om)
    return ra, dec, z, radecz_to_xyz(ra, dec, z, om)


@dataclass
class Workload:
    """One BASELINE.json configuration: catalogues + the binning it is counted with.

    `kind` is one of "monopole", "angular", "rmu", "radial"; `data`/`rand` are tuples of
    float arrays in the coordinates of that kind (xyz | ra,dec (deg) | ra,dec,z);
    `bins` holds n1, lo1, hi1, log1, n2, lo2, hi2, aperture, box_L in the units of the kind's
    variable: Mpc/h for r, RADIANS for theta and the aperture (catalogue RA/Dec are degrees).
    """
    name: str
    kind: str
    data: tuple
    rand: tuple | None
    bins: dict
    pairs: tuple = ("DD",)
    grid: dict = field(default_factory=dict)
    notes: str = ""


def workload(config: int, scale: float = 1.0) -> Workload:
    """BASELINE.json config 1..5.  scale<1 shrinks the catalogue sizes (and, for the box
    configs, the box volume so that the number density is kept) for tests."""
    s = float(scale)
    if config == 1:
        n = max(8, int(round(20000 * s)))
        L = 1000.0
        x = uniform_box(n, L, seed_for(1, 0))
        return Workload("C1", "monopole", tuple(x), None,
                        dict(n1=50, lo1=0.0, hi1=150.0, log1=0, n2=0, lo2=0.0, hi2=0.0,
                             aperture=0.0, box_L=L), ("DD",), dict(mode="none"),
                        "periodic brute force; RR analytic")
    if config == 2:
        nd, nr = max(8, int(round(200000 * s))), max(8, int(round(400000 * s)))
        d = thomas_cap(nd, 1000.0, 0.1, 10.0, seed_for(2, 0))
        r = uniform_cap(nr, 1000.0, seed_for(2, 1))
        return Workload("C2", "angular", d, r,
                        dict(n1=64, lo1=math.radians(1e-3), hi1=math.radians(10.0), log1=1, n2=0,
                             lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0), ("DD", "DR", "RR"),
                        dict(mode="none"), "64 log bins 1e-3..10 deg (limits in radians); brute force")
    if config == 3:
        nd, nr = max(8, int(round(500000 * s))), max(8, int(round(1000000 * s)))
        d = thomas_cap_shell(nd, 5000.0, 0.4, 0.7, 5.0, 10.0, seed_for(3, 0))
        r = uniform_cap_shell(nr, 5000.0, 0.4, 0.7, seed_for(3, 1))
        return Workload("C3", "rmu", tuple(d[3]), tuple(r[3]),
                        dict(n1=40, lo1=0.0, hi1=200.0, log1=0, n2=50, lo2=0.0, hi2=1.0,
                             aperture=0.0, box_L=0.0), ("DD", "DR", "RR"),
                        dict(mode="box3d", rmax=200.0), "mid-point line of sight")
    if config == 4:
        n = max(8, int(round(2000000 * s)))
        ra, dec, z = gaussian_nz_cap(n, 5000.0, 0.7, 0.2, 0.2, 1.2, seed_for(4, 0))
        return Workload("C4", "radial", (ra, dec, z), None,
                        dict(n1=20, lo1=0.2, hi1=1.2, log1=0, n2=64, lo2=0.0, hi2=0.05,
                             aperture=math.radians(1.0 / 60.0), box_L=0.0), ("DD",),
                        dict(mode="sphere", thetamax=math.radians(1.0 / 60.0)),
                        "aperture 1 arcmin (in radians)")
    if config == 5:
        n = max(8, int(round(10000000 * s)))
        L = 2000.0 * s ** (1.0 / 3.0)
        d = thomas_box(n, L, 5.0, 10.0, seed_for(5, 0), np.float32)
        r = uniform_box(n, L, seed_for(5, 1), np.float32)
        hi = min(200.0, L / 2.0 * 0.8)
        return Workload("C5", "monopole", tuple(d), tuple(r),
                        dict(n1=40, lo1=0.0, hi1=hi, log1=0, n2=0, lo2=0.0, hi2=0.0,
                             aperture=0.0, box_L=L), ("DD", "DR"),
                        dict(mode="box3d", rmax=hi), "float32 positions; 3-D cell list")
    raise ValueError("config must be 1..5")
