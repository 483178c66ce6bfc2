"""ctypes front end of the ORACLE (oracle/cute_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this.  It neither imports nor is imported
by the CUDA path (paper_1210_1833_b200).  See the C file's header for what is computed and
the paper passages it follows.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "cute_oracle.c")
_LIB = os.path.join(_HERE, "libcute_oracle.so")

KINDS = {"angular": 0, "monopole": 1, "rmu": 2, "radial": 3, "pisigma": 4}

# float64, no FMA contraction, no fast-math: the arithmetic is the definition's
CFLAGS = ["-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-std=c11"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", *CFLAGS, "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Bins(C.Structure):
    _fields_ = [("n1", C.c_int), ("lo1", C.c_double), ("hi1", C.c_double), ("log1", C.c_int),
                ("n2", C.c_int), ("lo2", C.c_double), ("hi2", C.c_double),
                ("aperture", C.c_double), ("box_L", C.c_double)]


_lib = None


def _load():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        dp = C.POINTER(C.c_double)
        up = C.POINTER(C.c_uint64)
        _lib.orc_count.argtypes = [C.c_int, C.c_int, C.c_int64, dp, dp, dp, C.c_int64, dp, dp, dp,
                                   C.POINTER(_Bins), C.c_int64, C.c_int64, C.c_int, up, up, up, up, up]
        wp = C.POINTER(C.c_uint32)
        _lib.orc_count_w.argtypes = [C.c_int, C.c_int, C.c_int64, dp, dp, dp, wp, C.c_int64, dp, dp, dp, wp,
                                     C.POINTER(_Bins), C.c_int64, C.c_int64, C.c_int, up, up, up, up, up]
        _lib.orc_pixelize.argtypes = [C.c_int64, dp, dp, C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                      dp, dp, wp, C.POINTER(C.c_int64)]
        _lib.orc_edges.argtypes = [C.POINTER(_Bins), C.c_int, dp]
        _lib.orc_landy_szalay.argtypes = [up, up, up, C.c_uint64, C.c_uint64, C.c_int, dp]
        _lib.orc_natural.argtypes = [up, up, C.c_uint64, C.c_uint64, C.c_int, dp]
        _lib.orc_periodic_rr.argtypes = [C.c_uint64, C.c_double, C.POINTER(_Bins), dp]
        _lib.orc_multipoles.argtypes = [dp, C.c_int, C.c_int, dp]
        _lib.orc_tsc_assign.argtypes = [C.c_int64, dp, dp, dp, C.c_double, C.c_int, dp]
        _lib.orc_overdensity.argtypes = [C.c_int64, C.c_int, dp, dp]
        _lib.orc_grid_correlation.argtypes = [dp, C.c_int, C.c_double, C.POINTER(_Bins), dp, dp, up]
    return _lib


def _bins(b: dict) -> _Bins:
    return _Bins(int(b["n1"]), float(b["lo1"]), float(b["hi1"]), int(b.get("log1", 0)),
                 int(b.get("n2", 0)), float(b.get("lo2", 0.0)), float(b.get("hi2", 0.0)),
                 float(b.get("aperture", 0.0)), float(b.get("box_L", 0.0)))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _up(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def _cols(cat, kind):
    need = 2 if kind == "angular" else 3
    cols = [np.ascontiguousarray(np.asarray(c, dtype=np.float64)) for c in cat[:need]]
    while len(cols) < 3:
        cols.append(cols[0])
    return cols


def max_threads() -> int:
    return int(_load().orc_max_threads())


def edges(bins: dict, axis: int = 0) -> np.ndarray:
    b = _bins(bins)
    n = b.n1 if axis == 0 else b.n2
    e = np.zeros(n + 1)
    rc = _load().orc_edges(C.byref(b), axis, _dp(e))
    if rc:
        raise ValueError(f"orc_edges failed ({rc})")
    return e


def count(kind: str, cat1, cat2, bins: dict, mode: str = "plain", i_range=None, nthreads: int = 0, w1=None, w2=None):
    """Histogram of the pairs of cat1 x cat2 (cat2 None: unordered pairs of cat1).

    Returns dict(hist, amb_cell, amb_e1, amb_e2, npairs); hist has n1*max(n2,1) uint64 entries
    (first variable major); amb_cell has one extra trailing entry for the out-of-range cell.
    """
    lib = _load()
    b = _bins(bins)
    c1 = _cols(cat1, kind)
    n1 = c1[0].size
    if cat2 is None:
        c2, n2 = None, 0
    else:
        c2 = _cols(cat2, kind)
        n2 = c2[0].size
    ncell = b.n1 * max(b.n2, 1)
    hist = np.zeros(ncell, dtype=np.uint64)
    amb_cell = np.zeros(ncell + 1, dtype=np.uint64)
    amb_e1 = np.zeros(b.n1 + 1, dtype=np.uint64)
    amb_e2 = np.zeros(b.n2 + 2, dtype=np.uint64)
    npairs = np.zeros(1, dtype=np.uint64)
    i0, i1 = (0, n1) if i_range is None else i_range
    null = C.POINTER(C.c_double)()
    wnull = C.POINTER(C.c_uint32)()
    w1 = None if w1 is None else np.ascontiguousarray(np.asarray(w1, dtype=np.uint32))
    w2 = None if w2 is None else np.ascontiguousarray(np.asarray(w2, dtype=np.uint32))
    wptr = lambda w: wnull if w is None else w.ctypes.data_as(C.POINTER(C.c_uint32))
    rc = lib.orc_count_w(KINDS[kind], {"plain": 0, "celled": 1}[mode],
                       n1, _dp(c1[0]), _dp(c1[1]), _dp(c1[2]), wptr(w1),
                       n2, _dp(c2[0]) if c2 else null, _dp(c2[1]) if c2 else null, _dp(c2[2]) if c2 else null, wptr(w2),
                       C.byref(b), int(i0), int(i1), int(nthreads),
                       _up(hist), _up(amb_cell), _up(amb_e1), _up(amb_e2), _up(npairs))
    if rc:
        raise ValueError(f"orc_count failed ({rc})")
    return dict(hist=hist, amb_cell=amb_cell, amb_e1=amb_e1, amb_e2=amb_e2, npairs=int(npairs[0]))


def pixelize(ra, dec, ra0: float, dra: float, u0: float, du: float, n_ra: int, n_u: int):
    """Pixel map: centres (RA, Dec in degrees) and counts of the non-empty pixels."""
    ra = np.ascontiguousarray(np.asarray(ra, dtype=np.float64))
    dec = np.ascontiguousarray(np.asarray(dec, dtype=np.float64))
    npx = int(n_ra) * int(n_u)
    pra, pdec, pw = np.zeros(npx), np.zeros(npx), np.zeros(npx, dtype=np.uint32)
    m = C.c_int64(0)
    rc = _load().orc_pixelize(ra.size, _dp(ra), _dp(dec), float(ra0), float(dra), float(u0), float(du), int(n_ra), int(n_u),
                              _dp(pra), _dp(pdec), pw.ctypes.data_as(C.POINTER(C.c_uint32)), C.byref(m))
    if rc:
        raise ValueError(f"orc_pixelize failed ({rc})")
    return pra[:m.value].copy(), pdec[:m.value].copy(), pw[:m.value].copy()


def landy_szalay(dd, dr, rr, nd: int, nr: int):
    dd, dr, rr = (np.ascontiguousarray(np.asarray(a, dtype=np.uint64)).ravel() for a in (dd, dr, rr))
    xi = np.zeros(dd.size)
    empty = _load().orc_landy_szalay(_up(dd), _up(dr), _up(rr), int(nd), int(nr), dd.size, _dp(xi))
    return xi, int(empty)


def natural(dd, rr, nd: int, nr: int):
    dd, rr = (np.ascontiguousarray(np.asarray(a, dtype=np.uint64)).ravel() for a in (dd, rr))
    xi = np.zeros(dd.size)
    empty = _load().orc_natural(_up(dd), _up(rr), int(nd), int(nr), dd.size, _dp(xi))
    return xi, int(empty)


def periodic_rr(n: int, L: float, bins: dict) -> np.ndarray:
    b = _bins(bins)
    rr = np.zeros(b.n1)
    rc = _load().orc_periodic_rr(int(n), float(L), C.byref(b), _dp(rr))
    if rc:
        raise ValueError(f"orc_periodic_rr failed ({rc})")
    return rr


def multipoles(xi_rmu, n_r: int, n_mu: int) -> np.ndarray:
    """xi_0, xi_2, xi_4 of xi(r, mu) ([n_r][n_mu], mu in [0,1]); returns shape (3, n_r)."""
    xi = np.ascontiguousarray(np.asarray(xi_rmu, dtype=np.float64)).ravel()
    out = np.zeros((3, n_r))
    rc = _load().orc_multipoles(_dp(xi), int(n_r), int(n_mu), _dp(out))
    if rc:
        raise ValueError(f"orc_multipoles failed ({rc})")
    return out


def tsc_assign(cat, L: float, ng: int) -> np.ndarray:
    """TSC particle number per grid point, shape (ng, ng, ng) indexed [gz, gy, gx]."""
    c = [np.ascontiguousarray(np.asarray(a, dtype=np.float64)) for a in cat[:3]]
    rho = np.zeros(ng * ng * ng)
    rc = _load().orc_tsc_assign(c[0].size, _dp(c[0]), _dp(c[1]), _dp(c[2]), float(L), int(ng), _dp(rho))
    if rc:
        raise ValueError(f"orc_tsc_assign failed ({rc})")
    return rho.reshape(ng, ng, ng)


def overdensity(rho: np.ndarray, n: int) -> np.ndarray:
    ng = rho.shape[0]
    r = np.ascontiguousarray(rho, dtype=np.float64).ravel()
    d = np.zeros_like(r)
    rc = _load().orc_overdensity(int(n), int(ng), _dp(r), _dp(d))
    if rc:
        raise ValueError(f"orc_overdensity failed ({rc})")
    return d.reshape(ng, ng, ng)


def grid_correlation(delta: np.ndarray, L: float, bins: dict):
    """Eq. 17 on a periodic grid: dict(xi, sum_dd, npairs, empty)."""
    ng = delta.shape[0]
    d = np.ascontiguousarray(delta, dtype=np.float64).ravel()
    b = _bins(bins)
    xi, sdd, npr = np.zeros(b.n1), np.zeros(b.n1), np.zeros(b.n1, dtype=np.uint64)
    rc = _load().orc_grid_correlation(_dp(d), int(ng), float(L), C.byref(b), _dp(xi), _dp(sdd), _up(npr))
    if rc < 0:
        raise ValueError(f"orc_grid_correlation failed ({rc})")
    return dict(xi=xi, sum_dd=sdd, npairs=npr, empty=int(rc))


def density_grid_xi(cat, L: float, ng: int, bins: dict):
    """the whole density-grid monopole: TSC -> delta -> Eq. 17"""
    rho = tsc_assign(cat, L, ng)
    delta = overdensity(rho, len(cat[0]))
    out = grid_correlation(delta, L, bins)
    out["delta"] = delta
    return out


def parity_ok(gpu_hist, orc: dict):
    """The north star's parity rule: exact per cell and in total, except for flagged pairs.
    Returns (ok, message)."""
    g = np.asarray(gpu_hist).astype(np.int64).ravel()
    h = orc["hist"].astype(np.int64)
    amb = orc["amb_cell"].astype(np.int64)
    if g.size != h.size:
        return False, f"size {g.size} != {h.size}"
    d = np.abs(g - h)
    bad = np.nonzero(d > amb[:-1])[0]
    if bad.size:
        k = int(bad[0])
        return False, f"cell {k}: gpu {g[k]} oracle {h[k]} amb {amb[k]} ({bad.size} cells differ)"
    if abs(int(g.sum()) - int(h.sum())) > int(amb[-1]):
        return False, f"total: gpu {g.sum()} oracle {h.sum()} amb_out {amb[-1]}"
    return True, f"ok (sum {h.sum()}, cells differing within flags: {int((d > 0).sum())})"
