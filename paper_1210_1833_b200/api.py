"""Thin Python binding of the C ABI in include/cute_b200.h (same names, argument marshalling only).

PyTorch is used for device memory and streams; every step of the hot path runs inside
libcute_b200.so.  There is no CPU fallback: importing this module without the built library
raises, and so does calling it without a CUDA device.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libcute_b200.so")

ANGULAR, MONOPOLE, RMU, RADIAL, PISIGMA = 0, 1, 2, 3, 4
KINDS = {"angular": ANGULAR, "monopole": MONOPOLE, "rmu": RMU, "radial": RADIAL, "pisigma": PISIGMA}
COORD_XYZ, COORD_RADEC, COORD_RADECZ = 0, 1, 2
F32, F64 = 0, 1
GRID_NONE, GRID_BOX3D, GRID_SPHERE = 0, 1, 2
WARN_EMPTY_BIN = 1
ERR_STATIC_SCRATCH_LIMIT = -8
STATIC_SCRATCH_BYTES = 65536


class cute_catalog(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("n", C.c_int64), ("coord", C.c_int), ("dtype", C.c_int),
                ("c0", C.c_void_p), ("c1", C.c_void_p), ("c2", C.c_void_p), ("weight", C.c_void_p)]


class cute_grid_spec(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("mode", C.c_int), ("periodic", C.c_int),
                ("origin", C.c_double * 3), ("size", C.c_double * 3), ("ncell", C.c_int * 3),
                ("rmax", C.c_double), ("kind_mask", C.c_int), ("no_perm", C.c_int), ("build_path", C.c_int)]


class cute_bin_spec(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("n1", C.c_int), ("lo1", C.c_double), ("hi1", C.c_double),
                ("log1", C.c_int), ("n2", C.c_int), ("lo2", C.c_double), ("hi2", C.c_double),
                ("aperture_rad", C.c_double), ("box_L", C.c_double)]


class cute_count_opts(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("blocks", C.c_int), ("item_begin", C.c_int64),
                ("item_end", C.c_int64), ("tau_scale", C.c_double), ("force_refine", C.c_int),
                ("flush_items", C.c_int), ("warps", C.c_int), ("hist_cols", C.c_int), ("shard", C.c_int)]


class cute_grid_info(C.Structure):
    _fields_ = [("struct_size", C.c_size_t), ("n", C.c_int64), ("mode", C.c_int), ("periodic", C.c_int),
                ("kind_coord", C.c_int), ("dtype", C.c_int), ("has_lo", C.c_int), ("has_f64", C.c_int),
                ("ncell", C.c_int * 3), ("origin", C.c_double * 3), ("cell", C.c_double * 3), ("size", C.c_double * 3),
                ("ncells", C.c_int64), ("nrows", C.c_int64), ("nchunks", C.c_int64),
                ("d_hi", C.c_void_p), ("d_lo", C.c_void_p), ("d_perm", C.c_void_p),
                ("d_cell_start", C.c_void_p), ("build_bytes", C.c_double)]


# every symbol include/cute_b200.h declares
SYMBOLS = ["cute_version", "cute_strerror", "cute_launch_count", "cute_catalog_bounds", "cute_pixelize_workspace_bytes", "cute_pixelize", "cute_grid_workspace_bytes", "cute_make_grid", "cute_free_grid",
           "cute_grid_get_info", "cute_count_scratch_bytes", "cute_count_pairs", "cute_count_items",
           "cute_count_status", "cute_host_workspace_bytes", "cute_count_pairs_host", "cute_bin_edges",
           "cute_landy_szalay", "cute_natural_estimator", "cute_multipoles", "cute_periodic_rr", "cute_periodic_xi",
           "cute_peak_count", "cute_peak_name", "cute_measure_peaks", "cute_shard_items", "cute_auto_grid_spec",
           "cute_density_grid_workspace_bytes", "cute_density_grid_xi", "cute_count_pairs_static"]


def _load() -> C.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_1210_1833_b200.build` "
                          "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    vp, dp, up = C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_uint64)
    lib.cute_version.restype = C.c_int
    lib.cute_strerror.restype = C.c_char_p
    lib.cute_strerror.argtypes = [C.c_int]
    lib.cute_launch_count.restype = C.c_uint64
    lib.cute_catalog_bounds.argtypes = [C.POINTER(cute_catalog), vp, vp, dp]
    lib.cute_pixelize_workspace_bytes.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_size_t)]
    lib.cute_pixelize.argtypes = [C.POINTER(cute_catalog), C.c_double, C.c_double, C.c_double, C.c_double, C.c_int, C.c_int,
                                  vp, vp, vp, C.POINTER(C.c_int64), vp, C.c_size_t, vp]
    lib.cute_grid_workspace_bytes.argtypes = [C.POINTER(cute_catalog), C.POINTER(cute_grid_spec), C.POINTER(C.c_size_t)]
    lib.cute_make_grid.argtypes = [C.POINTER(cute_catalog), C.POINTER(cute_grid_spec), vp, C.c_size_t, vp, C.POINTER(vp)]
    lib.cute_free_grid.argtypes = [vp]
    lib.cute_free_grid.restype = None
    lib.cute_grid_get_info.argtypes = [vp, C.POINTER(cute_grid_info)]
    lib.cute_count_scratch_bytes.argtypes = [C.POINTER(cute_bin_spec), C.POINTER(cute_count_opts), C.POINTER(C.c_size_t)]
    lib.cute_count_pairs.argtypes = [C.c_int, vp, vp, C.POINTER(cute_bin_spec), vp, vp, C.c_size_t,
                                     C.POINTER(cute_count_opts), vp]
    lib.cute_count_items.argtypes = [C.c_int, vp, vp, C.POINTER(cute_bin_spec), C.POINTER(cute_count_opts), C.POINTER(C.c_int64)]
    lib.cute_count_status.argtypes = [vp, vp, up]
    lib.cute_count_pairs_static.argtypes = [C.c_int, vp, vp, C.POINTER(cute_bin_spec), vp, C.POINTER(cute_count_opts), vp, up]
    lib.cute_host_workspace_bytes.argtypes = [C.POINTER(cute_catalog), C.POINTER(cute_catalog), C.POINTER(cute_grid_spec),
                                              C.POINTER(cute_bin_spec), C.POINTER(C.c_size_t)]
    lib.cute_count_pairs_host.argtypes = [C.c_int, C.POINTER(cute_catalog), C.POINTER(cute_catalog), C.POINTER(cute_grid_spec),
                                          C.POINTER(cute_bin_spec), C.POINTER(cute_count_opts), up, vp, C.c_size_t, vp]
    lib.cute_shard_items.argtypes = [C.c_int64, C.c_int64, C.c_int, C.c_int, C.c_int, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
    lib.cute_auto_grid_spec.argtypes = [C.c_int, C.c_int, C.POINTER(C.POINTER(cute_catalog)), C.c_int, C.c_double, C.c_double,
                                        C.c_double, C.POINTER(C.c_int), C.c_int, vp, vp, C.POINTER(cute_grid_spec)]
    lib.cute_density_grid_workspace_bytes.argtypes = [C.c_int, C.POINTER(cute_bin_spec), C.c_double, C.POINTER(C.c_size_t)]
    lib.cute_density_grid_xi.argtypes = [C.POINTER(cute_catalog), C.c_double, C.c_int, C.POINTER(cute_bin_spec), dp, dp, up, vp, vp,
                                         C.c_size_t, vp]
    lib.cute_peak_count.restype = C.c_int
    lib.cute_peak_name.restype = C.c_char_p
    lib.cute_peak_name.argtypes = [C.c_int]
    lib.cute_measure_peaks.argtypes = [dp, dp, C.c_int, vp, C.c_size_t, vp]
    lib.cute_bin_edges.argtypes = [C.POINTER(cute_bin_spec), C.c_int, dp]
    lib.cute_landy_szalay.argtypes = [up, up, up, C.c_uint64, C.c_uint64, C.c_int, dp]
    lib.cute_natural_estimator.argtypes = [up, up, C.c_uint64, C.c_uint64, C.c_int, dp]
    lib.cute_multipoles.argtypes = [dp, C.c_int, C.c_int, dp]
    lib.cute_periodic_rr.argtypes = [C.c_uint64, C.c_double, C.POINTER(cute_bin_spec), dp]
    lib.cute_periodic_xi.argtypes = [up, C.c_uint64, C.c_double, C.POINTER(cute_bin_spec), dp]
    return lib


lib = _load()


class CuteError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__(f"{where}: {lib.cute_strerror(status).decode()} ({status})")


def _check(rc: int, where: str) -> int:
    if rc < 0:
        raise CuteError(rc, where)
    return rc


def cute_version() -> int:
    return int(lib.cute_version())


def cute_launch_count() -> int:
    return int(lib.cute_launch_count())


def cute_strerror(status: int) -> str:
    return lib.cute_strerror(int(status)).decode()


# ------------------------------------------------------------------------------- spec marshalling
def bin_spec(bins: dict) -> cute_bin_spec:
    """bins: n1, lo1, hi1, log1, n2, lo2, hi2, aperture (rad), box_L -- the dict synth.workload() gives."""
    return cute_bin_spec(C.sizeof(cute_bin_spec), int(bins["n1"]), float(bins["lo1"]), float(bins["hi1"]),
                         int(bins.get("log1", 0)), int(bins.get("n2", 0)), float(bins.get("lo2", 0.0)),
                         float(bins.get("hi2", 0.0)), float(bins.get("aperture", 0.0)), float(bins.get("box_L", 0.0)))


def grid_spec(mode="none", periodic=False, origin=(0, 0, 0), size=(0, 0, 0), ncell=(0, 0, 0), rmax=0.0,
              kind_mask=0, no_perm=0, build_path=0) -> cute_grid_spec:
    m = {"none": GRID_NONE, "box3d": GRID_BOX3D, "sphere": GRID_SPHERE}[mode] if isinstance(mode, str) else int(mode)
    return cute_grid_spec(C.sizeof(cute_grid_spec), m, int(bool(periodic)), (C.c_double * 3)(*map(float, origin)),
                          (C.c_double * 3)(*map(float, size)), (C.c_int * 3)(*map(int, ncell)), float(rmax), int(kind_mask), int(no_perm), int(build_path))


def count_opts(**kw) -> cute_count_opts:
    o = cute_count_opts()
    o.struct_size = C.sizeof(cute_count_opts)
    for k, v in kw.items():
        setattr(o, k, v)
    return o


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_1210_1833_b200 needs a CUDA device (there is no CPU fallback)")
    return torch


def _stream_ptr(stream=None) -> int:
    torch = _torch()
    s = stream if stream is not None else torch.cuda.current_stream()
    return int(s.cuda_stream)


def _catalog(cols, coord: int, device_ptrs: bool, weight=None):
    """cols: 2 or 3 arrays (torch CUDA tensors when device_ptrs, numpy otherwise), one dtype; weight: optional
    uint32 array of the same kind (torch int32 tensors carry the uint32 bits)."""
    need = 2 if coord == COORD_RADEC else 3
    cols = list(cols)[:need]
    if device_ptrs:
        torch = _torch()
        dt = F64 if cols[0].dtype == torch.float64 else F32
        assert all(c.is_cuda and c.is_contiguous() and c.dtype == cols[0].dtype for c in cols)
        ptrs = [c.data_ptr() for c in cols]
        n = cols[0].numel()
    else:
        dt = F64 if cols[0].dtype == np.float64 else F32
        assert all(c.flags.c_contiguous and c.dtype == cols[0].dtype for c in cols)
        ptrs = [c.ctypes.data for c in cols]
        n = cols[0].size
    while len(ptrs) < 3:
        ptrs.append(None)
    wptr = None
    if weight is not None:
        if device_ptrs:
            assert weight.is_cuda and weight.is_contiguous() and weight.element_size() == 4 and weight.numel() == n
            wptr = weight.data_ptr()
        else:
            assert weight.dtype == np.uint32 and weight.flags.c_contiguous and weight.size == n
            wptr = weight.ctypes.data
        cols = cols + [weight]
    return cute_catalog(C.sizeof(cute_catalog), n, coord, dt, *ptrs, wptr), cols


# ------------------------------------------------------------------------------- grids
class Grid:
    """Owns the torch workspace a cute_grid handle points into."""

    def __init__(self, handle, workspace, spec):
        self.handle, self.workspace, self.spec = handle, workspace, spec

    def info(self) -> cute_grid_info:
        inf = cute_grid_info()
        inf.struct_size = C.sizeof(cute_grid_info)
        _check(lib.cute_grid_get_info(self.handle, C.byref(inf)), "cute_grid_get_info")
        return inf

    def free(self):
        if self.handle:
            lib.cute_free_grid(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def cute_catalog_bounds(cols, coord: int, stream=None) -> np.ndarray:
    """min (3) and max (3) of the raw coordinate columns (torch CUDA tensors)."""
    torch = _torch()
    cat, keep = _catalog(cols, coord, True)
    tmp = torch.empty(16, dtype=torch.float64, device=keep[0].device)
    out = np.zeros(6)
    _check(lib.cute_catalog_bounds(C.byref(cat), C.c_void_p(tmp.data_ptr()), C.c_void_p(_stream_ptr(stream)), _dp(out)),
           "cute_catalog_bounds")
    return out


def cute_pixelize(cols, ra0: float, dra: float, u0: float, du: float, n_ra: int, n_u: int, stream=None):
    """Pixel map of a device RA/Dec catalogue: returns (ra, dec, weight) CUDA tensors of the non-empty
    pixels (float64 degrees, int32 counts)."""
    torch = _torch()
    cat, keep = _catalog(cols, COORD_RADEC, True)
    nb = C.c_size_t(0)
    _check(lib.cute_pixelize_workspace_bytes(int(n_ra), int(n_u), C.byref(nb)), "cute_pixelize_workspace_bytes")
    ws = torch.empty(nb.value + 256, dtype=torch.uint8, device=keep[0].device)
    off = (-ws.data_ptr()) % 256
    cap = max(1, min(int(cat.n), int(n_ra) * int(n_u)))
    pra = torch.empty(cap, dtype=torch.float64, device=keep[0].device)
    pdec = torch.empty(cap, dtype=torch.float64, device=keep[0].device)
    pw = torch.empty(cap, dtype=torch.int32, device=keep[0].device)
    m = C.c_int64(0)
    _check(lib.cute_pixelize(C.byref(cat), float(ra0), float(dra), float(u0), float(du), int(n_ra), int(n_u),
                             C.c_void_p(pra.data_ptr()), C.c_void_p(pdec.data_ptr()), C.c_void_p(pw.data_ptr()), C.byref(m),
                             C.c_void_p(ws.data_ptr() + off), ws.numel() - off, C.c_void_p(_stream_ptr(stream))), "cute_pixelize")
    k = int(m.value)
    return pra[:k].contiguous(), pdec[:k].contiguous(), pw[:k].contiguous()


def cute_grid_workspace_bytes(cat: cute_catalog, spec: cute_grid_spec) -> int:
    b = C.c_size_t(0)
    _check(lib.cute_grid_workspace_bytes(C.byref(cat), C.byref(spec), C.byref(b)), "cute_grid_workspace_bytes")
    return int(b.value)


def cute_make_grid(cols, coord: int, spec: cute_grid_spec, stream=None, workspace=None, weight=None) -> Grid:
    """cols: torch CUDA tensors (SoA); weight: optional int32/uint32 CUDA tensor.  Runs G0-G4 on the device."""
    torch = _torch()
    cat, keep = _catalog(cols, coord, True, weight)
    nbytes = cute_grid_workspace_bytes(cat, spec)
    if workspace is None:
        workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=keep[0].device)
    base = workspace.data_ptr()
    off = (-base) % 256
    h = C.c_void_p()
    _check(lib.cute_make_grid(C.byref(cat), C.byref(spec), C.c_void_p(base + off), workspace.numel() - off,
                              C.c_void_p(_stream_ptr(stream)), C.byref(h)), "cute_make_grid")
    return Grid(h, workspace, spec)


# ------------------------------------------------------------------------------- pair counts
class Counter:
    """Scratch + output histogram for cute_count_pairs (reusable across calls with the same bins)."""

    def __init__(self, bins: dict, device="cuda"):
        torch = _torch()
        self.bins = bin_spec(bins)
        b = C.c_size_t(0)
        _check(lib.cute_count_scratch_bytes(C.byref(self.bins), None, C.byref(b)), "cute_count_scratch_bytes")
        self.scratch = torch.empty(b.value + 256, dtype=torch.uint8, device=device)
        self.soff = (-self.scratch.data_ptr()) % 256
        self.nhist = self.bins.n1 * max(self.bins.n2, 1)
        self.hist = torch.zeros(self.nhist, dtype=torch.int64, device=device)

    def scratch_ptr(self):
        return C.c_void_p(self.scratch.data_ptr() + self.soff)


def cute_count_pairs(kind: int, g1: Grid, g2: Grid | None, counter: Counter, opts: cute_count_opts | None = None, stream=None):
    """Enqueue the pair count; the result lands in counter.hist (device int64 == uint64 bits)."""
    _check(lib.cute_count_pairs(int(kind), g1.handle, g2.handle if g2 is not None else None, C.byref(counter.bins),
                                C.c_void_p(counter.hist.data_ptr()), counter.scratch_ptr(),
                                counter.scratch.numel() - counter.soff, C.byref(opts) if opts is not None else None,
                                C.c_void_p(_stream_ptr(stream))), "cute_count_pairs")
    return counter.hist


def cute_count_items(kind: int, g1: Grid, g2: Grid | None, counter: Counter, opts=None) -> int:
    n = C.c_int64(0)
    _check(lib.cute_count_items(int(kind), g1.handle, g2.handle if g2 is not None else None, C.byref(counter.bins),
                                C.byref(opts) if opts is not None else None, C.byref(n)), "cute_count_items")
    return int(n.value)


def cute_count_status(counter: Counter, stream=None) -> dict:
    st = (C.c_uint64 * 4)()
    _check(lib.cute_count_status(counter.scratch_ptr(), C.c_void_p(_stream_ptr(stream)), st), "cute_count_status")
    return dict(evaluated=int(st[0]), refined=int(st[1]), items=int(st[2]), flushes=int(st[3]))


def cute_count_pairs_static(kind: int, g1: Grid, g2: Grid | None, bins: dict, hist, opts: cute_count_opts | None = None, stream=None) -> dict:
    """The pair count for callers that cannot allocate device memory (a hook inside a simulation that owns the whole
    device, a plug-in under a fixed memory budget, a thread that must not call cudaMalloc): same count as
    cute_count_pairs, but its scratch is a fixed STATIC_SCRATCH_BYTES array inside the library instead of a buffer of
    the caller's.  `hist`: the caller's device tensor of n1 * max(n2, 1) int64 (uint64 bits), overwritten.  Waits for
    the stream; returns the kernel's statistics.  Raises CuteError(ERR_STATIC_SCRATCH_LIMIT) when n1 + n2 > 8182.  All
    calls on a device share the one array, so the library runs them one at a time; the first call on a device should
    not be made during a stream capture."""
    b = bin_spec(bins)
    assert hist.is_cuda and hist.is_contiguous() and hist.element_size() == 8 and hist.numel() == b.n1 * max(b.n2, 1)
    st = (C.c_uint64 * 4)()
    _check(lib.cute_count_pairs_static(int(kind), g1.handle, g2.handle if g2 is not None else None, C.byref(b),
                                       C.c_void_p(hist.data_ptr()), C.byref(opts) if opts is not None else None,
                                       C.c_void_p(_stream_ptr(stream)), st), "cute_count_pairs_static")
    return dict(evaluated=int(st[0]), refined=int(st[1]), items=int(st[2]), flushes=int(st[3]))


def cute_count_pairs_host(kind: int, cat1, cat2, coord: int, spec: cute_grid_spec, bins: dict, workspace=None, stream=None,
                          opts: cute_count_opts | None = None, w1=None, w2=None):
    """End to end with HOST (numpy) buffers: H2D copies, grid build, count, D2H of the histogram."""
    torch = _torch()
    c1, k1 = _catalog([np.ascontiguousarray(c) for c in cat1], coord, False, None if w1 is None else np.ascontiguousarray(w1, dtype=np.uint32))
    c2 = k2 = None
    if cat2 is not None:
        c2, k2 = _catalog([np.ascontiguousarray(c) for c in cat2], coord, False, None if w2 is None else np.ascontiguousarray(w2, dtype=np.uint32))
    b = bin_spec(bins)
    nb = C.c_size_t(0)
    _check(lib.cute_host_workspace_bytes(C.byref(c1), C.byref(c2) if c2 is not None else None, C.byref(spec), C.byref(b),
                                         C.byref(nb)), "cute_host_workspace_bytes")
    if workspace is None or workspace.numel() < nb.value + 256:
        workspace = torch.empty(nb.value + 256, dtype=torch.uint8, device="cuda")
    off = (-workspace.data_ptr()) % 256
    hist = np.zeros(b.n1 * max(b.n2, 1), dtype=np.uint64)
    _check(lib.cute_count_pairs_host(int(kind), C.byref(c1), C.byref(c2) if c2 is not None else None, C.byref(spec), C.byref(b),
                                     C.byref(opts) if opts is not None else None, hist.ctypes.data_as(C.POINTER(C.c_uint64)), C.c_void_p(workspace.data_ptr() + off),
                                     workspace.numel() - off, C.c_void_p(_stream_ptr(stream))), "cute_count_pairs_host")
    return hist, workspace


# ------------------------------------------------------------------------------- host helpers
def _up(a):
    return a.ctypes.data_as(C.POINTER(C.c_uint64))


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


def cute_bin_edges(bins: dict, axis: int = 0) -> np.ndarray:
    b = bin_spec(bins)
    e = np.zeros((b.n1 if axis == 0 else b.n2) + 1)
    _check(lib.cute_bin_edges(C.byref(b), axis, _dp(e)), "cute_bin_edges")
    return e


def cute_landy_szalay(dd, dr, rr, nd: int, nr: int):
    dd, dr, rr = (np.ascontiguousarray(np.asarray(a).astype(np.uint64)).ravel() for a in (dd, dr, rr))
    xi = np.zeros(dd.size)
    rc = _check(lib.cute_landy_szalay(_up(dd), _up(dr), _up(rr), int(nd), int(nr), dd.size, _dp(xi)), "cute_landy_szalay")
    return xi, rc


def cute_natural_estimator(dd, rr, nd: int, nr: int):
    dd, rr = (np.ascontiguousarray(np.asarray(a).astype(np.uint64)).ravel() for a in (dd, rr))
    xi = np.zeros(dd.size)
    rc = _check(lib.cute_natural_estimator(_up(dd), _up(rr), int(nd), int(nr), dd.size, _dp(xi)), "cute_natural_estimator")
    return xi, rc


def cute_multipoles(xi_rmu, n_r: int, n_mu: int) -> np.ndarray:
    """xi_0, xi_2, xi_4 (shape (3, n_r)) of xi(r, mu) given as [n_r][n_mu] over mu in [0,1] (Eqs. 3-4)."""
    xi = np.ascontiguousarray(np.asarray(xi_rmu, dtype=np.float64)).ravel()
    out = np.zeros((3, n_r))
    _check(lib.cute_multipoles(_dp(xi), int(n_r), int(n_mu), _dp(out)), "cute_multipoles")
    return out


def cute_periodic_rr(n: int, L: float, bins: dict) -> np.ndarray:
    b = bin_spec(bins)
    rr = np.zeros(b.n1)
    _check(lib.cute_periodic_rr(int(n), float(L), C.byref(b), _dp(rr)), "cute_periodic_rr")
    return rr


def cute_periodic_xi(dd, n: int, L: float, bins: dict):
    b = bin_spec(bins)
    dd = np.ascontiguousarray(np.asarray(dd).astype(np.uint64)).ravel()
    xi = np.zeros(b.n1)
    rc = _check(lib.cute_periodic_xi(_up(dd), int(n), float(L), C.byref(b), _dp(xi)), "cute_periodic_xi")
    return xi, rc


def cute_density_grid_xi(cols, L: float, ng: int, bins: dict, want_delta: bool = False, workspace=None, stream=None):
    """Density-grid monopole (Eq. 17) of device xyz columns: dict(xi, sum_dd, npairs, status[, delta])."""
    torch = _torch()
    cat, keep = _catalog(cols, COORD_XYZ, True)
    b = bin_spec(bins)
    nb = C.c_size_t(0)
    _check(lib.cute_density_grid_workspace_bytes(int(ng), C.byref(b), float(L), C.byref(nb)), "cute_density_grid_workspace_bytes")
    if workspace is None or workspace.numel() < nb.value + 256:
        workspace = torch.empty(nb.value + 256, dtype=torch.uint8, device=keep[0].device)
    off = (-workspace.data_ptr()) % 256
    xi, sdd, npr = np.zeros(b.n1), np.zeros(b.n1), np.zeros(b.n1, dtype=np.uint64)
    delta = torch.empty(ng * ng * ng, dtype=torch.float64, device=keep[0].device) if want_delta else None
    rc = _check(lib.cute_density_grid_xi(C.byref(cat), float(L), int(ng), C.byref(b), _dp(xi), _dp(sdd), _up(npr),
                                         C.c_void_p(delta.data_ptr()) if delta is not None else None,
                                         C.c_void_p(workspace.data_ptr() + off), workspace.numel() - off, C.c_void_p(_stream_ptr(stream))),
                "cute_density_grid_xi")
    out = dict(xi=xi, sum_dd=sdd, npairs=npr, status=rc, workspace=workspace)
    if delta is not None:
        out["delta"] = delta.view(ng, ng, ng)
    return out


def cute_measure_peaks(stream=None) -> dict:
    """{name: (lane-operations per clock per SM, warp-instructions per clock per SM)} measured on the current device."""
    torch = _torch()
    n = int(lib.cute_peak_count())
    ops, ins = np.zeros(n), np.zeros(n)
    tmp = torch.empty((1 << 20) + 256, dtype=torch.uint8, device="cuda")
    off = (-tmp.data_ptr()) % 256
    _check(lib.cute_measure_peaks(_dp(ops), _dp(ins), n, C.c_void_p(tmp.data_ptr() + off), tmp.numel() - off,
                                  C.c_void_p(_stream_ptr(stream))), "cute_measure_peaks")
    return {lib.cute_peak_name(k).decode(): (float(ops[k]), float(ins[k])) for k in range(n)}


# ------------------------------------------------------------------------------- workload convenience
COORD_OF_KIND = {"monopole": COORD_XYZ, "rmu": COORD_XYZ, "pisigma": COORD_XYZ, "angular": COORD_RADEC, "radial": COORD_RADECZ}


def cute_shard_items(nitems: int, nchunks: int, rank: int, world: int, auto_brute: bool):
    """[begin, end) of the work-item list for this rank (the library's sharding policy; needs no GPU)."""
    b, e = C.c_int64(0), C.c_int64(0)
    _check(lib.cute_shard_items(int(nitems), int(nchunks), int(rank), int(world), int(bool(auto_brute)), C.byref(b), C.byref(e)),
           "cute_shard_items")
    return int(b.value), int(e.value)


def auto_spec(kind: str, bins: dict, grid: dict, cats_dev, coord: int) -> cute_grid_spec:
    """Grid spec for a workload (cute_auto_grid_spec): `grid` is synth.Workload.grid (mode + rmax/thetamax [+ ncell, pix]);
    cats_dev: the device catalogues that will share the spec.  Marshalling only: the geometry is the library's."""
    torch = _torch()
    mode = {"none": GRID_NONE, "box3d": GRID_BOX3D, "sphere": GRID_SPHERE}[grid.get("mode", "none")]
    cats, keep = [], []
    for c in cats_dev:
        cat, k = _catalog(c, coord, True)
        cats.append(cat)
        keep.append(k)
    arr = (C.POINTER(cute_catalog) * len(cats))(*[C.pointer(c) for c in cats])
    rmax = float(grid.get("rmax", grid.get("thetamax", 0.0)))
    ncell = (C.c_int * 3)(*map(int, grid.get("ncell", (0, 0, 0))))
    tmp = torch.empty(16, dtype=torch.float64, device="cuda")
    spec = cute_grid_spec()
    _check(lib.cute_auto_grid_spec(KINDS[kind], mode, arr, len(cats), rmax, float(bins.get("box_L", 0.0)) if mode == GRID_BOX3D else 0.0,
                                   float(grid.get("pix", 2.0)), ncell, int(grid.get("no_perm", 0)), C.c_void_p(tmp.data_ptr()),
                                   C.c_void_p(_stream_ptr()), C.byref(spec)), "cute_auto_grid_spec")
    spec.build_path = int(grid.get("build_path", 0))
    return spec
