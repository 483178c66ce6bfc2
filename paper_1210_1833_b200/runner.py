"""Driving the C ABI for a whole workload (used by bench.py, smoke() and the GPU tests).

Only plumbing lives here: host->device copies with torch, building the grids, enqueuing the pair
counts of DD / DR / RR and reading the histograms back.  All arithmetic is in libcute_b200.so.
"""
from __future__ import annotations

import numpy as np

from . import api


def to_device(cat, coord: int, dtype=None):
    """numpy SoA columns -> contiguous torch CUDA tensors (one dtype)."""
    import torch
    need = 2 if coord == api.COORD_RADEC else 3
    cols = []
    for c in list(cat)[:need]:
        a = np.ascontiguousarray(c)
        if dtype is not None:
            a = a.astype(dtype, copy=False)
        elif a.dtype not in (np.float32, np.float64):
            a = a.astype(np.float64)
        cols.append(torch.from_numpy(a).cuda())
    return cols


class Job:
    """One correlation-function job: catalogues resident on the device, grids built, counters ready."""

    def __init__(self, kind: str, data, rand, bins: dict, grid: dict | None = None, opts: dict | None = None,
                 w_data=None, w_rand=None):
        self.kind_name = kind
        self.kind = api.KINDS[kind]
        self.coord = api.COORD_OF_KIND[kind]
        self.bins = dict(bins)
        self.grid = dict(grid or {"mode": "none"})
        self.opts = api.count_opts(**opts) if opts else None
        self.d_data = to_device(data, self.coord)
        self.d_rand = to_device(rand, self.coord) if rand is not None else None
        import torch
        as_w = lambda w: None if w is None else torch.from_numpy(np.ascontiguousarray(w, dtype=np.uint32).view(np.int32)).cuda()
        self.w_data, self.w_rand = as_w(w_data), as_w(w_rand)      # integer weights (pixel maps), uint32 bits
        self.nd = int(self.d_data[0].numel())
        self.nr = int(self.d_rand[0].numel()) if self.d_rand is not None else 0
        self.counter = api.Counter(self.bins)
        self.g_data = self.g_rand = None
        self.spec = None

    def build(self, share=None):
        """G0-G4 for every catalogue (cute_make_grid).

        share: N > 1 only -- a callable that overwrites a device uint8 tensor on every rank with rank 0's copy (a broadcast).
        The order of the points INSIDE a cell is decided by atomic cursors and differs from build to build, so the work
        items (128 consecutive sorted points) of two ranks that each built their own grid do not hold the same points and
        their item shards would not partition the pairs.  Every rank therefore builds (same layout, same host-side handle:
        cell counts, chunk counts and bounds do not depend on that order) and then takes rank 0's workspace bytes."""
        cats = [self.d_data] + ([self.d_rand] if self.d_rand is not None else [])
        if self.spec is None:
            self.spec = api.auto_spec(self.kind_name, self.bins, self.grid, cats, self.coord)
        if self.g_data is not None:
            self.g_data.free()
        self.g_data = api.cute_make_grid(self.d_data, self.coord, self.spec, workspace=getattr(self, "_ws_d", None), weight=self.w_data)
        self._ws_d = self.g_data.workspace
        if self.d_rand is not None and self.spec.mode == api.GRID_BOX3D:
            # the two grids of a cross-correlation must carry one spec: hand the second build the cell counts
            # (and box) the library resolved for the first
            inf = self.g_data.info()
            self.spec = api.grid_spec("box3d", periodic=bool(self.spec.periodic), origin=tuple(inf.origin),
                                      size=tuple(inf.size), ncell=tuple(inf.ncell),
                                      rmax=self.spec.rmax, kind_mask=self.spec.kind_mask, no_perm=self.spec.no_perm,
                                      build_path=self.spec.build_path)
        if self.d_rand is not None:
            if self.g_rand is not None:
                self.g_rand.free()
            self.g_rand = api.cute_make_grid(self.d_rand, self.coord, self.spec, workspace=getattr(self, "_ws_r", None), weight=self.w_rand)
            self._ws_r = self.g_rand.workspace
        if share is not None:
            for g in (self.g_data, self.g_rand):
                if g is not None:
                    off = (-g.workspace.data_ptr()) % 256
                    share(g.workspace[off:])
        return self

    def grids(self, which: str):
        return {"DD": (self.g_data, None), "DR": (self.g_data, self.g_rand), "RR": (self.g_rand, None)}[which]

    def enqueue(self, which: str):
        g1, g2 = self.grids(which)
        return api.cute_count_pairs(self.kind, g1, g2, self.counter, self.opts)

    def count(self, which: str = "DD"):
        """Histogram (numpy uint64) and the kernel's statistics for one of DD / DR / RR."""
        h = self.enqueue(which)
        st = api.cute_count_status(self.counter)
        return h.cpu().numpy().astype(np.uint64), st

    def total_pairs(self, which: str) -> int:
        if which == "DD":
            return self.nd * (self.nd - 1) // 2
        if which == "RR":
            return self.nr * (self.nr - 1) // 2
        return self.nd * self.nr


def job_for_workload(w, opts: dict | None = None) -> Job:
    return Job(w.kind, w.data, w.rand, w.bins, w.grid, opts)
