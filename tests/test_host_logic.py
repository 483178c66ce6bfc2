"""CPU-side tests (no GPU): the C-ABI library loads and exports every symbol include/cute_b200.h declares,
the host-side helpers agree with the oracle, argument validation, and the multi-GPU sharding logic
(world_size-2 gloo)."""
import ctypes as C
import os
import re
import subprocess
import sys

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def api():
    from paper_1210_1833_b200 import build
    build.build()
    from paper_1210_1833_b200 import api as a
    return a


def test_library_exports_every_declared_symbol(api):
    hdr = open(os.path.join(ROOT, "include", "cute_b200.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(cute_[a-z_0-9]+)\s*\(", hdr))
    assert len(declared) >= 18
    lib = C.CDLL(api.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), f"{name} declared in the header but not exported"
    assert declared == set(api.SYMBOLS)
    assert api.cute_version() == 1
    assert "invalid" in api.cute_strerror(-1)


def test_struct_sizes_match_header(api, tmp_path):
    """the ctypes mirrors have the sizes the C compiler gives the header's structs"""
    src = tmp_path / "sz.c"
    src.write_text('#include <stdio.h>\n#include "cute_b200.h"\nint main(){printf("%zu %zu %zu %zu %zu\\n",sizeof(cute_catalog),'
                   'sizeof(cute_grid_spec),sizeof(cute_bin_spec),sizeof(cute_count_opts),sizeof(cute_grid_info));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.check_call(["gcc", "-I", os.path.join(ROOT, "include"), str(src), "-o", str(exe)])
    sizes = [int(x) for x in subprocess.check_output([str(exe)]).split()]
    assert sizes == [C.sizeof(api.cute_catalog), C.sizeof(api.cute_grid_spec), C.sizeof(api.cute_bin_spec),
                     C.sizeof(api.cute_count_opts), C.sizeof(api.cute_grid_info)]


@pytest.mark.parametrize("bins", [dict(n1=50, lo1=0.0, hi1=150.0), dict(n1=64, lo1=1.7e-5, hi1=0.1745, log1=1),
                                  dict(n1=40, lo1=0.0, hi1=200.0, n2=50, lo2=0.0, hi2=1.0)])
def test_bin_edges_equal_oracle(api, oracle, bins):
    """S1: one definition of the edges on both sides (bitwise)"""
    assert np.array_equal(api.cute_bin_edges(bins, 0), oracle.edges(bins, 0))
    if bins.get("n2", 0):
        assert np.array_equal(api.cute_bin_edges(bins, 1), oracle.edges(bins, 1))


def test_estimators_equal_oracle(api, oracle):
    """Eq. 15 / Eq. 14 / Eq. 13 on identical histograms: within 1e-6 absolute (north star), in fact 1e-12"""
    rng = np.random.default_rng(3)
    rr = rng.integers(0, 10**9, 40).astype(np.uint64)
    rr[5] = 0
    dd = rng.integers(0, 10**8, 40).astype(np.uint64)
    dr = rng.integers(0, 10**9, 40).astype(np.uint64)
    xi, rc = api.cute_landy_szalay(dd, dr, rr, 200000, 400000)
    xo, empty = oracle.landy_szalay(dd, dr, rr, 200000, 400000)
    assert np.max(np.abs(xi - xo)) <= 1e-12 * np.max(np.abs(xo)) and rc == api.WARN_EMPTY_BIN and empty == 1 and xi[5] == 0.0
    xn, _ = api.cute_natural_estimator(dd, rr, 200000, 400000)
    xno, _ = oracle.natural(dd, rr, 200000, 400000)
    assert np.allclose(xn, xno, rtol=1e-13, atol=0)
    b = dict(n1=50, lo1=0.0, hi1=150.0, box_L=1000.0)
    assert np.allclose(api.cute_periodic_rr(20000, 1000.0, b), oracle.periodic_rr(20000, 1000.0, b), rtol=1e-14)
    # closed form, bin 0 and last bin of C1 (RR_0 = 22.6, RR_49 = 1.66e5)
    rr1 = api.cute_periodic_rr(20000, 1000.0, b)
    assert abs(rr1[0] - 22.6) < 0.05 and abs(rr1[49] / 1.66e5 - 1) < 0.01
    xp, _ = api.cute_periodic_xi(np.round(rr1).astype(np.uint64), 20000, 1000.0, b)
    assert np.max(np.abs(xp)) < 0.03


def test_multipoles_equal_oracle(api, oracle):
    """Eqs. 3-4 on the host: library == oracle, and a pure quadrupole comes back"""
    rng = np.random.default_rng(8)
    xi = rng.normal(size=(40, 50))
    assert np.allclose(api.cute_multipoles(xi, 40, 50), oracle.multipoles(xi, 40, 50), rtol=1e-12, atol=1e-14)
    mu = (np.arange(50) + 0.5) / 50
    m = api.cute_multipoles(np.tile(0.5 * (3 * mu**2 - 1), (3, 1)), 3, 50)
    assert np.allclose(m[0], 0, atol=1e-3) and np.allclose(m[1], 1, atol=5e-3)


def test_validation_without_gpu(api):
    """host-side argument checks return error codes (no exceptions, no abort) before anything touches the device"""
    lib = api.lib
    b = api.bin_spec(dict(n1=0, lo1=0.0, hi1=1.0))
    n = C.c_size_t(0)
    assert lib.cute_count_scratch_bytes(C.byref(b), None, C.byref(n)) == -1
    e = (C.c_double * 4)()
    assert lib.cute_bin_edges(C.byref(api.bin_spec(dict(n1=3, lo1=0.0, hi1=1.0, log1=1))), 0, e) == -1   # log needs lo > 0
    assert lib.cute_bin_edges(C.byref(api.bin_spec(dict(n1=3, lo1=2.0, hi1=1.0))), 0, e) == -1
    cat = api.cute_catalog(C.sizeof(api.cute_catalog), 10, api.COORD_XYZ, api.F32, 256, 512, 768)
    bad = api.grid_spec("sphere", rmax=0.1)          # sphere grid on XYZ coordinates
    assert lib.cute_grid_workspace_bytes(C.byref(cat), C.byref(bad), C.byref(n)) == -1
    ok = api.grid_spec("box3d", periodic=True, size=(100, 100, 100), rmax=10.0)
    assert lib.cute_grid_workspace_bytes(C.byref(cat), C.byref(ok), C.byref(n)) == 0 and n.value > 0
    cat.struct_size = 3
    assert lib.cute_grid_workspace_bytes(C.byref(cat), C.byref(ok), C.byref(n)) == -1
    assert lib.cute_landy_szalay(None, None, None, 10, 10, 4, None) == -1


def test_product_path_does_not_touch_the_oracle():
    """the package never imports, includes, links or opens anything under oracle/, and the oracle never imports the
    package; the only shared module is synth.py, which holds no arithmetic of the method"""
    pkg = os.path.join(ROOT, "paper_1210_1833_b200")
    bad = re.compile(r"(^\s*import\s+oracle|^\s*from\s+oracle|#include.*oracle|cute_oracle|libcute_oracle|\borc_[a-z])")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".h")):
                for line in open(os.path.join(dirpath, f)):
                    assert not bad.search(line), (f, line)
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1210_1833_b200" not in txt and "cute_b200.h" not in txt and "libcute_b200" not in txt


# ------------------------------------------------------------------------------- sharding
def test_shard_bounds_partition(api):
    shard_bounds = lambda nitems, r, world, nchunks, auto: api.cute_shard_items(nitems, nchunks, r, world, auto)
    for nchunks, nsplit, world, auto in [(1563, 19, 2, True), (1563, 19, 8, True), (3125, 10, 4, False), (7, 1, 8, False),
                                         (78326, 1, 8, False), (1, 5, 4, True)]:
        nitems = nchunks * nsplit
        cuts = [shard_bounds(nitems, r, world, nchunks, auto) for r in range(world)]
        assert cuts[0][0] == 0 and cuts[-1][1] == nitems
        for (b0, e0), (b1, e1) in zip(cuts, cuts[1:]):
            assert e0 == b1 and b0 <= e0
        if auto and nchunks > 100:
            # equal triangle areas: work of chunk c ~ (nchunks - c)
            work = [sum(nchunks - c for c in range(b // nsplit, e // nsplit)) for b, e in cuts]
            assert max(work) / (sum(work) / world) < 1.05
    assert shard_bounds(100, 0, 1, 10, True) == (0, 100)


_WORKER = r"""
import os, sys
import numpy as np, torch, torch.distributed as dist
sys.path.insert(0, sys.argv[1])
from paper_1210_1833_b200 import api
shard_bounds = lambda nitems, r, world, nchunks, auto: api.cute_shard_items(nitems, nchunks, r, world, auto)
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
r, w = dist.get_rank(), dist.get_world_size()
# a fake pair count: item k contributes 1 to bin k % 7 and k to bin 7; shards must add up to the whole
nchunks, nsplit = 157, 13
n = nchunks * nsplit
b, e = shard_bounds(n, r, w, nchunks, True)
h = torch.zeros(8, dtype=torch.int64)
for k in range(b, e):
    h[k % 7] += 1
    h[7] += k
dist.all_reduce(h)
full = torch.zeros(8, dtype=torch.int64)
for k in range(n):
    full[k % 7] += 1
    full[7] += k
assert torch.equal(h, full), (h, full)
t = torch.tensor([float(r + 1)], dtype=torch.float64)
dist.all_reduce(t, op=dist.ReduceOp.MAX)
assert t.item() == w
dist.destroy_process_group()
print("ok", r)
"""


def test_two_rank_gloo_histogram_allreduce(tmp_path):
    """N>1 path on CPU: shard the item list over 2 ranks, all-reduce the partial int64 histograms (gloo)"""
    script = tmp_path / "worker.py"
    script.write_text(_WORKER)
    env = dict(os.environ, MASTER_ADDR="127.0.0.1", MASTER_PORT="29571", WORLD_SIZE="2")
    procs = [subprocess.Popen([sys.executable, str(script), ROOT], env=dict(env, RANK=str(r)), stdout=subprocess.PIPE,
                              stderr=subprocess.STDOUT) for r in range(2)]
    outs = [p.communicate(timeout=240)[0].decode() for p in procs]
    for p, o in zip(procs, outs):
        assert p.returncode == 0, o


def test_grid_workspace_reserves_the_partition_only_where_it_can_run(api):
    """the partition build's record buffer (16-32 bytes per point) and its bucket table are part of the workspace only when
    some cell count the build may choose can take that path; and the table always has room for the largest bucket
    count (kPartMaxBuckets = 1024 buckets x 2 SM-count CTAs x 2 tables)"""
    n = 1 << 21
    z = np.zeros(8, dtype=np.float32)

    def nbytes(dtype, mode, build_path, ncell=(0, 0, 0)):
        cat = api.cute_catalog(C.sizeof(api.cute_catalog), n, api.COORD_XYZ, dtype, z.ctypes.data, z.ctypes.data, z.ctypes.data, None)
        spec = api.grid_spec(mode, size=(1000.0,) * 3 if mode == "box3d" else (0, 0, 0), ncell=ncell,
                             rmax=50.0 if mode == "box3d" else 0.0, kind_mask=2, build_path=build_path)
        return api.cute_grid_workspace_bytes(cat, spec)

    # brute force, float32 xyz: at most 32^3 ordering cells, never partitioned unless forced
    assert nbytes(api.F32, "none", 2) - nbytes(api.F32, "none", 0) >= 16 * n
    assert nbytes(api.F32, "none", 0) == nbytes(api.F32, "none", 1)
    # float64 brute force may take it (32-byte records)
    assert nbytes(api.F64, "none", 0) - nbytes(api.F64, "none", 1) >= 32 * n
    # cell list, float32: explicit small ncell never partitions, automatic cells may
    assert nbytes(api.F32, "box3d", 0, (20, 20, 20)) == nbytes(api.F32, "box3d", 1, (20, 20, 20))
    assert nbytes(api.F32, "box3d", 0, (50, 50, 50)) - nbytes(api.F32, "box3d", 1, (50, 50, 50)) >= 16 * n + 2 * 1024 * 4
    assert nbytes(api.F32, "box3d", 0) - nbytes(api.F32, "box3d", 1) >= 16 * n + 2 * 1024 * 4


def test_static_scratch_entry_point_refuses_fine_binning_without_a_gpu(api):
    """cute_count_pairs_static checks its size limit before it touches CUDA: more bins than the built-in 64 KiB scratch
    holds (n1 + n2 > 8182) is CUTE_ERR_STATIC_SCRATCH_LIMIT whatever the other arguments are; the same spec with
    caller-provided scratch is a plain size query"""
    for n1, n2, want in ((8183, 0, api.ERR_STATIC_SCRATCH_LIMIT), (4000, 4183, api.ERR_STATIC_SCRATCH_LIMIT), (70000, 0, -1)):
        b = api.bin_spec(dict(n1=n1, lo1=0.0, hi1=100.0, n2=n2, lo2=0.0, hi2=1.0))
        rc = api.lib.cute_count_pairs_static(api.MONOPOLE if n2 == 0 else api.RMU, None, None, C.byref(b), None, None, None, None)
        if want == -1:
            assert rc < 0        # (n1 beyond what any count accepts: refused one way or the other)
        else:
            assert rc == want
    b = api.bin_spec(dict(n1=8183, lo1=0.0, hi1=100.0))
    nb = C.c_size_t(0)
    assert api.lib.cute_count_scratch_bytes(C.byref(b), None, C.byref(nb)) == 0 and nb.value > api.STATIC_SCRATCH_BYTES
    b = api.bin_spec(dict(n1=8182, lo1=0.0, hi1=100.0))
    assert api.lib.cute_count_scratch_bytes(C.byref(b), None, C.byref(nb)) == 0 and nb.value == api.STATIC_SCRATCH_BYTES
    assert "cute_count_pairs" in api.cute_strerror(api.ERR_STATIC_SCRATCH_LIMIT)
