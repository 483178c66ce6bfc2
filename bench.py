#!/usr/bin/env python
"""bench.py -- headline benchmark of the CUTE pair-counting hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: the cell-list
build (G0-G4, cute_make_grid) of the data and random catalogues, the DD, DR and RR pair counts
(P1-P5, cute_count_pairs) and the Landy-Szalay estimator on the host (H1).  The default workload
is BASELINE.json configs[1] ("C2": angular w(theta), 200k data x 400k randoms, 64 log bins,
brute force, 1.8e11 pairs per step).  One JSON line is printed by rank 0.

N > 1 (torchrun): the work-item list of every pair count is split over the ranks (catalogues and
grids replicated), and the partial uint64 histograms are summed with one NCCL all-reduce -- the
only exchange step the method has.  Total work is fixed: "scaling": "strong".

--impl reference times the float64 oracle (oracle/) on the host cores, as it stands, on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "pairs/sec (1e9) counted into bins on 1 B200; % of pair-kernel roofline"
UNIT = "1e9 pairs/s"
SM_COUNT, LANES_PER_SM, SM_MAX_MHZ = 148, 128, 1965.0
# dram__bytes_read.sum + dram__bytes_write.sum per pair-kernel launch from the committed `ncu --set full` capture
# (profiles/r01_pair_kernel_c2.md: 11.3 MB DD, 33.8 MB DR; RR as DR), averaged over the 3 launches of a C2 step
NCU_TRAFFIC_BYTES = {2: (11.29e6 + 33.82e6 + 33.82e6) / 3.0}


# ------------------------------------------------------------------------------- sharding (host logic)
def shard_bounds(nitems: int, rank: int, world: int, nchunks: int, is_auto_brute: bool):
    """[begin, end) of the work-item list for this rank.  Items are chunk-major (item = chunk*nsplit
    + split).  Cross-correlations and grid-assisted counts have ~uniform work per item; a brute-force
    auto-correlation is a triangle (chunk c meets only j > i), so its boundaries are placed at equal
    areas: the fraction of work before chunk fraction x is 1-(1-x)^2."""
    if world <= 1:
        return 0, nitems
    nsplit = max(1, nitems // max(nchunks, 1))

    def cut(r):
        f = r / world
        x = 1.0 - math.sqrt(max(0.0, 1.0 - f)) if is_auto_brute else f
        c = int(round(x * nchunks))
        return min(nitems, max(0, c * nsplit))
    b, e = cut(rank), cut(rank + 1)
    if rank == world - 1:
        e = nitems
    return b, e


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples SM clock and throttle reasons with NVML every 100 ms while running."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz = [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _run(self):
        nv = self.nv
        names = {"hw_slowdown": 0x8, "sw_thermal_slowdown": 0x20, "hw_thermal_slowdown": 0x40,
                 "hw_power_brake_slowdown": 0x80, "sw_power_cap": 0x4}
        while not self._stop.is_set():
            try:
                self.samples.append(float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)) if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons") \
                    else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if r & bit:
                        self.reasons.add(k)
            except Exception:
                pass
            self._stop.wait(0.1)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()
        med = float(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------- the oracle legs
def oracle_sample(w, seconds: float = 15.0):
    """Time the oracle, as it stands, on a bounded sample of the workload's DR count (all host cores).
    Returns (pairs per second, cores, description)."""
    from oracle import oracle as o
    o.build()
    cores = o.max_threads()
    c2 = w.rand if w.rand is not None else None
    mode = "plain" if w.grid.get("mode", "none") == "none" else "celled"
    n1 = len(w.data[0])
    m = min(n1, 256)
    t0 = time.perf_counter()
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, m))
    dt = time.perf_counter() - t0
    rate = r["npairs"] / max(dt, 1e-9)
    per_row = r["npairs"] / m
    m2 = int(min(n1, max(m, seconds * rate / max(per_row, 1.0))))
    t0 = time.perf_counter()
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, m2))
    dt = time.perf_counter() - t0
    what = "DR" if c2 is not None else "DD"
    return r["npairs"] / dt, cores, f"{what} rows [0,{m2}) of {n1} x all of catalogue 2, mode {mode}: {r['npairs']} separations in {dt:.2f} s"


def run_reference(args, w, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import oracle as o
    o.build()
    cores = o.max_threads()
    c2 = w.rand if w.rand is not None else None
    mode = "plain" if w.grid.get("mode", "none") == "none" else "celled"
    n1 = len(w.data[0])
    # bounded sample per step: ~3 s of CPU work
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, min(n1, 128)))
    t0 = time.perf_counter()
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, min(n1, 128)))
    rate = r["npairs"] / max(time.perf_counter() - t0, 1e-9)
    rows = int(min(n1, max(128, 3.0 * rate / (r["npairs"] / min(n1, 128)))))
    for _ in range(args.warmup):
        o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, rows))
    pairs, t0 = 0, time.perf_counter()
    for _ in range(args.steps):
        pairs += o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, rows))["npairs"]
    dt = time.perf_counter() - t0
    v = pairs / dt / 1e9
    sample = f"each step: rows [0,{rows}) of {n1} x catalogue 2 ({'DR' if c2 is not None else 'DD'}), oracle mode {mode}"
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "strong",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ------------------------------------------------------------------------------- our arm
# Algorithmic FP32-lane instructions per pair: (every evaluated pair, extra per binned pair)
ALG_INSTR = {
    ("angular", "none"): (13.0, 15.0),    # 9 FADD + FMUL + 2 FFMA + range test | LG2 + 3 poly + 2 + 2 FFMA + 2 floor + cmp + range + addr + atomic
    ("angular", "sphere"): (13.0, 15.0),
    ("monopole", "none"): (16.0, 9.0),    # periodic brute: + 9 for the minimum image | SQRT + 2 FFMA + 2 floor + cmp + range + addr + atomic
    ("monopole", "box3d"): (7.0, 9.0),    # 3 FADD + FMUL + 2 FFMA + range test
    ("rmu", "box3d"): (7.0, 21.0),        # + 3 FADD (s.l) + 2 (|l|^2) + FMUL + RSQ + FMUL + 2 FFMA + 2 FADD + 2 floor + cmp + range + IMAD
    ("rmu", "none"): (7.0, 21.0),
    ("pisigma", "box3d"): (7.0, 24.0),
    ("pisigma", "none"): (7.0, 24.0),
    ("radial", "sphere"): (8.0, 0.0),
    ("radial", "none"): (8.0, 0.0),
}


def build_report(job, build_ms):
    """The cell-list build (G0-G4) against the HBM roofline: algorithmic bytes / CUDA-event time of
    cute_make_grid for all catalogues of the step (includes its host read-backs)."""
    peak, src = 6650.0, "fallback (B200_PROFILING.md)"
    try:
        peak, src = float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        pass
    nbytes = job.g_data.info().build_bytes + (job.g_rand.info().build_bytes if job.g_rand is not None else 0.0)
    ms = float(np.mean(build_ms)) if build_ms else 0.0
    gbs = nbytes / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
    return {"bound": "hbm", "ms": ms, "algorithmic_bytes": nbytes, "achieved": gbs, "peak": peak, "unit": "GB/s",
            "frac": gbs / peak, "peak_source": src}


def run_ours(args, w, cfg):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1210_1833_b200 import api, runner

    job = runner.job_for_workload(w)          # catalogues resident in HBM from here on
    whichs = list(w.pairs)
    brute = w.grid.get("mode", "none") == "none"
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    nh = job.counter.nhist
    acc = {k: torch.zeros(nh, dtype=torch.int64, device="cuda") for k in whichs}
    pair_ms, pair_pairs, pair_binned = [], [], []

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    build_ms = []

    def one_step(record):
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0.record()
        job.build()                                           # G0-G4 for both catalogues
        b1.record()
        evs = []
        for which in whichs:
            g1, g2 = job.grids(which)
            n = api.cute_count_items(job.kind, g1, g2, job.counter)
            b, e = shard_bounds(n, rank, world, g1.info().nchunks, brute and g2 is None)
            job.opts = api.count_opts(item_begin=b, item_end=max(e, b)) if world > 1 else None
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if not (world > 1 and e <= b):
                job.enqueue(which)                            # P1-P5
            else:
                job.counter.hist.zero_()
            e1.record()
            skipped = world > 1 and e <= b
            st = api.cute_count_status(job.counter) if not skipped else {"evaluated": 0}
            acc[which].copy_(job.counter.hist)
            evs.append((e0, e1, st["evaluated"]))
        if dist is not None:                                  # the one exchange step: sum of partial histograms
            allh = torch.stack([acc[k] for k in whichs])
            dist.all_reduce(allh)
            for i, k in enumerate(whichs):
                acc[k].copy_(allh[i])
        hs = {k: acc[k].cpu().numpy().astype(np.uint64) for k in whichs}
        xi = None
        if set(whichs) >= {"DD", "DR", "RR"}:                 # H1: Landy-Szalay on the host
            xi, _ = api.cute_landy_szalay(hs["DD"], hs["DR"], hs["RR"], job.nd, job.nr)
        elif w.bins.get("box_L", 0.0) > 0 and whichs == ["DD"]:
            xi, _ = api.cute_periodic_xi(hs["DD"], job.nd, w.bins["box_L"], w.bins)
        torch.cuda.synchronize()
        ev_pairs = 0
        if record:
            build_ms.append(b0.elapsed_time(b1))
        for (e0, e1, npairs), k in zip(evs, whichs):
            ev_pairs += npairs
            if record:
                pair_ms.append(e0.elapsed_time(e1))
                pair_pairs.append(npairs)
                pair_binned.append(int(hs[k].sum()) if world == 1 else None)
        return ev_pairs, hs, xi

    for _ in range(args.warmup):
        one_step(False)
    sampler = ClockSampler(local)
    launches0 = api.cute_launch_count()
    barrier()
    sampler.start()
    total_ms, total_pairs = 0.0, 0
    hs = None
    for _ in range(args.steps):
        flush.fill_(1)                                        # L2 flush between timed iterations (untimed)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record()
        npairs, hs, xi = one_step(True)
        s1.record()
        torch.cuda.synchronize()
        total_ms += s0.elapsed_time(s1)
        total_pairs += npairs
    barrier()
    clocks = sampler.stop()
    launches = api.cute_launch_count() - launches0
    t = torch.tensor([total_ms, float(total_pairs)], dtype=torch.float64, device="cuda")
    if dist is not None:
        tmax = t.clone()
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total_ms, total_pairs = float(tmax[0]), float(t[1])
    value = total_pairs / (total_ms * 1e-3) / 1e9

    # ---- end to end through the public host API: host buffers in, host histogram out
    import torch as _t
    host = {}
    for name, cat in (("data", w.data), ("rand", w.rand)):
        if cat is None:
            continue
        need = 2 if job.coord == api.COORD_RADEC else 3
        host[name] = [(_t.from_numpy(np.ascontiguousarray(c)).pin_memory()).numpy() for c in list(cat)[:need]]
    e2e_ws = None
    h2d = d2h = 0

    def e2e_step():
        nonlocal e2e_ws, h2d, d2h
        h2d = d2h = 0
        pairs = 0
        for which in whichs:
            c1 = host["data"] if which in ("DD", "DR") else host["rand"]
            c2 = host["rand"] if which == "DR" else None
            opts = None
            if world > 1:
                g1, g2 = job.grids(which)
                n = api.cute_count_items(job.kind, g1, g2, job.counter)
                b, e = shard_bounds(n, rank, world, g1.info().nchunks, brute and g2 is None)
                opts = api.count_opts(item_begin=b, item_end=max(e, b))
                if e <= b:
                    continue
            h, e2e_ws = api.cute_count_pairs_host(job.kind, c1, c2, job.coord, job.spec, w.bins, workspace=e2e_ws, opts=opts)
            h2d += sum(a.nbytes for a in c1) + (sum(a.nbytes for a in c2) if c2 is not None else 0)
            d2h += h.nbytes
            n1, n2 = len(c1[0]), (len(c2[0]) if c2 is not None else 0)
            pairs += n1 * n2 if c2 is not None else n1 * (n1 - 1) // 2
        return pairs

    e2e_step()
    barrier()
    t0 = time.perf_counter()
    e2e_pairs = 0
    for _ in range(args.steps):
        e2e_pairs += e2e_step()
    barrier()
    e2e_s = time.perf_counter() - t0
    if brute and world == 1:
        e2e_val = e2e_pairs / e2e_s / 1e9
    else:   # grid-assisted or sharded: the evaluated separations are the device arm's
        e2e_val = (total_pairs / args.steps) * args.steps / e2e_s / 1e9 if world == 1 else None
    if dist is not None:
        te = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e_val = total_pairs / float(te[0]) / 1e9

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return
    # ---- roofline of the dominant kernel (the pair kernel): algorithmic lane-instructions / duration
    i_all, i_bin = ALG_INSTR[(w.kind, w.grid.get("mode", "none"))]
    ops = sum(p * i_all + (b or 0) * i_bin for p, b in zip(pair_pairs, pair_binned))
    kern_s = sum(pair_ms) * 1e-3
    achieved = ops / kern_s / 1e12 if kern_s > 0 else 0.0
    peak = SM_COUNT * LANES_PER_SM * SM_MAX_MHZ * 1e6 / 1e12
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic", "config": cfg, "clocks": clocks, "gpu_launches": int(launches),
           "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
           "roofline": {"bound": "alu", "kernel": "pair_kernel", "achieved": achieved, "peak": peak, "unit": "T lane-instr/s",
                        "frac": achieved / peak,
                        "traffic": NCU_TRAFFIC_BYTES.get(args.config) if args.scale == 1.0 and world == 1 else None,
                        "traffic_unit": "bytes of DRAM per pair-kernel launch (ncu, profiles/r01_pair_kernel_c2.md)",
                        "peak_source": "148 SMs x 128 FP32 lanes x 1965 MHz (guide unit counts and max clock; DESIGN.md)",
                        "pair_kernel_share_of_step": kern_s / (total_ms * 1e-3),
                        "pairs_per_s_in_kernel": sum(pair_pairs) / kern_s if kern_s > 0 else 0.0,
                        "alg_instr_per_pair": [i_all, i_bin]},
           "build": build_report(job, build_ms),
           "rates": {"evaluated_pairs_per_step": total_pairs / args.steps,
                     "binned_pairs_per_step": (sum(b for b in pair_binned if b is not None) / args.steps) if world == 1 else None}}
    if world == 1 and not args.no_cpu_baseline:
        v, cores, sample = oracle_sample(w)
        out["cpu_baseline"] = {"value": v / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config 1..5 (default 2: the metric's workload)")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the catalogues (debugging only; 1.0 = the named config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--grid", default="default", choices=["default", "none", "sphere", "box3d"],
                    help="override the workload's neighbour search (default: the one BASELINE.json names)")
    ap.add_argument("--pix", type=float, default=0.1, help="--grid sphere: pixel side in units of theta_max")
    args = ap.parse_args()
    from paper_1210_1833_b200 import synth
    w = synth.workload(args.config, args.scale)
    if args.grid == "none":
        w.grid = dict(mode="none")
    elif args.grid == "sphere":
        w.grid = dict(mode="sphere", thetamax=w.bins["aperture"] if w.kind == "radial" else w.bins["hi1"], pix=args.pix)
    elif args.grid == "box3d":
        w.grid = dict(mode="box3d", rmax=w.bins["hi1"])
    cfg = {"workload": f"BASELINE.json configs[{args.config - 1}] ({w.name}: {w.kind}, {'+'.join(w.pairs)}, "
                       f"nd={len(w.data[0])}, nr={len(w.rand[0]) if w.rand is not None else 0}, bins={w.bins['n1']}x{max(w.bins.get('n2', 0), 1)}, "
                       f"grid={w.grid.get('mode', 'none')})",
           "scale": args.scale, "l2": "256 MiB buffer written between timed iterations (L2 flush)",
           "parallelism": f"work items sharded over {args.gpus} GPU(s), catalogues replicated, one all-reduce of the histogram"}
    w.grid = dict(w.grid, no_perm=1)      # pair counting never reads the sort permutation: do not write it
    if args.impl == "reference":
        run_reference(args, w, cfg)
    else:
        run_ours(args, w, cfg)


if __name__ == "__main__":
    main()
