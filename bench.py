#!/usr/bin/env python
"""bench.py -- headline benchmark of the CUTE pair-counting hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl ours|reference]

A "step" is one pass of the whole hot path over one batch of synthetic input: the cell-list
build (G0-G4, cute_make_grid) of the data and random catalogues, the pair counts the config names
(P1-P5, cute_count_pairs: DD, DR, RR) and the estimator on the host (H1).  The headline workload is
BASELINE.json configs[4] ("C5": periodic-box monopole, 10M x 10M float32 points through the 3-D
cell list, DD + DR, 1.6e12 separations per step) -- the largest single-GPU configuration.  The same
JSON line carries `per_config`: every one of the five configurations at full size, each with its
per-count times, the three rates of SURVEY.md 8(d) (evaluated / binned / brute-equivalent pairs per
second), the pair kernel's roofline, the cell build against the HBM roofline, the end-to-end
number through cute_count_pairs_host and the oracle timed on the host cores beside it.

N > 1 (torchrun): the work-item list of every pair count is split over the ranks (catalogues
replicated; every rank builds the grids and then takes rank 0's cell-sorted arrays by one NCCL
broadcast, because the order inside a cell differs from build to build and the shards must
enumerate the same points), and the partial uint64 histograms are summed with one NCCL
all-reduce.  Total work is fixed: "scaling": "strong".

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
HEADLINE = 5
SM_MAX_MHZ_FALLBACK = 1965.0
VALUE_IS = ("binned pairs per second: the sum of the histograms the step fills (pairs counted into bins, Eq. 11 PAPER.md:85) over the "
            "time of the whole step (build + counts + estimator); evaluated separations/s and brute-force-equivalent pairs/s are in rates")


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
def oracle_setup_seconds(o, w, c2, mode):
    """The oracle's one-off set-up per call (argument conversion, and for mode `celled` its serial cell list over both
    catalogues), measured with an EMPTY i-range: no pair is evaluated."""
    t0 = time.perf_counter()
    o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, 0))
    return time.perf_counter() - t0


def oracle_sample(w, seconds: float = 12.0):
    """Time the oracle, as it stands, on all host cores on a bounded sample of the workload's cross (or only) count: a
    fixed slice of the i-range, 1/64 of it unless that would exceed about `seconds`.  The rate is the
    STEADY-STATE one: the per-call set-up (measured with an empty i-range) is subtracted and stated.
    Returns (binned pairs per second, evaluated separations per second, cores, description)."""
    from oracle import oracle as o
    o.build()
    cores = o.max_threads()
    c2 = w.rand if w.rand is not None else None
    mode = "plain" if w.grid.get("mode", "none") == "none" else "celled"
    n1 = len(w.data[0])
    setup = min(oracle_setup_seconds(o, w, c2, mode) for _ in range(2))
    probe = min(n1, 256)
    t0 = time.perf_counter()
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, probe))
    per_row = max(time.perf_counter() - t0 - setup, 1e-6) / probe
    m = int(min(n1, max(probe, 2.0 / per_row, min(n1 // 64, seconds / per_row))))   # 1/64, but between ~2 s and ~`seconds` of work
    t0 = time.perf_counter()
    r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, m))
    dt = time.perf_counter() - t0
    work = max(dt - setup, 1e-9)
    what = "DR" if c2 is not None else "DD"
    frac = "1/64 of the i-range" if m == n1 // 64 else f"{m / n1:.4f} of the i-range"
    return (float(r["hist"].sum()) / work, r["npairs"] / work, cores,
            f"{what} rows [0,{m}) of {n1} ({frac}) x all of catalogue 2, oracle mode {mode}: {r['npairs']} separations evaluated, "
            f"{int(r['hist'].sum())} binned, in {dt:.2f} s of which {setup:.2f} s is the oracle's per-call set-up "
            f"(measured with an empty i-range and EXCLUDED from the rate: steady state)")


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
    setup = min(oracle_setup_seconds(o, w, c2, mode) for _ in range(2))
    probe = min(n1, 256)
    t0 = time.perf_counter()
    o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, probe))
    per_row = max(time.perf_counter() - t0 - setup, 1e-6) / probe
    # bounded sample per step: 1/64 of the i-range, but between ~1 s and ~6 s of pair work (plus the set-up)
    rows = int(min(n1, max(probe, 1.0 / per_row, min(n1 // 64, 6.0 / per_row))))
    for _ in range(args.warmup):
        o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, rows))
    binned = evaluated = 0
    t0 = time.perf_counter()
    for _ in range(args.steps):
        r = o.count(w.kind, w.data, c2, w.bins, mode=mode, i_range=(0, rows))
        binned += int(r["hist"].sum())
        evaluated += r["npairs"]
    dt = time.perf_counter() - t0
    work = max(dt - args.steps * setup, 1e-9)
    v = binned / work / 1e9
    sample = (f"each step: rows [0,{rows}) of {n1} x catalogue 2 ({'DR' if c2 is not None else 'DD'}), oracle mode {mode}; rate = binned pairs / "
              f"(time - {setup:.2f} s per-call set-up, measured with an empty i-range): steady state; evaluated separations/s = {evaluated / work / 1e9:.4f}e9")
    print(json.dumps({"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
                      "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "strong",
                      "vs_baseline": None, "dtype": "f64", "data": "synthetic", "config": cfg,
                      "value_is": VALUE_IS,
                      "rates": {"binned_per_s": binned / work, "evaluated_per_s": evaluated / work, "setup_s_per_call_excluded": setup},
                      "cpu_baseline": {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


# ------------------------------------------------------------------------------- our arm
# The roofline yardstick, pinned to SURVEY.md 8(d) R3 so that it cannot move with the implementation.  Lane-operations per
# pair that the METHOD needs (scalar float32 / integer operations, independent of our SASS):
#   all  = per evaluated pair: the separation (3 FADD + FMUL + 2 FFMA) + the range test            [R3: "8 flops", compare]
#   bin  = extra per binned pair: the map to a bin (SQRT or LG2 (+ the theta cubic), one scale FFMA per axis, the (r,mu) /
#          (pi,sigma) geometry), the address and the increment                                     [R3: MUFU, FFMA, address, atomic]
#   filt = extra per binned pair that exists ONLY because of this implementation's float32-filter design (round-to-nearest +
#          distance to the edge, clamps onto the dump borders, the certainty test): reported separately, NOT in `frac`
# Recorded changes of method against R3's table: angular and (r,mu) use float32 unit vectors / coordinates with the rare float64
# recomputation instead of hi/lo arithmetic on every pair (R3's 9 FADD -> 3); the periodic brute-force minimum image costs
# 2 per axis (L - |d|, min) as in R3.  fp_* = the float32-pipe part, mufu and atom per binned pair.
ALG = {
    "angular": dict(all=7.0, bin=8.0, filt=7.0, fp_all=6.0, fp_bin=8.0, mufu=1.0, atom=1.0),     # cubic (3) + FMUL + LG2 + FFMA + address + increment
    "monopole": dict(all=7.0, bin=4.0, filt=5.0, fp_all=6.0, fp_bin=4.0, mufu=1.0, atom=1.0),    # SQRT + FFMA + address + increment | filt: 3 (rint, frac) + clamp + test
    "monopole_minimg": dict(all=13.0, bin=4.0, filt=5.0, fp_all=9.0, fp_bin=4.0, mufu=1.0, atom=1.0),
    "rmu": dict(all=7.0, bin=14.0, filt=7.0, fp_all=6.0, fp_bin=15.0, mufu=2.0, atom=1.0),       # s.l (3) + |l|^2 (2) + FMUL + RSQ + FMUL + SQRT + 2 FFMA + IMAD + address + increment
    "pisigma": dict(all=7.0, bin=17.0, filt=7.0, fp_all=6.0, fp_bin=18.0, mufu=2.0, atom=1.0),   # + pi = r mu, sigma^2 = r^2 - pi^2, SQRT
    "radial": dict(all=8.0, bin=0.0, filt=0.0, fp_all=6.0, fp_bin=0.0, mufu=0.0, atom=0.0),
}


def alg_for(w):
    if w.kind == "monopole" and w.grid.get("mode", "none") == "none" and w.bins.get("box_L", 0.0) > 0:
        return ALG["monopole_minimg"]
    return ALG[w.kind]


def hbm_peak():
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


def ncu_traffic(cfg_id: int):
    """dram bytes per pair-kernel launch, and the issue-slot utilisation, from the committed ncu captures, if there are any."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "r02_traffic.json")))
        e = t.get(f"C{cfg_id}")
        return (e["dram_bytes_per_launch"], e["source"]) if e else (None, None)
    except Exception:
        return None, None


def ncu_issue_active(cfg_id: int):
    try:
        e = json.load(open(os.path.join(ROOT, "profiles", "ncu_readings.json"))).get(f"C{cfg_id}")
        return e if e else None
    except Exception:
        return None


def workload_for(cfg_id: int, scale: float, args=None):
    from paper_1210_1833_b200 import synth
    w = synth.workload(cfg_id, scale)
    if args is not None:
        if args.grid == "none":
            w.grid = dict(mode="none")
        elif args.grid == "sphere":
            w.grid = dict(mode="sphere", thetamax=w.bins["aperture"] if w.kind == "radial" else w.bins["hi1"], pix=args.pix)
        elif args.grid == "box3d":
            w.grid = dict(mode="box3d", rmax=w.bins["hi1"])
    w.grid = dict(w.grid, no_perm=1)      # pair counting never reads the sort permutation: do not write it
    return w


def describe(cfg_id, w, scale):
    return (f"BASELINE.json configs[{cfg_id - 1}] ({w.name}: {w.kind}, {'+'.join(w.pairs)}, "
            f"nd={len(w.data[0])}, nr={len(w.rand[0]) if w.rand is not None else 0}, bins={w.bins['n1']}x{max(w.bins.get('n2', 0), 1)}, "
            f"grid={w.grid.get('mode', 'none')}, scale={scale})")


class Runner:
    """One configuration resident on the device; times steps of the whole hot path."""

    def __init__(self, cfg_id, w, rank, world, dist, flush):
        from paper_1210_1833_b200 import api, runner
        import torch
        self.api, self.torch = api, torch
        self.cfg_id, self.w, self.rank, self.world, self.dist, self.flush = cfg_id, w, rank, world, dist, flush
        self.job = runner.job_for_workload(w)          # catalogues resident in HBM from here on
        self.whichs = list(w.pairs)
        self.brute = w.grid.get("mode", "none") == "none"
        nh = self.job.counter.nhist
        self.acc = {k: torch.zeros(nh, dtype=torch.int64, device="cuda") for k in self.whichs}
        # launch-latency-scale counts (C1, C4) are looped inside the events: one count = the mean of `inner`
        self.inner = 100 if cfg_id in (1, 4) else 1

    def step(self, record=None):
        """One pass: build both grids, every pair count, all-reduce (N > 1), estimator on the host."""
        torch, api, job = self.torch, self.api, self.job
        b0, b1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b0.record()
        # G0-G4 for both catalogues; N > 1: every rank then takes rank 0's cell-sorted arrays (the order inside a cell
        # differs from build to build, and the item shards must enumerate the same points on every rank)
        job.build(share=(lambda t: self.dist.broadcast(t, src=0)) if self.dist is not None else None)
        b1.record()
        evs = []
        for which in self.whichs:
            g1, g2 = job.grids(which)
            skipped = False
            if self.world > 1:
                n = api.cute_count_items(job.kind, g1, g2, job.counter)
                b, e = api.cute_shard_items(n, g1.info().nchunks, self.rank, self.world, self.brute and g2 is None)
                job.opts = api.count_opts(item_begin=b, item_end=e, shard=1)
                skipped = e <= b
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            if skipped:
                job.counter.hist.zero_()
            else:
                job.enqueue(which)                            # P1-P5
            e1.record()
            st = api.cute_count_status(job.counter) if not skipped else {"evaluated": 0, "refined": 0}
            self.acc[which].copy_(job.counter.hist)
            evs.append((e0, e1, st))
        if self.dist is not None:                             # the one exchange step: sum of partial histograms
            allh = torch.stack([self.acc[k] for k in self.whichs])
            self.dist.all_reduce(allh)
            for i, k in enumerate(self.whichs):
                self.acc[k].copy_(allh[i])
        hs = {k: self.acc[k].cpu().numpy().astype(np.uint64) for k in self.whichs}
        w = self.w
        if set(self.whichs) >= {"DD", "DR", "RR"}:            # H1: Landy-Szalay on the host
            api.cute_landy_szalay(hs["DD"], hs["DR"], hs["RR"], job.nd, job.nr)
        elif w.bins.get("box_L", 0.0) > 0 and self.whichs == ["DD"]:
            api.cute_periodic_xi(hs["DD"], job.nd, w.bins["box_L"], w.bins)
        torch.cuda.synchronize()
        ev_pairs = 0
        binned = sum(int(hs[k].sum()) for k in self.whichs)   # the whole job's (N > 1: after the all-reduce)
        for (e0, e1, st), k in zip(evs, self.whichs):
            ev_pairs += st["evaluated"]
            if record is not None:
                record["counts"].setdefault(k, []).append(dict(ms=e0.elapsed_time(e1), evaluated=st["evaluated"], refined=st["refined"],
                                                               binned=int(hs[k].sum()) if self.world == 1 else None))
        if record is not None:
            record["build_ms"].append(b0.elapsed_time(b1))
        return ev_pairs, binned

    def time_counts_looped(self, record):
        """C1 / C4: one pair count lasts ~0.2-0.4 ms, so it is looped >= 100x inside one pair of events."""
        torch, job = self.torch, self.job
        for which in self.whichs:
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(self.inner):
                job.enqueue(which)
            e1.record()
            torch.cuda.synchronize()
            for c in record["counts"][which]:
                c["ms"] = e0.elapsed_time(e1) / self.inner
                c["looped"] = self.inner

    def timed(self, steps, warmup, sampler=None):
        torch = self.torch
        for _ in range(warmup):
            self.step(None)
        record = {"counts": {}, "build_ms": []}
        if self.dist is not None:
            self.dist.barrier()
        torch.cuda.synchronize()
        if sampler is not None:
            sampler.start()
        total_ms, total_pairs, total_binned = 0.0, 0, 0
        for _ in range(steps):
            self.flush.fill_(1)                               # L2 flush between timed iterations (untimed)
            torch.cuda.synchronize()
            s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            s0.record()
            ev, bn = self.step(record)
            total_pairs += ev
            total_binned += bn
            s1.record()
            torch.cuda.synchronize()
            total_ms += s0.elapsed_time(s1)
        if self.dist is not None:
            self.dist.barrier()
        torch.cuda.synchronize()
        clocks = sampler.stop() if sampler is not None else None
        if self.inner > 1 and self.world == 1:
            self.time_counts_looped(record)
        return total_ms, (total_pairs, total_binned), record, clocks

    def e2e(self, steps):
        """The same metric through cute_count_pairs_host: pinned host buffers in, host histogram out, every step."""
        torch, api, job, w = self.torch, self.api, self.job, self.w
        host = {}
        for name, cat in (("data", w.data), ("rand", w.rand)):
            if cat is None:
                continue
            need = 2 if job.coord == api.COORD_RADEC else 3
            dt = np.float64 if np.asarray(cat[0]).dtype not in (np.float32, np.float64) else np.asarray(cat[0]).dtype
            host[name] = [(torch.from_numpy(np.ascontiguousarray(c, dtype=dt)).pin_memory()).numpy() for c in list(cat)[:need]]
        ws = None
        h2d = d2h = 0

        def one():
            nonlocal ws, h2d, d2h
            h2d = d2h = 0
            if self.world > 1:
                # N > 1: the item shards need identical grids on every rank (Job.build(share)), which the one-call host entry
                # point cannot give: the same public calls one by one -- pinned host -> device copies, cute_make_grid,
                # broadcast, cute_count_pairs on this rank's items, all-reduce, histograms back to the host (Runner.step)
                for name, dev in (("data", job.d_data), ("rand", job.d_rand)):
                    if dev is None:
                        continue
                    for d, hcol in zip(dev, host[name]):
                        d.copy_(torch.from_numpy(hcol), non_blocking=True)
                        h2d += hcol.nbytes
                self.step(None)
                d2h += 8 * job.counter.nhist * len(self.whichs)
                return
            for which in self.whichs:
                c1 = host["data"] if which in ("DD", "DR") else host["rand"]
                c2 = host["rand"] if which == "DR" else None
                opts = None
                if self.world > 1:
                    g1, g2 = job.grids(which)
                    n = api.cute_count_items(job.kind, g1, g2, job.counter)
                    b, e = api.cute_shard_items(n, g1.info().nchunks, self.rank, self.world, self.brute and g2 is None)
                    if e <= b:
                        continue
                    opts = api.count_opts(item_begin=b, item_end=e, shard=1)
                h, ws = api.cute_count_pairs_host(job.kind, c1, c2, job.coord, job.spec, w.bins, workspace=ws, opts=opts)
                h2d += sum(a.nbytes for a in c1) + (sum(a.nbytes for a in c2) if c2 is not None else 0)
                d2h += h.nbytes

        one()
        if self.dist is not None:
            self.dist.barrier()
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            one()
        torch.cuda.synchronize()
        if self.dist is not None:
            self.dist.barrier()
        return time.perf_counter() - t0, h2d, d2h


def summarise(cfg_id, w, scale, rn, total_ms, record, steps, peaks, clock_mhz, e2e=None, cpu=None):
    """The per-config entry: times, the three rates, rooflines."""
    job = rn.job
    a = alg_for(w)
    counts = {}
    kern_ms = ops = fp_ops = filt_ops = 0.0
    evaluated = binned = brute = mufu = atoms = 0.0
    for which, lst in record["counts"].items():
        ms = float(np.mean([c["ms"] for c in lst]))
        ev = float(np.mean([c["evaluated"] for c in lst]))
        bn = float(np.mean([c["binned"] or 0 for c in lst]))
        tot = float(job.total_pairs(which))
        counts[which] = {"ms": ms, "evaluated_pairs": ev, "binned_pairs": bn, "brute_equivalent_pairs": tot, "refined_pairs": float(np.mean([c["refined"] for c in lst])),
                         "evaluated_per_s": ev / (ms * 1e-3), "binned_per_s": bn / (ms * 1e-3), "brute_equivalent_per_s": tot / (ms * 1e-3)}
        if lst[0].get("looped"):
            counts[which]["looped_inside_events"] = lst[0]["looped"]
        kern_ms += ms
        evaluated += ev; binned += bn; brute += tot
        ops += ev * a["all"] + bn * a["bin"]
        filt_ops += bn * a["filt"]
        fp_ops += ev * a["fp_all"] + bn * a["fp_bin"]
        mufu += bn * a["mufu"]; atoms += bn * a["atom"]
    kern_s = kern_ms * 1e-3
    sms = peaks["sms"]
    clk = clock_mhz * 1e6
    issue_peak = peaks["lane_instr_per_clk_sm"] * sms * clk / 1e12           # T lane-instr/s
    achieved = ops / kern_s / 1e12 if kern_s > 0 else 0.0
    achieved_f = (ops + filt_ops) / kern_s / 1e12 if kern_s > 0 else 0.0
    ncu = ncu_issue_active(cfg_id) if scale == 1.0 else None
    # the other units of SURVEY.md 8(d) R2, as upper bounds on evaluated pairs per second for THIS workload's mix
    per_pair = lambda x: x / max(evaluated, 1.0)
    bounds = {"issue": peaks["lane_instr_per_clk_sm"] / max(per_pair(ops + filt_ops), 1e-9),
              "fp32_pipe": peaks["fp32_lane_ops_per_clk_sm"] / max(per_pair(fp_ops), 1e-9),
              "mufu": peaks["mufu_per_clk_sm"] / max(per_pair(mufu), 1e-9) if mufu > 0 else None,
              "shared_atomic": peaks["atoms_per_clk_sm"] / max(per_pair(atoms), 1e-9) if atoms > 0 else None}
    bounds_s = {k: (v * sms * clk if v is not None else None) for k, v in bounds.items()}
    binding = min((k for k in bounds_s if bounds_s[k] is not None), key=lambda k: bounds_s[k])
    nbytes = job.g_data.info().build_bytes + (job.g_rand.info().build_bytes if job.g_rand is not None else 0.0)
    bms = float(np.mean(record["build_ms"])) if record["build_ms"] else 0.0
    hbm, hsrc = hbm_peak()
    gbs = nbytes / (bms * 1e-3) / 1e9 if bms > 0 else 0.0
    traffic, tsrc = ncu_traffic(cfg_id) if scale == 1.0 else (None, None)
    out = {"config": f"C{cfg_id}", "workload": describe(cfg_id, w, scale), "steps": steps, "ms_per_step": total_ms / steps,
           "counts": counts,
           "rates": {"evaluated_per_s": evaluated / kern_s if kern_s else 0.0, "binned_per_s": binned / kern_s if kern_s else 0.0,
                     "brute_equivalent_per_s": brute / kern_s if kern_s else 0.0, "in_range_fraction": binned / max(evaluated, 1.0),
                     "binned_per_s_whole_step": binned / (total_ms / steps * 1e-3) if total_ms > 0 else 0.0,
                     "rates_are": "per second of pair-kernel time (sum of the counts' events); binned_per_s_whole_step divides by the whole step",
                     "time_to_solution_ms": total_ms / steps},
           "roofline": {"bound": "alu", "kernel": "pair_kernel", "achieved": achieved, "peak": issue_peak, "unit": "T lane-instr/s",
                        "frac": achieved / issue_peak if issue_peak else 0.0,
                        "frac_is": "the METHOD's lane-operations (SURVEY.md 8(d) R3: alg_instr_per_pair = [per evaluated pair, extra per binned pair]) "
                                   "over time, against the measured issue rate; the float32-filter instructions of this implementation are NOT counted",
                        "alg_instr_per_pair": [a["all"], a["bin"]],
                        "alg_instr_per_evaluated_pair": per_pair(ops),
                        "filter_overhead_instr_per_binned_pair": a["filt"],
                        "filter_overhead_instr_per_evaluated_pair": per_pair(filt_ops),
                        "frac_incl_filter_overhead": achieved_f / issue_peak if issue_peak else 0.0,
                        "ncu_issue_active": ncu,
                        "binding_unit": binding,
                        "bounds_pairs_per_s": bounds_s, "frac_of_binding_bound": (evaluated / kern_s) / bounds_s[binding] if kern_s else 0.0,
                        "pair_kernel_share_of_step": kern_s / (total_ms / steps * 1e-3) if rn.inner == 1 else None,
                        "traffic": traffic, "traffic_source": tsrc},
           "build": {"bound": "hbm", "ms": bms, "algorithmic_bytes": nbytes, "achieved": gbs, "peak": hbm, "unit": "GB/s",
                     "frac": gbs / hbm, "peak_source": hsrc}}
    if e2e is not None:
        out["e2e"] = e2e
    if cpu is not None:
        out["cpu_baseline"] = cpu
    return out


def density_grid_entry(api, torch, peaks_hbm, peaks, clock_mhz):
    """the density-grid monopole (Eq. 17) on the C5 data catalogue, 128^3 grid,
    C5's bins.  The TSC scatter is timed alone through a bin spec no offset falls in (the stencil is then skipped)."""
    from paper_1210_1833_b200 import synth
    w = synth.workload(5, 1.0)
    cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in w.data]
    L, ng, n = w.bins["box_L"], 128, len(w.data[0])
    bins = dict(n1=w.bins["n1"], lo1=0.0, hi1=w.bins["hi1"])
    tiny = dict(n1=1, lo1=0.0, hi1=0.5 * L / ng)

    def timed(b, reps=3):
        out = api.cute_density_grid_xi(cols, L, ng, b)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            out = api.cute_density_grid_xi(cols, L, ng, b, workspace=out["workspace"])
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / reps, out

    ms_tsc, _ = timed(tiny)
    ms_all, out = timed(bins)
    pairs = float(out["npairs"].sum())
    hbm, hsrc = peaks_hbm
    tsc_bytes = n * 12.0 + 2.0 * ng ** 3 * 8.0          # read the particles once; zero and write the grid
    ms_st = max(ms_all - ms_tsc, 1e-6)
    return {"config": "N4", "workload": f"density-grid monopole (PAPER.md:250-260): C5 data, n={n}, grid {ng}^3, {bins['n1']} bins to {bins['hi1']}",
            "ms_total": ms_all, "ms_tsc_and_overdensity": ms_tsc, "ms_stencil": ms_st,
            "grid_point_pairs": pairs, "grid_point_pairs_per_s": pairs / (ms_st * 1e-3),
            "tsc": {"bound": "hbm", "algorithmic_bytes": tsc_bytes, "achieved": tsc_bytes / (ms_tsc * 1e-3) / 1e9, "peak": hbm, "unit": "GB/s",
                    "frac": tsc_bytes / (ms_tsc * 1e-3) / 1e9 / hbm, "peak_source": hsrc,
                    "note": "27 float64 atomics per particle into the L2-resident grid (three lanes per particle: adjacent triples per instruction): bound by the L2 atomic units, not by HBM"},
            "stencil": {"bound": "alu", "unit": "T float64 multiply-adds/s", "algorithmic_fma": pairs, "executed_fma": 0.5 * pairs,
                        "achieved": 0.5 * pairs / (ms_st * 1e-3) / 1e12,
                        "peak": peaks["table"].get("dfma", 0.0) * peaks["sms"] * clock_mhz * 1e6 / 1e12,
                        "frac": (0.5 * pairs / (ms_st * 1e-3)) / max(peaks["table"].get("dfma", 0.0) * peaks["sms"] * clock_mhz * 1e6, 1.0),
                        "peak_source": "cute_measure_peaks `dfma` (this device, this run) x SMs x SM clock",
                        "note": "one float64 multiply-add per ORDERED grid-point pair is the algorithmic count (Eq. 17); the kernel sweeps "
                                "half of the offsets (xi is even) and counts them twice: `achieved` and `frac` are the EXECUTED multiply-adds "
                                "(algorithmic / 2) over time.  ms_stencil = ms_total - ms_tsc still contains the host-side offset table and "
                                "the read-back of the sums (built once per call), so the kernel alone is somewhat faster than this"}}


def paper_table2_entry(api, torch):
    """CONTEXT ONLY: the five shapes of the paper's Table II -- "the time to
    fill one DR histogram by brute force" -- on a synthetic stand-in for its MICE subset: 3e5 uniform objects in the
    wedge 0 < RA, Dec < 18 deg, 0.5 < z < 0.6, against as many randoms (the paper never states the size of its random
    catalogue: ASSUMED equal to the data).  Not the metric, not a target; the paper's times are other hardware."""
    from paper_1210_1833_b200 import runner, synth
    n = 300000
    ra, dec, z, xyz = synth.uniform_wedge(n, 18.0, 18.0, 0.5, 0.6, synth.seed_for(9, 0))
    rra, rdec, rz, rxyz = synth.uniform_wedge(n, 18.0, 18.0, 0.5, 0.6, synth.seed_for(9, 1))
    base = dict(log1=0, n2=0, lo2=0.0, hi2=0.0, aperture=0.0, box_L=0.0)
    th = math.radians(30.0)
    shapes = [
        ("xi(r), 256 linear bins, r < 100 Mpc/h", "monopole", tuple(xyz), tuple(rxyz), dict(base, n1=256, lo1=0.0, hi1=100.0), 13.0),
        ("xi_log(r), 256 log bins, 50 per decade, r < 100 Mpc/h", "monopole", tuple(xyz), tuple(rxyz),
         dict(base, n1=256, lo1=100.0 / 10.0 ** (256 / 50.0), hi1=100.0, log1=1), 20.0),
        ("w(theta), 256 linear bins, theta < 30 deg", "angular", (ra, dec), (rra, rdec), dict(base, n1=256, lo1=0.0, hi1=th), 22.0),
        ("xi(pi,sigma), 64 x 64 bins to 100 Mpc/h", "pisigma", tuple(xyz), tuple(rxyz),
         dict(base, n1=64, lo1=0.0, hi1=100.0, n2=64, lo2=0.0, hi2=100.0), 27.0),
    ]
    rows = []

    def time_dr(job, reps=3):
        job.build()
        job.count("DR")
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            job.enqueue("DR")
        e1.record()
        torch.cuda.synchronize()
        st = api.cute_count_status(job.counter)
        return e0.elapsed_time(e1) / reps, st

    for name, kind, d, r, bins, paper_s in shapes:
        job = runner.Job(kind, d, r, bins, dict(mode="none"))
        ms, st = time_dr(job)
        rows.append({"shape": name, "ms_per_DR_histogram": ms, "pairs": float(n) * n, "pairs_per_s": float(n) * n / (ms * 1e-3),
                     "refined_pairs": float(st["refined"]), "paper_server_gpu_s": paper_s})
        del job
    # w_pix(theta): pixels of 5e-3 sq-deg, both catalogues pixelised on the device, weighted pixel-pixel counts
    side = math.sqrt(5e-3)
    nra = int(round(18.0 / side))
    u1 = math.sin(math.radians(18.0))
    nu = int(round(u1 / (5e-3 / (18.0 / nra) * math.pi / 180.0)))
    pix = []
    for a, b in ((ra, dec), (rra, rdec)):
        cols = [torch.from_numpy(np.ascontiguousarray(c)).cuda() for c in (a, b)]
        pra, pdec, pw = api.cute_pixelize(cols, 0.0, 18.0, 0.0, u1, nra, nu)
        pix.append(((pra.cpu().numpy(), pdec.cpu().numpy()), pw.cpu().numpy().view(np.uint32)))
    (cd, wd), (cr, wr) = pix
    job = runner.Job("angular", cd, cr, dict(base, n1=256, lo1=0.0, hi1=th), dict(mode="none"), None, w_data=wd, w_rand=wr)
    ms, st = time_dr(job)
    rows.append({"shape": f"w_pix(theta), pixels of 5e-3 sq-deg ({len(wd)} x {len(wr)} non-empty pixels), 256 linear bins",
                 "ms_per_DR_histogram": ms, "pairs": float(len(wd)) * len(wr), "pairs_per_s": float(len(wd)) * len(wr) / (ms * 1e-3),
                 "refined_pairs": float(st["refined"]), "paper_server_gpu_s": 0.46})
    return {"config": "paper_table2", "workload": "CONTEXT: the shapes of the paper's Table II on a synthetic wedge (3e5 x 3e5, randoms ASSUMED as "
            "many as data; brute force, one DR histogram each); paper_server_gpu_s = Tesla C2070 (PAPER.md:296-302)", "rows": rows}


def measured_peaks(api, torch):
    """Roofline denominators measured on this device in this run (cute_measure_peaks: SURVEY.md 8(d) R2)."""
    pk = api.cute_measure_peaks()
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    return {"sms": sms,
            "lane_instr_per_clk_sm": max(pk["ffma"][0], pk["fmnmx"][0], pk["iadd"][0]),   # one instruction slot per lane and clock
            "fp32_lane_ops_per_clk_sm": max(pk["ffma2"][0], pk["fadd2"][0], pk["ffma"][0]),
            "mufu_per_clk_sm": pk["mufu_sqrt"][0],
            "atoms_per_clk_sm": pk["atoms_inc_cols8_random_bins"][0],
            "table": {k: v[0] for k, v in pk.items()},
            "source": "cute_measure_peaks (clock64 microbenchmarks on this device, this run): lane-operations per clock per SM"}


def run_ours(args):
    import torch
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    from paper_1210_1833_b200 import api

    peaks = measured_peaks(api, torch)
    if args.n4_only:                                   # the density-grid entry alone (profiling: profiles/r03_n4.md)
        print(json.dumps(density_grid_entry(api, torch, hbm_peak(), peaks, SM_MAX_MHZ_FALLBACK)))
        return
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    head_id = args.config
    w = workload_for(head_id, args.scale, args)
    rn = Runner(head_id, w, rank, world, dist, flush)
    sampler = ClockSampler(local)
    launches0 = api.cute_launch_count()
    total_ms, (total_pairs, total_binned), record, clocks = rn.timed(args.steps, args.warmup, sampler)
    launches = api.cute_launch_count() - launches0
    t = torch.tensor([total_ms, float(total_pairs)], dtype=torch.float64, device="cuda")
    if dist is not None:
        tmax = t.clone()
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
        total_ms, total_pairs = float(tmax[0]), float(t[1])     # (total_binned is already the whole job's: all-reduced histograms)
    value = total_binned / (total_ms * 1e-3) / 1e9              # the metric as worded: pairs counted into bins per second
    clock_mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz") or SM_MAX_MHZ_FALLBACK

    # ---- end to end through the public host API
    e2e_s, h2d, d2h = rn.e2e(args.steps)
    if dist is not None:
        te = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(te, op=dist.ReduceOp.MAX)
        e2e_s = float(te[0])
    e2e_val = total_binned / e2e_s / 1e9      # the same binned pairs, over the end-to-end wall time
    e2e = {"value": e2e_val, "evaluated_per_s": total_pairs / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
           "ms_per_step": 1e3 * e2e_s / args.steps, "api": "cute_count_pairs_host"}
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        v, vev, cores, sample = oracle_sample(w)
        cpu = {"value": v / 1e9, "unit": UNIT, "evaluated_per_s": vev, "cores": cores, "kind": "oracle", "sample": sample}
    head = summarise(head_id, w, args.scale, rn, total_ms, record, args.steps, peaks, clock_mhz, e2e, cpu) if world == 1 else None
    del rn
    torch.cuda.empty_cache()

    # ---- every other configuration at full size (world == 1; the headline's own entry is reused)
    per_config = []
    if world == 1 and not args.only:
        for cid in (1, 2, 3, 4, 5):
            if cid == head_id:
                per_config.append(head)
                continue
            wc = workload_for(cid, args.scale)
            rc = Runner(cid, wc, 0, 1, None, flush)
            ksteps = max(3, min(args.steps, 5))
            tms, (tp, tb), rec, _ = rc.timed(ksteps, 3)
            es, eh, ed = rc.e2e(ksteps)
            ec = {"value": tb / es / 1e9, "evaluated_per_s": tp / es, "unit": UNIT, "h2d_bytes_per_step": int(eh), "d2h_bytes_per_step": int(ed),
                  "ms_per_step": 1e3 * es / ksteps, "api": "cute_count_pairs_host"}
            cc = None
            if not args.no_cpu_baseline:
                v, vev, cores, sample = oracle_sample(wc, seconds=6.0)
                cc = {"value": v / 1e9, "unit": UNIT, "evaluated_per_s": vev, "cores": cores, "kind": "oracle", "sample": sample}
            per_config.append(summarise(cid, wc, args.scale, rc, tms, rec, ksteps, peaks, clock_mhz, ec, cc))
            del rc
            torch.cuda.empty_cache()
        if args.scale == 1.0:
            per_config.append(density_grid_entry(api, torch, hbm_peak(), peaks, clock_mhz))
            per_config.append(paper_table2_entry(api, torch))

    cfg = {"workload": describe(head_id, w, args.scale), "scale": args.scale,
           "l2": "256 MiB buffer written between timed iterations (L2 flush)",
           "parallelism": f"work items sharded over {world} GPU(s), catalogues replicated, grids broadcast from rank 0, one all-reduce of the histogram"}
    out = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
           "dtype": "f32", "data": "synthetic", "config": cfg, "clocks": clocks, "gpu_launches": int(launches), "e2e": e2e,
           "value_is": VALUE_IS}
    if head is not None:
        out["roofline"] = dict(head["roofline"], peak_source=peaks["source"], clock_mhz_used=clock_mhz)
        out["build"] = head["build"]
        out["rates"] = head["rates"]
        out["counts"] = head["counts"]
        if cpu is not None:
            out["cpu_baseline"] = cpu
        out["per_config"] = per_config
    out["peaks"] = {k: peaks[k] for k in ("lane_instr_per_clk_sm", "fp32_lane_ops_per_clk_sm", "mufu_per_clk_sm", "atoms_per_clk_sm", "source")}
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=HEADLINE, help="headline BASELINE.json config 1..5 (default 5: the largest single-GPU one)")
    ap.add_argument("--scale", type=float, default=1.0, help="shrink the catalogues (debugging only; 1.0 = the named configs)")
    ap.add_argument("--only", action="store_true", help="measure the headline config only (no per_config sweep)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--n4-only", action="store_true", help="run only the density-grid monopole entry (SURVEY 8(f) N4) and print it")
    ap.add_argument("--grid", default="default", choices=["default", "none", "sphere", "box3d"],
                    help="override the headline workload's neighbour search (default: the one BASELINE.json names)")
    ap.add_argument("--pix", type=float, default=0.1, help="--grid sphere: pixel side in units of theta_max")
    args = ap.parse_args()
    if args.impl == "reference":
        w = workload_for(args.config, args.scale, args)
        cfg = {"workload": describe(args.config, w, args.scale), "scale": args.scale,
               "parallelism": "oracle on the host cores (rank 0 only)"}
        run_reference(args, w, cfg)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
