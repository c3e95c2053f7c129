#!/usr/bin/env python
"""bench.py -- throughput of the CuBA hot path on B200 (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl cuba|reference]

A "step" is one pass of the whole hot path (S1-S5: stream, reflect, bin, pair, collide)
over the full particle store of BASELINE.json:configs[C] (default C = 2, the ~25M-particle
Riemann problem north_star's target is quoted on).  `value` = particle-updates/s =
N * K / t with the state resident in HBM; t from CUDA events on the launching stream,
max over ranks.  The state (1.3 GB per copy) is far larger than the 126 MB L2, so no
flush is needed between steps.  N > 1 GPUs run N independent replicas (different seeds),
no collective on the data path ("replicas only", scaling "weak").

`--impl reference` times the CPU oracle, as it stands, on the same inputs (the configuration
itself, every particle) for as many of the K steps as fit into about a minute of one host
core; --quick (and the 54M / 100M-particle variants) use a transverse slice of the box instead.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "particle_updates_per_s"
UNIT = "particle-updates/s"

# algorithmic HBM bytes per particle-step of each kernel
BYTES_STREAM_HIST = 48      # reads x,y,z,px,py,pz
BYTES_SCATTER = 104         # reads 6 fp64 + pid, writes 6 fp64 + pid
BYTES_COLLIDE = 52          # reads px,py,pz,pid, writes px,py,pz (cells with n >= 2)
BYTES_COLLIDE_FUSED = 76    # + reads x,y,z: the kernel also does S1-S3 + histogram of the next step (no k_stream_hist pass)
BYTES_STEP = BYTES_STREAM_HIST + BYTES_SCATTER + BYTES_COLLIDE   # 204: the method as specified
BYTES_STEP_FUSED = BYTES_SCATTER + BYTES_COLLIDE_FUSED           # 180: what the fused schedule actually has to move


# ncu evidence: the raw per-launch metric export of one step under profiles/ (written by the command named in
# the .md beside it), keyed by a hash of the kernel sources so that a stale capture reads as null, never as a
# number.  Metrics: dram__bytes_read.sum, dram__bytes_write.sum, smsp__inst_executed.sum,
# sm__inst_executed_pipe_fp64.sum (warp-level), gpu__time_duration.sum, launch__registers_per_thread,
# sm__warps_active.avg.pct_of_peak_sustained_active.
NCU_EXPORT = os.path.join(ROOT, "profiles", "r03_ncu_step_c%d.csv")
ISSUE_SLOTS_PER_CLOCK = 148 * 4


def kernel_source_hash():
    """sha256 over the CUDA sources of the library (csrc/*.cu, *.cuh, sorted by name)."""
    import glob
    import hashlib
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_1208_0961_b200", "csrc", "*.cu*"))):
        h.update(os.path.basename(f).encode())
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def ncu_export(config):
    """{kernel base name: {metric: summed value over the launches of ONE step}} from the tracked export, or
    (None, why).  The first line of the file is '# source_sha256: <hash> ...'."""
    path = NCU_EXPORT % config
    if not os.path.exists(path):
        return None, "no tracked ncu export for this config"
    import csv
    with open(path) as f:
        lines = f.read().splitlines()
    head = [l for l in lines if l.startswith("#")]
    sha = next((l.split("source_sha256:")[1].split()[0] for l in head if "source_sha256:" in l), None)
    if sha != kernel_source_hash():
        return None, "stale: kernel sources changed since %s was captured" % os.path.relpath(path, ROOT)
    rows = list(csv.DictReader([l for l in lines if l.startswith('"')]))
    # the export lists every launch of a short run; ONE step = the last launch of every distinct kernel
    # instantiation (the size classes of k_collide are distinct instantiations)
    last_id = {}
    for r in rows:
        last_id[r["Kernel Name"]] = r["ID"]
    out = {}
    for r in rows:
        if last_id[r["Kernel Name"]] != r["ID"]:
            continue
        name = r["Kernel Name"].replace("void ", "").replace("cuba::", "")
        base = name.split("<")[0].split("(")[0]
        try:
            v = float(r["Metric Value"].replace(",", ""))
        except ValueError:
            continue
        unit = r["Metric Unit"]
        scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0, "ms": 1e6, "us": 1e3, "ns": 1.0, "s": 1e9}.get(unit, 1.0)
        d = out.setdefault(base, {})
        m = r["Metric Name"]
        if m in ("launch__registers_per_thread", "sm__warps_active.avg.pct_of_peak_sustained_active"):
            d[m] = max(d.get(m, 0.0), v)
        else:
            d[m] = d.get(m, 0.0) + v * scale
    return out, os.path.relpath(path, ROOT)


def import_ncu(raw_csv, config):
    """`python bench.py --import-ncu <ncu --csv log> --config C`: writes the tracked export profiles/r03_ncu_step_cC.csv:
    the rows of the LAST launch of every kernel instantiation (one step), headed by the hash of the kernel
    sources they were measured on."""
    import csv
    with open(raw_csv) as f:
        lines = [l for l in f.read().splitlines() if l.startswith('"')]
    rows = list(csv.DictReader(lines))
    last_id = {}
    for r in rows:
        last_id[r["Kernel Name"]] = r["ID"]
    keep = [lines[0]] + [l for l, r in zip(lines[1:], rows) if last_id[r["Kernel Name"]] == r["ID"]]
    path = NCU_EXPORT % config
    with open(path, "w") as f:
        f.write("# source_sha256: %s  (csrc/*.cu, *.cuh this export was measured on; bench.py reports null once they change)\n"
                % kernel_source_hash())
        f.write("\n".join(keep) + "\n")
    print("wrote %s: %d rows of %d kernel instantiations" % (os.path.relpath(path, ROOT), len(keep) - 1, len(last_id)))


def issue_roofline(warp_inst, ms, clocks, source):
    """Secondary roofline of an issue-bound kernel: warp instructions per launch (tracked ncu export) / measured
    duration against 592 issue slots x the SM clock sampled during the run."""
    mhz = (clocks or {}).get("sm_mhz") or (clocks or {}).get("sm_max_mhz")
    if not warp_inst or not ms or not mhz:
        return None
    achieved = warp_inst / (ms * 1e-3) / 1e9
    peak = ISSUE_SLOTS_PER_CLOCK * mhz * 1e6 / 1e9
    return {"bound": "issue", "achieved": achieved, "peak": peak, "unit": "G warp-inst/s", "frac": achieved / peak,
            "source": "smsp__inst_executed.sum from %s / CUDA-event duration of this run" % source}


def fp64_roofline(fp64_warp_inst, ms, peak_dfma_per_s, source):
    """fp64 leg (BASELINE.json: 'fp64 pipe utilisation against the chip's fp64 peak'): fp64-pipe warp
    instructions per launch (tracked ncu export) / measured duration against the DFMA rate measured by
    cuba_probe_fp64 in this run (thread-level rate / 32)."""
    if not fp64_warp_inst or not ms or not peak_dfma_per_s:
        return None
    achieved = fp64_warp_inst / (ms * 1e-3) / 1e9
    peak = peak_dfma_per_s / 32.0 / 1e9
    return {"bound": "fp64", "achieved": achieved, "peak": peak, "unit": "G fp64 warp-inst/s", "frac": achieved / peak,
            "peak_tflops": 2.0 * peak_dfma_per_s / 1e12,
            "source": "sm__inst_executed_pipe_fp64.sum from %s / CUDA-event duration; peak = cuba_probe_fp64 (this run)" % source}


def peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML every 10 ms while armed."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.armed, self.stop_flag = index, [], False, False
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag:
            if self.armed:
                try:
                    mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                    reasons = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(
                        nv, "nvmlDeviceGetCurrentClocksEventReasons") else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                    self.samples.append((mhz, int(reasons)))
                except Exception:
                    pass
            time.sleep(0.01)

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": getattr(self, "max_mhz", None), "reasons": ["unsampled"]}
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        bits = 0
        for _, r in self.samples:
            bits |= r
        reasons = [n for b, n in names.items() if bits & b and n != "gpu_idle"]
        return {"sm_mhz": float(np.median([m for m, _ in self.samples])), "sm_max_mhz": float(self.max_mhz),
                "reasons": reasons, "samples": len(self.samples)}


def oracle_sample_workload(config, quick=False, w_full=None):
    """(workload, description, same_inputs) the CPU oracle is timed on.  Default: configs[config] ITSELF, every
    particle (the same inputs, fewer steps) -- the bounded sample is then a few steps of it.  Only the
    ~54M / ~100M-particle configs[4] variants, and --quick, fall back to a transverse slice of the box (same
    densities, cell size, dt and sigma, a quarter of the extent in y and z)."""
    if not quick and config in (0, 1, 2, 3):
        w = w_full if w_full is not None else workloads.make(config)
        return w, "configs[%d] itself, all %d particles" % (config, w.n), True
    if config in (1, 2):
        r = 10.0 if config == 1 else 100.0
        w = workloads.riemann(L=(32.0, 8.0, 8.0), ncell=(32, 8, 8), r_test=r, seed=config + 1)
        return w, "configs[%d] restricted to a 32x8x8 fm^3 transverse slice (same T, r_test, cells, dt, sigma)" % config, False
    if config == 3:
        w = workloads.riemann(L=(32.0, 8.0, 8.0), ncell=(64, 8, 8), r_test=40.0, sigma_gev2=50.0, dt=0.05, seed=4)
        return w, "configs[3] restricted to a 32x8x8 fm^3 transverse slice", False
    if config in (4, 5):
        w = workloads.skewed(L=(64.0, 8.0, 8.0), ncell=(64, 8, 8), r_test=100.0 if config == 4 else 185.5, seed=5)
        return w, "configs[4] restricted to a 64x8x8 fm^3 transverse slice", False
    w = workloads.make(0)
    return w, "configs[0] whole", True


def oracle_step_budget(n, steps, warmup, seconds):
    """(timed steps, warm-up steps) of the oracle that fit into about `seconds` of one host core, assuming the
    ~2.5 M particle-updates/s it reaches on stores far larger than the caches; never more than asked for."""
    per_step = max(n, 1) / 2.5e6
    timed = max(2, min(steps, int(seconds / per_step)))
    return timed, (min(warmup, 1) if timed < steps else warmup)


def time_oracle(w, steps, warmup):
    import oracle
    o = oracle.Oracle.from_workload(w)
    if warmup:
        o.step(warmup, w.dt, w.sigma)
    t0 = time.perf_counter()
    o.step(steps, w.dt, w.sigma)
    dt = time.perf_counter() - t0
    c = o.counters()
    o.close()
    return dt, c


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle as it stands, host cores, rank 0 only."""
    if rank != 0:
        return
    w, sample, same = oracle_sample_workload(args.config, args.quick)
    steps, warmup = oracle_step_budget(w.n, args.steps, args.warmup, 60.0)
    dt, c = time_oracle(w, steps, warmup)
    value = w.n * steps / dt
    full = workloads_name(args.config)
    sample = "%s, %d timed steps after %d warm-up (asked: %d / %d), %.1f s" % (sample, steps, warmup, args.steps, args.warmup, dt)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "steps_timed": steps, "warmup_run": warmup, "ms_per_step": 1e3 * dt / steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": full, "sample": sample, "n_particles": w.n, "same_inputs": same},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def short_run(cuba, torch, dev, config, steps, warmup):
    """One short device-timed run of another configuration (no repeats, no per-kernel pass): W warm-up steps,
    then K steps between CUDA events on the launching stream, state resident in HBM (far larger than L2)."""
    w = workloads.CONFIGS[config]()
    sim = cuba.Cuba.from_workload(w, device=dev)
    sim.step(warmup, w.dt, w.sigma)
    torch.cuda.synchronize()
    c0 = sim.counters()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    sim.step(steps, w.dt, w.sigma)
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1)
    c1 = sim.counters()
    if c1.device_flags:
        raise SystemExit("device error flags %d in configs[%d]" % (c1.device_flags, config))
    out = {"workload": workloads_name(config), "n_particles": w.n, "steps": steps, "warmup": warmup,
           "ms_per_step": ms / steps, "value": w.n * steps / (ms * 1e-3), "unit": UNIT,
           "pair_evals_per_s": (c1.pairs - c0.pairs) / (ms * 1e-3), "max_occupancy": c1.max_occupancy,
           "overflow_cells": c1.overflow_cells}
    sim.close()
    del sim
    torch.cuda.empty_cache()
    return out


def run_two_stream_probe(args):
    """--two-stream-probe (diagnostic): how much do the kernels of two independent problems overlap on one GPU?
    Two half-size copies of configs[2] (32x32x16 fm^3 each: the same cell populations, half the cells) are stepped
    K times (a) one after the other and (b) on two streams with their step(1) calls interleaved; wall clock
    between device synchronisations.  A proxy for running the scatter of some cell layers under the collisions of
    others (round 3); no bench value."""
    import torch
    import paper_1208_0961_b200 as cuba
    dev = torch.device("cuda", 0)
    K = args.steps
    ws = [workloads.riemann(L=(32.0, 32.0, 16.0), ncell=(32, 32, 16), r_test=100.0, seed=s) for s in (3, 4)]
    streams = [torch.cuda.Stream(device=dev) for _ in ws]
    ctx = []
    for w, st in zip(ws, streams):
        with torch.cuda.stream(st):
            ctx.append(cuba.Cuba.from_workload(w, device=dev, stream=st))
    for c, w in zip(ctx, ws):
        c.step(max(args.warmup, 3), w.dt, w.sigma)

    def timed(fn):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        fn()
        torch.cuda.synchronize()
        return 1e3 * (time.perf_counter() - t0)

    def one_after_the_other():
        for c, w in zip(ctx, ws):
            c.step(K, w.dt, w.sigma)
            torch.cuda.synchronize()

    def interleaved():
        for _ in range(K):
            for c, w in zip(ctx, ws):
                c.step(1, w.dt, w.sigma)

    seq = [timed(one_after_the_other) for _ in range(2)]
    con = [timed(interleaved) for _ in range(2)]
    line = {"probe": "two half-size copies of configs[2] on two streams", "n_particles_each": ws[0].n, "steps": K,
            "sequential_ms_per_step_of_both": min(seq) / K, "interleaved_ms_per_step_of_both": min(con) / K,
            "gain": 1.0 - min(con) / min(seq), "lib": cuba.lib_path(),
            "grid_c4_knob": os.environ.get("CUBA_DEBUG_GRID_C4"), "note": "diagnostic, not a bench value"}
    for c in ctx:
        if c.counters().device_flags:
            raise SystemExit("device error flags")
        c.close()
    print(json.dumps(line), flush=True)


def reduce_over_ranks(dist, device, ms, e2e_s, n, pairs, launches):
    """Whole-job aggregation for N independent replicas: the time is the MAX over ranks, the
    work (particles, pair evaluations, launches) the SUM.  `dist` is torch.distributed or None."""
    if dist is None:
        return ms, e2e_s, float(n), float(pairs), int(launches)
    import torch
    t = torch.tensor([ms, e2e_s], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    s = torch.tensor([float(n), float(pairs), float(launches)], device=device, dtype=torch.float64)
    dist.all_reduce(s, op=dist.ReduceOp.SUM)
    return float(t[0]), float(t[1]), float(s[0]), float(s[1]), int(s[2])


def workloads_name(config):
    return {0: "configs[0] thermal box 8^3 fm^3, r_test=2 (13.8k particles)",
            1: "configs[1] Riemann 32^3 fm^3, r_test=10 (2.49M particles)",
            2: "configs[2] Riemann 32^3 fm^3, T=0.4/0.2 GeV, r_test=100 (24.9M particles), sigma=10 GeV^-2, dt=0.1 fm/c",
            3: "configs[3] Riemann fine cells 0.5x1x1 fm, r_test=40 (9.96M particles), sigma=50 GeV^-2, dt=0.05",
            4: "configs[4] skewed occupancy 64x32x32 fm^3, r_test=100 (53.9M particles)",
            5: "configs[4] at ~100M particles: skewed occupancy 64x32x32 fm^3, r_test=185.5 (100.0M particles)"}[config]


def run_slab(args, rank, world, local):
    """--decomp slab: ONE problem (configs[C]) sharded by x-layers of cells over the ranks (strong scaling), halo
    exchange by torch.distributed point-to-point after every step (paper_1208_0961_b200/slab.py).  With
    --slab-emulate R on one GPU the R ranks' contexts are stepped one after the other in one process: the
    per-rank device times project the step of an R-GPU run (max over ranks; transfers not included)."""
    import torch
    import torch.distributed as dist
    import paper_1208_0961_b200 as cuba
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    w = workloads.CONFIGS[args.config]()
    emul = args.slab_emulate
    if emul:
        grp = cuba.LocalSlabGroup(w, emul, device=dev, balance=True)
        grp.step(args.warmup, w.dt, w.sigma)
        per_rank = [0.0] * emul
        evs = [[torch.cuda.Event(enable_timing=True) for _ in range(6)] for _ in range(emul)]
        torch.cuda.synchronize()
        for _ in range(args.steps):
            for k, r in enumerate(grp.ranks):
                evs[k][0].record(); r.step(1, w.dt, w.sigma); evs[k][1].record()
            sent = []
            for k, r in enumerate(grp.ranks):
                lo, hi = cuba.neighbours(k, emul)
                evs[k][2].record()
                sent.append((r.pack(0) if lo is not None else None, r.pack(1) if hi is not None else None))
                evs[k][3].record()
            for k, r in enumerate(grp.ranks):
                lo, hi = cuba.neighbours(k, emul)
                evs[k][4].record()
                r.unpack(sent[lo][1] if lo is not None else None, sent[hi][0] if hi is not None else None)
                evs[k][5].record()
            torch.cuda.synchronize()
            for k in range(emul):
                per_rank[k] += sum(evs[k][2 * q].elapsed_time(evs[k][2 * q + 1]) for q in range(3))
        ms = max(per_rank) / args.steps
        halo = [sum(r.count(s) for s in (0, 1) if cuba.neighbours(k, emul)[s] is not None) for k, r in enumerate(grp.ranks)]
        print(json.dumps({"metric": METRIC, "unit": UNIT, "value": w.n / (ms * 1e-3), "n_gpus": 1, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "dtype": "f64",
                          "data": "synthetic", "vs_baseline": None,
                          "config": {"workload": workloads_name(args.config), "decomposition": "x-slabs of whole cell layers, cuts balanced by particles per layer",
                                     "emulated_ranks": emul, "layers": grp.layers,
                                     "note": "PROJECTION: %d ranks stepped one after the other on ONE GPU; ms_per_step = slowest rank's "
                                             "device time (step + pack + unpack), NVLink transfers not included" % emul},
                          "per_rank_ms": [round(v / args.steps, 4) for v in per_rank],
                          "halo_particles_sent_per_rank": halo, "halo_bytes_sent_per_rank": [52 * h for h in halo]}), flush=True)
        return
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)
    lo, hi = cuba.slab_layers(int(w.ncell[0]), world, cuba.layer_weights(w.x, float(w.box[0]), int(w.ncell[0])))[rank]
    ctx = cuba.SlabRank(w, lo, hi, device=dev)
    for _ in range(args.warmup):
        cuba.slab_step(ctx, dist, rank, world, w.dt, w.sigma)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    for _ in range(args.steps):
        cuba.slab_step(ctx, dist, rank, world, w.dt, w.sigma)
    ev1.record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    t = torch.tensor([ev0.elapsed_time(ev1)], device=dev, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t[0]) / args.steps
    if rank == 0:
        print(json.dumps({"metric": METRIC, "unit": UNIT, "value": w.n / (ms * 1e-3), "n_gpus": world, "steps": args.steps,
                          "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "strong", "dtype": "f64",
                          "data": "synthetic", "vs_baseline": None,
                          "config": {"workload": workloads_name(args.config), "decomposition": "x-slabs of whole cell layers",
                                     "parallelism": "slab x%d, halo exchange by NCCL point-to-point" % world}}), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="index into BASELINE.json:configs")
    ap.add_argument("--impl", default="cuba", choices=["cuba", "reference"])
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: independent replicas (default, weak scaling) or ONE problem in x-slabs (strong scaling)")
    ap.add_argument("--slab-emulate", type=int, default=0, help="diagnostic: R slab ranks stepped in turn on one GPU (projection)")
    ap.add_argument("--two-stream-probe", action="store_true",
                    help="diagnostic: two half-size copies of configs[2] stepped one after the other vs interleaved on two streams")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--quick", action="store_true", help="time the oracle on a transverse slice of the box instead of the configuration itself")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-other-configs", dest="other_configs", action="store_false",
                    help="skip the short runs of configs[3] and configs[4] that the default line carries under other_configs")
    ap.add_argument("--no-fuse", action="store_true", help="run the separate k_stream_hist pass every step (A/B diagnostic)")
    ap.add_argument("--slots", type=int, default=-1, help="CUBA_OPT_SLOTS: 0 compact schedule, 1/2 slotted schedule; -1 library default (A/B diagnostic)")
    ap.add_argument("--import-ncu", default=None, help="ncu --csv log of a short bench run: write the tracked export under profiles/ and exit")
    ap.add_argument("--repeats", type=int, default=3, help="timed repeats of K steps each; the line reports the median")
    ap.add_argument("--profile-mode", type=int, default=1, help="1: normal operation; 2: serialise the collision classes (diagnostic)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "cuba" else args.warmup
    if args.import_ncu:
        import_ncu(args.import_ncu, args.config)
        return

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
        return
    if args.two_stream_probe:
        if rank == 0:
            run_two_stream_probe(args)
        return
    if args.decomp == "slab" or args.slab_emulate:
        run_slab(args, rank, world, local)
        return

    import torch
    import torch.distributed as dist
    import paper_1208_0961_b200 as cuba

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    cuba.lib()
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- workload: replica `rank` of configs[C] (independent seed per rank) -------------
    w = workloads.CONFIGS[args.config]()
    if rank:
        w.seed = w.seed + 1000 * rank
    host = [torch.from_numpy(a).pin_memory() for a in w.arrays()]
    n = w.n
    fused = not args.no_fuse
    bytes_collide = BYTES_COLLIDE_FUSED if fused else BYTES_COLLIDE

    def fresh():
        """A context on a fresh device copy of the initial state, warmed up: every repeat (and the per-kernel
        pass) times the SAME steps W..W+K of the run -- the cost of a step drifts as the Riemann profile evolves
        (fewer cells need a second round), so consecutive blocks of K steps are not repeats of one another."""
        sm = cuba.Cuba(w.box, w.ncell, *[h.to(dev) for h in host], w.n_test, w.seed)
        sm.set_option(1, 1 if fused else 0)
        if args.slots >= 0:
            sm.set_option(3, args.slots)
        sm.step(args.warmup, w.dt, w.sigma)
        return sm

    sampler = ClockSampler(local)
    sampler.start()

    # ---- W warm-up steps, then the timed region: K steps, CUDA events on the launching stream, profiling OFF
    # (the configuration a user runs); repeated from the same initial state, the line reports the median ----
    reps, pairs, launches = [], 0, 0
    for _ in range(args.repeats):
        sim = fresh()
        barrier()
        c0 = sim.counters()
        l0 = cuba.launch_count()
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        sampler.armed = True
        ev0.record()
        sim.step(args.steps, w.dt, w.sigma)
        ev1.record()
        barrier()
        sampler.armed = False
        reps.append(ev0.elapsed_time(ev1))
        launches = cuba.launch_count() - l0
        c1 = sim.counters()
        pairs = c1.pairs - c0.pairs
        if c1.device_flags:
            raise SystemExit("device error flags %d" % c1.device_flags)
        sim.close()
        del sim
    ms = float(np.median(reps))

    # ---- per-kernel split: a separate pass over the same K steps with a CUDA event after every launch ----
    sim = fresh()
    barrier()
    sim.profile_enable(args.profile_mode)
    sim.step(args.steps, w.dt, w.sigma)
    prof = sim.profile_read()
    sim.profile_enable(0)
    prof_ms = sum(v[0] for k, v in prof.items() if "(all classes" in k or not k.startswith("k_collide<"))
    fp64_peak = cuba.probe_fp64(sim._stream.cuda_stream, 5) if rank == 0 else 0.0

    # particles each collide class handled in the last step (for per-launch algorithmic bytes)
    import re
    counts = np.diff(sim.cell_start().astype(np.int64))
    collide_names = [k for k in prof if k.startswith("k_collide<") or k == "k_collide_overflow"]
    caps = [int(re.search(r"cap=(\d+)", k).group(1)) for k in collide_names if "cap=" in k]
    cls = np.searchsorted(caps, counts, side="left")
    class_particles = {name: int(counts[(cls == k) & (counts >= (1 if fused else 2))].sum())
                       for k, name in enumerate(collide_names)}

    # ---- observables timed separately --------------------------------------------------
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    tot, ed = sim.observables(w.nslab)
    obs_ms = 1e3 * (time.perf_counter() - t0)

    # ---- end to end through the C ABI with HOST buffers --------------------------------
    e2e = None
    if not args.no_e2e:
        e2e_steps = args.steps
        harr = [h.numpy() for h in host]
        barrier()
        t0 = time.perf_counter()
        cuba.run_host(w.box, w.ncell, *harr, w.n_test, w.seed, e2e_steps, w.dt, w.sigma, w.nslab)   # cold: the library's pool maps its memory
        torch.cuda.synchronize()
        cold_s = time.perf_counter() - t0
        barrier()
        t0 = time.perf_counter()
        cuba.run_host(w.box, w.ncell, *harr, w.n_test, w.seed, e2e_steps, w.dt, w.sigma, w.nslab)
        torch.cuda.synchronize()
        e2e_s = time.perf_counter() - t0
        e2e = {"s": e2e_s, "steps": e2e_steps, "cold_s": cold_s}
    ncells_main = sim.ncells
    sim.close()
    del sim
    torch.cuda.empty_cache()

    # ---- the other large configurations, short runs (the driver's record should carry them too) ----
    others = {}
    if args.other_configs and world == 1 and args.config == 2:
        for oc in (3, 4):
            others["configs[%d]" % oc] = short_run(cuba, torch, dev, oc, 10, 3)

    # ---- reduce over ranks: max time, summed work --------------------------------------
    ms, e2e_s, n_total, pairs_total, launches = reduce_over_ranks(
        dist if world > 1 else None, dev, ms, e2e["s"] if e2e else 0.0, n, pairs, launches)
    if e2e:
        e2e["s"] = e2e_s
    sampler.stop_flag = True

    if rank == 0:
        peak, peak_src = peaks()
        sec = ms * 1e-3
        value = n_total * args.steps / sec
        # dominant kernel by measured device time
        per_kernel = {k: {"ms_per_launch": (v[0] / v[1]) if v[1] else 0.0, "launches": v[1], "ms_total": v[0]}
                      for k, v in prof.items()}
        alg = {"k_stream_hist": BYTES_STREAM_HIST * n, "k_scatter": BYTES_SCATTER * n}
        alg.update({name: bytes_collide * cnt for name, cnt in class_particles.items()})
        alg["k_collide (all classes, concurrent)"] = bytes_collide * sum(class_particles.values())
        groups = {k: v for k, v in per_kernel.items() if not k.startswith("k_collide<") or args.profile_mode == 2}
        dom = max(groups, key=lambda k: groups[k]["ms_total"])
        dom_ms = per_kernel[dom]["ms_per_launch"]
        achieved = alg.get(dom, 0) / (dom_ms * 1e-3) / 1e9 if dom_ms else 0.0
        kernels = {}
        for k, v in per_kernel.items():
            if v["launches"]:
                gbs = alg.get(k, 0) / (v["ms_per_launch"] * 1e-3) / 1e9 if v["ms_per_launch"] else 0.0
                kernels[k] = {"ms_per_launch": round(v["ms_per_launch"], 5), "share": round(v["ms_total"] / prof_ms, 4) if prof_ms else None,
                              "alg_GBps": round(gbs, 1), "frac": round(gbs / peak, 4)}
        # ncu-derived figures of the dominant kernel group, from the tracked export of one step
        ncu, ncu_src = ncu_export(args.config)
        base = "k_slot_step" if dom.startswith("k_slot_step") else ("k_collide" if dom.startswith("k_collide") else dom)
        nk = {}
        if ncu:
            for name, d in ncu.items():
                if name == base or (base == "k_collide" and name == "k_collide_overflow"):
                    for m, v in d.items():
                        nk[m] = nk.get(m, 0.0) + v if not m.startswith(("launch__", "sm__warps")) else max(nk.get(m, 0.0), v)
        traffic = (nk.get("dram__bytes_read.sum", 0.0) + nk.get("dram__bytes_write.sum", 0.0)) or None
        clk = sampler.summary()
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "repeats": {"n": args.repeats, "ms_per_step": [round(r / args.steps, 5) for r in reps],
                        "median": ms / args.steps, "best": min(reps) / args.steps,
                        "note": "every repeat times steps W..W+K from the same initial state (the step cost drifts as the profile evolves); "
                                "value and ms_per_step are the median repeat; profiling off in the timed region"},
            "config": {"workload": workloads_name(args.config), "n_particles": n, "ncells": ncells_main,
                       "l2": "inputs larger than L2 (%.2f GB state per copy vs 126 MB L2), no flush" % (52 * n / 1e9)
                       if 52 * n > 4 * 126e6 else "state comparable to L2: cache-resident, not a roofline config",
                       "parallelism": "replicas x%d" % world if world > 1 else "single GPU",
                       "schedule": ("fused: collide(t) also writes the histogram of step t+1 (CUBA_OPT_FUSE_HIST=1)"
                                    if fused else "separate k_stream_hist pass (CUBA_OPT_FUSE_HIST=0)") +
                                   ("; CUBA_OPT_SLOTS=%d" % args.slots if args.slots >= 0 else "; CUBA_OPT_SLOTS default")},
            "pair_evals_per_s": pairs_total / sec,
            "pairs_per_step": pairs_total / args.steps,
            "observables_ms": obs_ms,
            "gpu_launches": int(launches),
            "clocks": clk,
            "roofline": {"bound": "hbm", "kernel": dom, "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                         "alg_bytes_per_launch": alg.get(dom, 0),
                         "duration_source": "CUDA events after every launch in a separate pass of %d steps (cuba_profile_enable)" % args.steps,
                         "ncu_source": ncu_src,
                         "ncu": {k: nk.get(k) for k in ("smsp__inst_executed.sum", "sm__inst_executed_pipe_fp64.sum",
                                                         "launch__registers_per_thread",
                                                         "sm__warps_active.avg.pct_of_peak_sustained_active")} if nk else None,
                         "issue": issue_roofline(nk.get("smsp__inst_executed.sum"), dom_ms, clk, ncu_src),
                         "fp64": fp64_roofline(nk.get("sm__inst_executed_pipe_fp64.sum"), dom_ms, fp64_peak, ncu_src),
                         "fp64_peak_measured": {"dfma_per_s": fp64_peak, "tflops": 2.0 * fp64_peak / 1e12,
                                                "source": "cuba_probe_fp64: 8 dependent DFMA chains per thread, 8 CTAs x 256 threads per SM, best of 5"},
                         "step": {"alg_bytes_per_particle": BYTES_STEP,
                                  "moved_bytes_per_particle": BYTES_STEP_FUSED if fused else BYTES_STEP,
                                  "achieved": BYTES_STEP * value / world / 1e9,
                                  "frac": BYTES_STEP * value / world / 1e9 / peak,
                                  "frac_moved_bytes": (BYTES_STEP_FUSED if fused else BYTES_STEP) * value / world / 1e9 / peak,
                                  "frac_of_8TBps_nominal": BYTES_STEP * value / world / 8e12,
                                  "note": "frac uses the model's 204 B per particle-step (SURVEY 8(d): the method as specified); "
                                          "frac_moved_bytes what the fused schedule really has to move"},
                         "kernels": kernels},
        }
        if e2e:
            line["e2e"] = {"value": n_total * e2e["steps"] / e2e["s"], "unit": UNIT,
                           "h2d_bytes_per_step": 48 * n / e2e["steps"], "d2h_bytes_per_step": 8 * (4 + w.nslab) / e2e["steps"],
                           "call": "cuba_run_host: pinned HOST arrays -> H2D -> cuba_init -> cuba_step(%d) -> cuba_observables -> D2H of "
                                   "the observables only (4 + nslab doubles: north_star's result; the particle store is not copied back)"
                                   % e2e["steps"], "seconds": e2e["s"],
                           "cold_value": n_total * e2e["steps"] / e2e["cold_s"], "cold_seconds": e2e["cold_s"],
                           "note": "value: second call (the library's memory pool already mapped); cold_value: first call of the process"}
        if not args.no_cpu_baseline:
            ow, sample, same = oracle_sample_workload(args.config, args.quick, w_full=w)
            osteps = max(2, min(60, int(40e6 // max(ow.n, 1)) + 1))   # about 10-30 s of one host core
            odt, oc = time_oracle(ow, osteps, 0)
            line["cpu_baseline"] = {"value": ow.n * osteps / odt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": "%s, N=%d, %d steps, %.1f s" % (sample, ow.n, osteps, odt),
                                    "same_inputs": same, "host_cores_available": os.cpu_count()}
        if others:
            pk = peak
            for v in others.values():
                v["roofline_step_frac"] = BYTES_STEP * v["value"] / 1e9 / pk
                v["roofline_step_frac_moved_bytes"] = BYTES_STEP_FUSED * v["value"] / 1e9 / pk
            line["other_configs"] = others
        line["paper_context"] = ("CuBA 58.09 s vs BAMPS 756 s (~13x), GPU and CPU models not named in the paper "
                                 "(Fermi-era CUDA 4.1), run size not stated (PAPER.md:92)")
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
