#!/usr/bin/env python
"""bench.py -- far-field Stokeslet GInteractions/s on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 0..4] [--precision f32|f64]
    python bench.py --impl reference ...        # the oracle, as it stands, on the host cores
    python bench.py --path masked|targets|aux|fmm [--order P] ...   # the NEXT rows, same JSON line

A *step* is one pass of the whole hot path (DESIGN.md rows a-1..a-5: arclength weights, packing,
pair sum, reduction, scaling) over one batch of synthetic input.  The default workload is
BASELINE.json configs[4] (8,000 vesicles x 128 points, fp32): a step is its ten consecutive
evaluations with perturbed positions, reusing the device buffers on one stream.  For workloads
0-3 a step is one evaluation.  `value` counts P*(P-npts) interactions per evaluation (own-vesicle
pairs are not counted) over device time (CUDA events, inputs resident in HBM, max over ranks);
`e2e` is the same work through vn_farfield_host with pinned HOST buffers (copies inside the
timed region).

--gpus N > 1 (one process per GPU, torchrun): the SAME suspension is evaluated by all ranks together
(DESIGN.md section 8): every rank owns a contiguous range of vesicles, one all-gather makes all
sources known everywhere, rank r runs blocks r, r+N, ... of the pair walk (vn_farfield_partial), one
integer reduce-scatter sums the fixed-point accumulators, vn_farfield_finish rounds the rank's shard.
Total work is fixed: "scaling": "strong".  The result is bit for bit the single-GPU result.

The default invocation (N = 1, configs[4], fp32) also measures, in the same run, the issue rates of
the FP32 / SFU / FP64 pipes (vn_pipe_peaks -> roofline.peak_measured), a `sweep` over the other
configurations north_star's target names (configs[3] fp32 and fp64, configs[1] fp32), and `next_rows`: the fast
multipole evaluation of the same sum (row f-4b) at configs[4] and configs[3].

One JSON line is printed by rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time
from types import SimpleNamespace

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "far-field Stokeslet GInteractions/s"
UNIT = "GInt/s"
# canonical per-pair work: 2 FADD + 3 FMUL + 6 FFMA = 11 FP32-pipe
# lane-instructions (17 flop) + 2 SFU ops; fp64: the same 11 DP instructions (17 flop).
LANE_OPS_PER_PAIR = 11
FLOP_PER_PAIR = 17
# what the kernels execute per directed interaction (symmetric evaluation; SASS counts)
EXECUTED_LANE_OPS = {("farfield", "f32"): 9.0, ("masked", "f32"): 9.0, ("farfield", "f64"): 12.85, ("masked", "f64"): 12.85,
                     ("targets", "f32"): 13.0, ("targets", "f64"): 19.0}
SMS, FP32_LANES, FP64_LANES = 148, 128, 64


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            return json.load(fh)
    except Exception:
        return {}


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons during the timed region (NVML)."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.stop_flag = index, threading.Event()
        self.sm, self.reasons, self.max_mhz, self.power = [], set(), None, []

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.max_mhz = nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)
            names = {nv.nvmlClocksThrottleReasonHwSlowdown: "hw_slowdown",
                     nv.nvmlClocksThrottleReasonHwThermalSlowdown: "hw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwThermalSlowdown: "sw_thermal_slowdown",
                     nv.nvmlClocksThrottleReasonSwPowerCap: "sw_power_cap",
                     nv.nvmlClocksThrottleReasonHwPowerBrakeSlowdown: "hw_power_brake"}
            while not self.stop_flag.is_set():
                self.sm.append(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM))
                try:
                    self.power.append(nv.nvmlDeviceGetPowerUsage(h) / 1000.0)
                except Exception:
                    pass
                mask = nv.nvmlDeviceGetCurrentClocksThrottleReasons(h)
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
                time.sleep(0.05)
        except Exception as exc:                      # no NVML: report that, do not fail the bench
            self.reasons.add(f"nvml_unavailable:{type(exc).__name__}")

    def stop(self):
        self.stop_flag.set()
        self.join()
        return self.summary()

    def summary(self):
        return {"sm_mhz": statistics.median(self.sm) if self.sm else None,
                "sm_max_mhz": self.max_mhz,
                "power_w_max": max(self.power) if self.power else None,
                "reasons": sorted(self.reasons)}


def nvml_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


def target_grid(susp, n_side, np_dtype):
    """n_side x n_side velocity-field grid over the suspension's bounding box plus a margin of 1
    (row f-4).  Grid points that fall close to a membrane simply get the plain trapezoid value."""
    P = susp.X.reshape(-1, 2)
    lo, hi = P.min(0) - 1.0, P.max(0) + 1.0
    gx = np.linspace(lo[0], hi[0], n_side)
    gy = np.linspace(lo[1], hi[1], n_side)
    return np.ascontiguousarray(np.stack(np.meshgrid(gx, gy, indexing="ij"), -1).reshape(-1, 2), dtype=np_dtype)


def oracle_rate(susp, np_dtype, seconds, rng_seed, path="farfield", fast=False):
    """Times the oracle (as it stands) on a bounded random sample of targets x ALL sources of the
    same workload; returns (GInt/s, cores, description).  fast=True times oracle/baseline_f64.c instead
    (plain double, vectorised: the CPU speed baseline, farfield path only)."""
    import oracle
    X = np.asarray(susp.X, dtype=np_dtype).astype(np.float64)
    F = np.asarray(susp.F, dtype=np_dtype).astype(np.float64)
    W = oracle.weights(X)
    P = susp.nves * susp.npts
    rng = np.random.Generator(np.random.PCG64(rng_seed))
    if fast:
        oracle.build_baseline(force=True)             # -march=native: compiled on the machine that times it
        pool, per_target = P, P - susp.npts
        run = lambda idx: oracle.baseline_farfield_subset(X, F, W, idx, susp.mu)
    elif path == "targets":
        xt = target_grid(susp, 512, np_dtype).astype(np.float64)
        pool, per_target = len(xt), P
        run = lambda idx: oracle.farfield_targets(X, F, W, xt[idx], susp.mu)
    elif path == "masked":
        pool, per_target = P, P - susp.npts
        run = lambda idx: oracle.farfield_masked_subset(X, F, W, idx, oracle.near_mask_subset(X, W, idx), susp.mu)
    else:
        pool, per_target = P, P - susp.npts
        run = lambda idx: oracle.farfield_subset(X, F, W, idx, susp.mu)
    probe = rng.choice(pool, size=min(pool, 64 * oracle.num_threads()), replace=False)
    t0 = time.perf_counter()
    run(probe)
    rate = len(probe) * per_target / (time.perf_counter() - t0)
    n = int(max(len(probe), min(pool, rate * seconds / per_target)))
    idx = rng.choice(pool, size=n, replace=False)
    t0 = time.perf_counter()
    run(idx)
    dt = time.perf_counter() - t0
    return n * per_target / dt / 1e9, oracle.num_threads(), f"{n} random targets x all {P} sources ({n * per_target:.3e} pairs, {dt:.1f} s)"


def cpu_baseline(susp, np_dtype, path):
    """The reported CPU baseline: the oracle as it stands (long double, the parity checker) and, for the farfield
    path, the same sum in plain vectorised double (oracle/baseline_f64.c) -- the checker is the right code to compare
    against and the wrong code to race against, so both are stated."""
    import oracle
    v, cores, sample = oracle_rate(susp, np_dtype, 15.0, 4242, path)
    out = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
           "code": "oracle/oracle_vesnet.c (long double, gcc -O2 -ffp-contract=off -fopenmp)"}
    if path == "farfield":
        vf, _, sf = oracle_rate(susp, np_dtype, 5.0, 4243, path, fast=True)
        out["fast_double"] = {"value": vf, "unit": UNIT, "cores": cores, "sample": sf,
                              "code": "oracle/baseline_f64.c (double, %s; pinned to the oracle at 1e-13)" % oracle.baseline_flags()}
    return out


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    from paper_2606_25569_b200 import inputs
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    susp = inputs.config(args.workload)
    np_dtype = np.float32 if args.precision == "f32" else np.float64
    total = max(1, args.steps + args.warmup)
    per_step = max(2.0, min(30.0, 150.0 / total))
    rates, cores, sample = [], 0, ""
    for s in range(total):
        r, cores, sample = oracle_rate(susp, np_dtype, per_step, 7000 + s, args.path)
        if s >= args.warmup:
            rates.append(r)
    value = statistics.mean(rates)
    P = susp.nves * susp.npts
    evals = 10 if args.workload == 4 else 1
    pairs_eval = 512 * 512 * P if args.path == "targets" else susp.pairs
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": evals * pairs_eval / (value * 1e9) * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, susp, "oracle on host cores; ms_per_step extrapolated from the sampled rate"),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"per step: {sample}"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


PATHS = {"farfield": "rows a-1..a-5: vn_arclength_weights + vn_farfield",
         "fmm": "row f-4b: vn_arclength_weights + vn_farfield_fmm (fast multipole, APPROXIMATE; value = the direct sum's pair count / time)",
         "masked": "row f-1: vn_arclength_weights + vn_near_pairs + vn_farfield_masked (the paper's DirectSingleLayerIntegral)",
         "targets": "row f-4: vn_arclength_weights + vn_farfield_targets on a 512x512 grid of free targets"}


def workload_config(args, susp, note=""):
    evals = 10 if args.workload == 4 else 1
    P = susp.nves * susp.npts
    return {"workload": f"BASELINE.json configs[{args.workload}]: {susp.name}", "path": PATHS[args.path],
            "nves": susp.nves, "npts": susp.npts, "points": P,
            "pairs_per_evaluation": 512 * 512 * P if args.path == "targets" else susp.pairs,
            "evaluations_per_step": evals,
            "precision": args.precision, "l2": "flushed between timed steps (256 MiB write); inputs < L2",
            "cuda_graph": bool(getattr(args, "graph", False)),
            "parallelism": (f"one suspension over {args.gpus} GPUs: vesicle ranges per rank, all-gather of X/F/W, blocks of the pair "
                            f"walk dealt round-robin, integer reduce-scatter of the accumulators" if args.gpus > 1 else "single GPU"),
            "note": note}


def run_aux(args, susp, vn, torch, tdtype, np_dtype, rank, world, local_rank):
    """--path aux: a step = vn_redistribute_arclength -> vn_arclength_weights -> vn_elastic_force on the
    workload's vesicles (rows f-3, a-1, f-2: everything O(P) that surrounds the pair sum in a time step).
    Reported in membrane points per second; the roofline object describes the dominant kernel
    (redistribute_kernel, FP64 pipe; algorithmic DFMA count per vesicle stated in DESIGN.md section 11)."""
    import oracle
    P = susp.nves * susp.npts
    X_h = torch.from_numpy(np.ascontiguousarray(susp.X, dtype=np_dtype)).pin_memory()
    sig_h = torch.ones((susp.nves, susp.npts), dtype=tdtype).pin_memory()
    X_d, sig_d = X_h.cuda(), sig_h.cuda()
    Xe_d, F_d = torch.empty_like(X_d), torch.empty_like(X_d)
    W_d = torch.empty((susp.nves, susp.npts), dtype=tdtype, device="cuda")
    F_host = torch.empty_like(X_h).pin_memory()
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")
    ev = lambda: torch.cuda.Event(enable_timing=True)
    parts = {"redistribute": [], "weights": [], "elastic_force": []}

    def step(record):
        e = [ev() for _ in range(4)]
        e[0].record()
        vn.vn_redistribute_arclength(X_d, out=Xe_d)
        e[1].record()
        vn.vn_arclength_weights(Xe_d, out=W_d)
        e[2].record()
        vn.vn_elastic_force(Xe_d, sig_d, 1.0, out=F_d)
        e[3].record()
        if record:
            e[3].synchronize()
            for k, name in enumerate(parts):
                parts[name].append(e[k].elapsed_time(e[k + 1]))

    for _ in range(max(args.warmup, 3)):
        step(False)
    torch.cuda.synchronize()
    sampler = ClockSampler(nvml_index(local_rank))
    sampler.start()
    n0 = vn.vn_launch_count()
    t_dev = 0.0
    for _ in range(args.steps):
        flush.fill_(1)
        torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record(); step(True); e1.record(); e1.synchronize()
        t_dev += e0.elapsed_time(e1) * 1e-3
    launches = vn.vn_launch_count() - n0
    t_e2e = 0.0
    for _ in range(args.steps):
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        X_d.copy_(X_h, non_blocking=True); sig_d.copy_(sig_h, non_blocking=True)
        step(False)
        F_host.copy_(F_d, non_blocking=True)
        torch.cuda.synchronize()
        t_e2e += time.perf_counter() - t0
    clocks = sampler.stop()
    rate, rate_e2e = args.steps * P / t_dev, args.steps * P / t_e2e
    N = susp.npts
    dfma_per_ves = 24 * N * N + 36 * N * N      # interpolant + derivative (4 x 6N x N), integration (6N x 6N)
    k_ms = statistics.mean(parts["redistribute"])
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = SMS * FP64_LANES * sm_max * 1e6 / 1e12
    achieved = dfma_per_ves * susp.nves / (k_ms * 1e-3) / 1e12
    es = 4 if args.precision == "f32" else 8
    line = {"metric": "membrane points/s through redistribution + weights + elastic force", "value": rate,
            "unit": "points/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True, "scaling": "strong", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"BASELINE.json configs[{args.workload}]: {susp.name}", "path": "rows f-3, a-1, f-2",
                       "nves": susp.nves, "npts": susp.npts, "storage": args.precision,
                       "l2": "flushed between timed steps (256 MiB write)"},
            "clocks": clocks, "gpu_launches": int(launches),
            "kernel_ms": {k: statistics.mean(v) for k, v in parts.items()},
            "roofline": {"bound": "alu", "kernel": "redistribute_kernel", "achieved": achieved, "peak": peak,
                         "unit": "T DFMA lane-instr/s (FP64 pipe)", "frac": achieved / peak,
                         "peak_source": "derived: 148 SMs x 64 lanes x %.0f MHz" % sm_max,
                         "dfma_per_vesicle": dfma_per_ves, "traffic": None},
            "e2e": {"value": rate_e2e, "unit": "points/s", "h2d_bytes_per_step": 3 * es * P, "d2h_bytes_per_step": 2 * es * P}}
    if not args.no_cpu_baseline:
        Xo = np.asarray(susp.X, dtype=np_dtype).astype(np.float64)
        nv = min(susp.nves, 4000)
        t0 = time.perf_counter()
        Xe = oracle.redistribute(Xo[:nv]); oracle.weights(Xe); oracle.elastic_force(Xe, np.ones((nv, susp.npts)), 1.0)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": nv * susp.npts / dt, "unit": "points/s", "cores": oracle.num_threads(),
                                "kind": "oracle", "sample": f"first {nv} vesicles ({dt:.1f} s)"}
    print(json.dumps(line), flush=True)


def traffic_from_profiles(workload, precision, path):
    """DRAM bytes per launch of the pair kernel from the committed `ncu --set full` capture (profiles/traffic.csv names
    the capture); a live run cannot measure it -- the profiler is not attached -- so it is looked up, or null."""
    try:
        import csv
        with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
            for row in csv.DictReader(fh):
                if (row["workload"] == f"config{workload}" and row["precision"] == precision
                        and row.get("path", "farfield") == path):
                    return int(row["dram_read_bytes"]) + int(row["dram_write_bytes"]), row.get("source")
    except Exception:
        pass
    return None, None


_SUSPENSIONS = {}          # workload index -> generated suspension (the default run measures several paths on configs[4])


def measure(ctx, m):
    """One workload / precision / path through the device-timed and (optionally) the host-buffer legs.
    ctx: torch, vn, multi, rank, world, local_rank, flush;  m: workload, precision, path, steps, warmup, order, graph, e2e.
    Returns a dict (every rank; rank 0 prints)."""
    torch, vn, multi = ctx.torch, ctx.vn, ctx.multi
    from paper_2606_25569_b200 import inputs
    rank, world = ctx.rank, ctx.world
    tdtype = torch.float32 if m.precision == "f32" else torch.float64
    np_dtype = np.float32 if m.precision == "f32" else np.float64
    susp = _SUSPENSIONS.get(m.workload) or _SUSPENSIONS.setdefault(m.workload, inputs.config(m.workload))   # same seed on every rank
    seq_np = susp.X_sequence if susp.X_sequence else [susp.X]
    evals = len(seq_np)
    P = susp.nves * susp.npts
    pairs_eval = 512 * 512 * P if m.path == "targets" else susp.pairs
    vb, ve = multi.shard_range(susp.nves, world, rank)  # this rank's vesicles (everything at world = 1)
    nloc = ve - vb

    # ---- device-resident inputs (value) and pinned host inputs (e2e): this rank's shard
    seq_h = [torch.from_numpy(np.ascontiguousarray(x[vb:ve], dtype=np_dtype)).pin_memory() for x in seq_np]
    F_h = torch.from_numpy(np.ascontiguousarray(susp.F[vb:ve], dtype=np_dtype)).pin_memory()
    U_h = torch.empty_like(seq_h[0]).pin_memory()
    seq_d = [x.cuda() for x in seq_h]
    F_d = F_h.cuda()
    X_d = torch.empty_like(seq_d[0])
    W_d = torch.empty((nloc, susp.npts), dtype=tdtype, device="cuda")
    U_d = torch.empty_like(X_d)
    fmm_order = m.order or (14 if m.precision == "f32" else 38)
    if m.path == "masked":                             # CSR buffers sized once (4 near vesicles per point is generous)
        near_ptr = torch.empty(P + 1, dtype=torch.int64, device="cuda")
        near_ves = torch.empty(4 * P, dtype=torch.int32, device="cuda")
    if m.path == "targets":
        Xt_h = torch.from_numpy(target_grid(susp, 512, np_dtype)).pin_memory()
        Xt_d = Xt_h.cuda()
        Ut_d = torch.empty_like(Xt_d)
        Ut_h = torch.empty_like(Xt_h).pin_memory()

    # the two calls of the hot path with their arguments marshalled once (the buffers are the same in every step)
    call_weights = vn.prepare_arclength_weights(X_d, W_d)
    call_farfield = vn.prepare_farfield(X_d, F_d, W_d, U_d, susp.mu)
    call_fmm = vn.prepare_farfield_fmm(X_d, F_d, W_d, U_d, susp.mu, fmm_order)

    def evaluate():
        call_weights()                                 # a-1 (on the rank's own vesicles)
        if world > 1:                                   # section 8e: all-gather, partial, reduce-scatter, finish
            U_d.copy_(multi.sharded_farfield_gpu(vn, X_d, F_d, W_d, susp.nves, susp.mu, rank, world))
        elif m.path == "farfield":
            call_farfield()                            # a-2 .. a-5
        elif m.path == "fmm":
            call_fmm()
        elif m.path == "masked":
            vn.vn_near_pairs(X_d, W_d, near_ptr, near_ves)
            vn.vn_farfield_masked(X_d, F_d, W_d, near_ptr, near_ves, susp.mu, out=U_d)
        else:
            vn.vn_farfield_targets(Xt_d, X_d, F_d, W_d, susp.mu, out=Ut_d, fmm_order=m.order)   # --order > 0: FMM

    if evals == 1:
        X_d.copy_(seq_d[0])                            # one evaluation per step: the input stays where it is

    def step_device():
        for c in range(evals):
            if evals > 1:
                X_d.copy_(seq_d[c])                    # the sequence's next positions: device-to-device, same stream
            evaluate()

    def step_host():
        for c in range(evals):
            if m.path == "farfield" and world == 1:
                vn.vn_farfield_host(seq_h[c], F_h, None, susp.mu, out=U_h)
            else:                                      # no host entry point for these: explicit copies around the C-ABI calls
                X_d.copy_(seq_h[c], non_blocking=True)
                F_d.copy_(F_h, non_blocking=True)
                if m.path == "targets":
                    Xt_d.copy_(Xt_h, non_blocking=True)
                evaluate()
                if m.path == "targets":
                    Ut_h.copy_(Ut_d, non_blocking=True)
                else:
                    U_h.copy_(U_d, non_blocking=True)
                torch.cuda.synchronize()

    def barrier():
        multi.barrier()
        torch.cuda.synchronize()

    def timed(step_fn, steps, use_events):
        """K steps; L2 flushed between steps outside the timed intervals.  Returns seconds (sum)."""
        total = 0.0
        for _ in range(steps):
            ctx.flush.fill_(1)
            barrier()
            if use_events:
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record()
                step_fn()
                e1.record()
                e1.synchronize()
                total += e0.elapsed_time(e1) * 1e-3
            else:
                t0 = time.perf_counter()
                step_fn()                              # synchronous call (returns after the D2H copy)
                total += time.perf_counter() - t0
            barrier()
        return total

    warm = max(m.warmup, 3)
    for _ in range(warm):
        step_device()
    torch.cuda.synchronize()
    launches_per_step = None
    if m.graph:                                        # every call only enqueues stream-ordered work: capturable
        step_eager = step_device
        cap = torch.cuda.Stream()
        cap.wait_stream(torch.cuda.current_stream())
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.stream(cap):
            step_eager()
            cap.synchronize()
            n_cap = vn.vn_launch_count()
            with torch.cuda.graph(graph, stream=cap):
                step_eager()
            launches_per_step = vn.vn_launch_count() - n_cap      # kernels recorded into the graph
        torch.cuda.synchronize()
        step_device = graph.replay
        for _ in range(2):
            step_device()
        torch.cuda.synchronize()

    sampler = ClockSampler(nvml_index(ctx.local_rank))
    sampler.start()
    vn.vn_profile_enable(True)
    vn.vn_profile_read()
    n0 = vn.vn_launch_count()
    t_dev = timed(step_device, m.steps, True)
    launches = vn.vn_launch_count() - n0
    if m.graph:
        launches = launches_per_step * m.steps               # replayed from the graph, not re-enqueued by the host
    kernel_ms = vn.vn_profile_read()
    vn.vn_profile_enable(False)
    clocks = sampler.stop()

    t_e2e = None
    if m.e2e:
        for _ in range(2 if m.path == "farfield" else 1):
            step_host()
        t_e2e = timed(step_host, m.steps, False)             # every step timed (none extrapolated)

    n_near = None
    if m.path == "masked":
        torch.cuda.synchronize()
        n_near = int(near_ptr[P].item())
        if n_near > near_ves.numel():
            raise SystemExit(f"near relation has {n_near} pairs, buffer holds {near_ves.numel()}")
    # whole-job numbers: the ranks share one job, so the work is the job's and the time the slowest rank's
    t_dev = multi.max_over_ranks(t_dev, "cuda")
    if t_e2e is not None:
        t_e2e = multi.max_over_ranks(t_e2e, "cuda")
    pairs_total = m.steps * evals * pairs_eval
    es = 4 if m.precision == "f32" else 8
    nt = 512 * 512
    return SimpleNamespace(susp=susp, evals=evals, P=P, pairs_eval=pairs_eval, value=pairs_total / t_dev / 1e9,
                           ms_per_step=t_dev / m.steps * 1e3, kernel_ms=kernel_ms, clocks=clocks, launches=int(launches),
                           e2e=None if t_e2e is None else pairs_total / t_e2e / 1e9, n_near=n_near, fmm_order=fmm_order,
                           h2d=evals * 2 * es * (2 * P + (nt if m.path == "targets" else 0)),
                           d2h=evals * 2 * es * (nt if m.path == "targets" else P), warm=warm)


def roofline_of(r, m, peaks, world):
    """The roofline object of one measurement (pair kernel of the exact paths)."""
    sm_max = r.clocks.get("sm_max_mhz") or measured_peaks().get("sm_max_mhz") or 1965.0
    lanes = FP32_LANES if m.precision == "f32" else FP64_LANES
    peak_nominal = SMS * lanes * sm_max * 1e6 / 1e12                   # T lane-instr/s at max clock
    peak_meas = None
    if peaks:
        peak_meas = (peaks["ffma2"] if m.precision == "f32" else peaks["dfma"]) / 1e12
    k_ms = statistics.mean(r.kernel_ms) if r.kernel_ms else None
    # with N GPUs each launch of the pair kernel processes 1/N of the blocks
    pairs_launch = r.pairs_eval / world
    achieved = LANE_OPS_PER_PAIR * pairs_launch / (k_ms * 1e-3) / 1e12 if k_ms else None
    executed = EXECUTED_LANE_OPS.get((m.path, m.precision))
    traffic, traffic_src = traffic_from_profiles(m.workload, m.precision, m.path)
    pipe = "FP32" if m.precision == "f32" else "FP64"
    return {"bound": "alu",
            "kernel": ("targets_%s_kernel" if m.path == "targets" else "farfield_%s_kernel") % m.precision,
            "achieved": achieved, "peak": peak_nominal,
            "unit": "T lane-instr/s (%s pipe; 11 CANONICAL lane-instructions per pair -- the symmetric kernels execute "
                    "fewer, so this fraction can exceed the pipe's busy fraction; its ceiling is 11 / executed_lane_ops_per_pair)" % pipe,
            "frac": achieved / peak_nominal if achieved else None,
            "frac_canonical": achieved / peak_nominal if achieved else None,
            "peak_nominal": peak_nominal,
            "peak_source": "nominal: 148 SMs x %d lanes x %.0f MHz (guide unit counts, clocks.max.sm); peak_measured is this "
                           "run's vn_pipe_peaks stream (%s)" % (lanes, sm_max, "FFMA2" if m.precision == "f32" else "DFMA"),
            "peak_measured": peak_meas,
            "frac_vs_measured_peak": achieved / peak_meas if achieved and peak_meas else None,
            "executed_lane_ops_per_pair": executed,
            "frac_executed": (executed / LANE_OPS_PER_PAIR) * achieved / peak_nominal if achieved and executed else None,
            "kernel_ms_avg": k_ms, "kernel_launches_timed": len(r.kernel_ms),
            "kernel_ginteractions_per_s": pairs_launch / (k_ms * 1e-3) / 1e9 if k_ms else None,
            "flop_frac": (FLOP_PER_PAIR * pairs_launch / (k_ms * 1e-3) / 1e12) / (2 * peak_nominal) if k_ms else None,
            "frac_at_sampled_clock": (achieved / (SMS * lanes * r.clocks["sm_mhz"] * 1e6 / 1e12)
                                      if achieved and r.clocks.get("sm_mhz") else None),
            "hbm_algorithmic_bytes": 28 * r.P if m.precision == "f32" else 56 * r.P,
            "traffic": traffic, "traffic_source": ("profiles/" + traffic_src) if traffic_src else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--path", default="farfield", choices=["farfield", "masked", "targets", "aux", "fmm"],
                    help="farfield: rows a-1..a-5 (the headline); masked: row f-1 (vn_near_pairs + "
                         "vn_farfield_masked); targets: row f-4 (vn_farfield_targets on a 512x512 grid); "
                         "aux: the O(P) rows around the sum (f-3 redistribution, a-1 weights, f-2 elastic force), "
                         "reported in points/s; fmm: vn_farfield_fmm (approximate, O(P)), reported in the direct sum's "
                         "interactions per second so that it compares with --path farfield")
    ap.add_argument("--order", type=int, default=0, help="expansion order of --path fmm (default 14 for f32, 38 for f64); with --path targets a value > 0 "
                         "selects vn_farfield_targets_fmm")
    ap.add_argument("--graph", action="store_true",
                    help="capture one step (all its evaluations) into a CUDA graph after the warm-up and time graph replays")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-sweep", action="store_true", help="skip the sweep over configs[3] / configs[1] of the default invocation")
    ap.add_argument("--no-peaks", action="store_true", help="skip the pipe-rate microbenchmark (vn_pipe_peaks)")
    args = ap.parse_args()
    if args.workload == 0:
        args.precision = "f64"          # config 0 is fp64 only

    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2606_25569_b200 as vn
    from paper_2606_25569_b200 import inputs, multi

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    if world > 1 and args.path != "farfield":
        raise SystemExit("only the farfield path is sharded over GPUs (DESIGN.md section 8); run the other paths with --gpus 1")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    vn.lib()                                           # fail loudly if the extension is missing

    tdtype = torch.float32 if args.precision == "f32" else torch.float64
    np_dtype = np.float32 if args.precision == "f32" else np.float64
    if args.path == "aux":
        return run_aux(args, inputs.config(args.workload), vn, torch, tdtype, np_dtype, rank, world, local_rank)

    ctx = SimpleNamespace(torch=torch, vn=vn, multi=multi, rank=rank, world=world, local_rank=local_rank,
                          flush=torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda"))
    m = SimpleNamespace(workload=args.workload, precision=args.precision, path=args.path, steps=args.steps,
                        warmup=args.warmup, order=args.order, graph=args.graph, e2e=not args.no_e2e)
    r = measure(ctx, m)

    default_run = (world == 1 and args.path == "farfield" and args.workload == 4 and args.precision == "f32"
                   and not args.graph)
    peaks = None
    if not args.no_peaks and world == 1:
        sampler = ClockSampler(nvml_index(local_rank))
        sampler.start()
        peaks = vn.vn_pipe_peaks()
        peaks["clocks"] = sampler.stop()
    sweep = []
    if default_run and not args.no_sweep:              # the other configurations north_star's target names, same run
        for w, prec, steps in ((3, "f32", 10), (3, "f64", 5), (1, "f32", 20)):
            ms = SimpleNamespace(workload=w, precision=prec, path="farfield", steps=steps, warmup=3, order=0,
                                 graph=False, e2e=False)
            rs = measure(ctx, ms)
            rl = roofline_of(rs, ms, peaks, 1)
            sweep.append({"workload": f"BASELINE.json configs[{w}]: {rs.susp.name}", "precision": prec, "value": rs.value,
                          "unit": UNIT, "steps": steps, "ms_per_step": rs.ms_per_step, "kernel_ms_avg": rl["kernel_ms_avg"],
                          "frac": rl["frac"], "frac_vs_measured_peak": rl["frac_vs_measured_peak"],
                          "frac_executed": rl["frac_executed"], "clocks": rs.clocks, "gpu_launches": rs.launches})

    next_rows = []
    if default_run and not args.no_sweep:              # row f-4b in the same run: the O(P) evaluation of the same sum
        for w, steps in ((4, 3), (3, 10)):
            ms = SimpleNamespace(workload=w, precision="f32", path="fmm", steps=steps, warmup=3, order=0,
                                 graph=False, e2e=False)
            rs = measure(ctx, ms)
            evals = len(rs.susp.X_sequence) if rs.susp.X_sequence else 1
            next_rows.append({"row": "f-4b vn_farfield_fmm (approximate, O(P))", "workload": f"BASELINE.json configs[{w}]: {rs.susp.name}",
                              "precision": "f32", "order": rs.fmm_order, "steps": steps, "ms_per_step": rs.ms_per_step,
                              "evaluations_per_step": evals, "ms_per_evaluation": rs.ms_per_step / evals,
                              "equivalent_value": rs.value, "unit": UNIT + " (the direct sum's pair count over this time)",
                              "clocks": rs.clocks, "gpu_launches": rs.launches})

    if rank == 0:
        line = {"metric": METRIC, "value": r.value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": r.warm, "ms_per_step": r.ms_per_step, "higher_is_better": True,
                "scaling": "strong", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
                "config": workload_config(args, r.susp), "clocks": r.clocks, "gpu_launches": r.launches,
                "roofline": roofline_of(r, m, peaks, world)}
        if peaks:
            sms = peaks["sms"]
            line["pipe_peaks"] = {"unit": "lane-ops per clock per SM at clocks.sm_max_mhz (nominal 128 / 128 / 16 / 64)",
                                  **{k: peaks[k] / (sms * (peaks["clocks"].get("sm_max_mhz") or 1965.0) * 1e6)
                                     for k in ("ffma2", "ffma", "mufu", "dfma", "ffma2_noreuse", "dfma_noreuse")},
                                  "lane_ops_per_s": {k: peaks[k] for k in ("ffma2", "ffma", "mufu", "dfma", "ffma2_noreuse", "dfma_noreuse")},
                                  "sms": sms, "clocks": peaks["clocks"]}
        if r.e2e is not None:
            line["e2e"] = {"value": r.e2e, "unit": UNIT, "h2d_bytes_per_step": r.h2d // world, "d2h_bytes_per_step": r.d2h // world,
                           "steps_timed": args.steps,
                           "api": "vn_farfield_host (pinned host buffers; weights computed on device)"
                                  if args.path == "farfield" and world == 1 else
                                  "pinned host buffers -> device copies -> the path's C-ABI calls -> copy back, synchronised"
                                  + (" (bytes per rank)" if world > 1 else "")}
        if args.path == "masked":
            line["config"]["near_pairs"] = r.n_near
        if args.path == "fmm" or (args.path == "targets" and args.order > 0):
            # an approximate O(P) algorithm does not execute the direct sum's interactions: no ALU roofline fraction
            # is claimed for it; `value` is the direct sum's pair count over the FMM's time ("equivalent" rate)
            line["config"]["order"] = r.fmm_order if args.path == "fmm" else args.order
            rl = line["roofline"]
            rl["kernel"] = "fmm kernels (P2M, M2M, M2L, L2L, L2P+P2P); kernel_ms_avg spans all of them"
            rl["equivalent_ginteractions_per_s"] = rl.pop("kernel_ginteractions_per_s", None)
            for k in ("achieved", "frac", "frac_canonical", "flop_frac", "frac_at_sampled_clock", "frac_vs_measured_peak",
                      "frac_executed", "executed_lane_ops_per_pair"):
                rl[k] = None
            rl["note"] = ("approximate algorithm (expansion order in config.order): no fraction of the pair kernels' "
                          "instruction roofline is claimed; see profiles/ for the FP64-pipe occupancy of its dominant kernels")
        if sweep:
            line["sweep"] = sweep
        if next_rows:
            line["next_rows"] = next_rows
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(r.susp, np_dtype, args.path)
        print(json.dumps(line), flush=True)

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
