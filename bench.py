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
timed region).  With --gpus N every rank evaluates its own, differently seeded suspension of the
same shape (independent problems, no data-path collective): "scaling": "weak".

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

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "far-field Stokeslet GInteractions/s"
UNIT = "GInt/s"
# canonical per-pair work: 2 FADD + 3 FMUL + 6 FFMA = 11 FP32-pipe lane
# instructions (17 flop) + 2 SFU ops; fp64: the same 11 DP instructions (17 flop).
LANE_OPS_PER_PAIR = 11
FLOP_PER_PAIR = 17
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
                time.sleep(0.1)
        except Exception as exc:                      # no NVML: report that, do not fail the bench
            self.reasons.add(f"nvml_unavailable:{type(exc).__name__}")

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


def make_workload(index, rank):
    """Suspension for this rank: rank 0 gets BASELINE.json's seed, rank r the same recipe with seed + 1000 r."""
    from paper_2606_25569_b200 import inputs
    from paper_2606_25569_b200 import multi
    if rank == 0 or index == 0:
        return inputs.config(index)
    kw = dict(inputs._CONFIGS[index])
    return inputs.suspension(seed=multi.shard_seed(inputs.BASE_SEED, index, rank), **kw)


def target_grid(susp, n_side, np_dtype):
    """n_side x n_side velocity-field grid over the suspension's bounding box plus a margin of 1
    (row f-4).  Grid points that fall close to a membrane simply get the plain trapezoid value."""
    P = susp.X.reshape(-1, 2)
    lo, hi = P.min(0) - 1.0, P.max(0) + 1.0
    gx = np.linspace(lo[0], hi[0], n_side)
    gy = np.linspace(lo[1], hi[1], n_side)
    return np.ascontiguousarray(np.stack(np.meshgrid(gx, gy, indexing="ij"), -1).reshape(-1, 2), dtype=np_dtype)


def oracle_rate(susp, np_dtype, seconds, rng_seed, path="farfield"):
    """Times the oracle (as it stands) on a bounded random sample of targets x ALL sources of the
    same workload; returns (GInt/s, cores, description)."""
    import oracle
    X = np.asarray(susp.X, dtype=np_dtype).astype(np.float64)
    F = np.asarray(susp.F, dtype=np_dtype).astype(np.float64)
    W = oracle.weights(X)
    P = susp.nves * susp.npts
    rng = np.random.Generator(np.random.PCG64(rng_seed))
    if path == "targets":
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


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric/config; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    susp = make_workload(args.workload, 0)
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
            "ms_per_step": evals * pairs_eval / (value * 1e9) * 1e3, "higher_is_better": True, "scaling": "weak",
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
            "parallelism": f"{args.gpus} independent suspensions (one per GPU)" if args.gpus > 1 else "single GPU",
            "note": note}


def run_aux(args, susp, vn, torch, tdtype, np_dtype, rank, world, local_rank):
    """--path aux: a step = vn_redistribute_arclength -> vn_arclength_weights -> vn_elastic_force on the
    workload's vesicles (rows f-3, a-1, f-2: everything O(P) that surrounds the pair sum in a time step).
    Reported in membrane points per second; the roofline object describes the dominant kernel
    (redistribute_kernel, FP64 pipe; algorithmic DFMA count per vesicle stated in DESIGN.md section 11)."""
    from paper_2606_25569_b200 import multi
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
        multi.barrier(); torch.cuda.synchronize()
        e0, e1 = ev(), ev()
        e0.record(); step(True); e1.record(); e1.synchronize()
        t_dev += e0.elapsed_time(e1) * 1e-3
    launches = vn.vn_launch_count() - n0
    t_e2e = 0.0
    for _ in range(args.steps):
        multi.barrier(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        X_d.copy_(X_h, non_blocking=True); sig_d.copy_(sig_h, non_blocking=True)
        step(False)
        F_host.copy_(F_d, non_blocking=True)
        torch.cuda.synchronize()
        t_e2e += time.perf_counter() - t0
    sampler.stop_flag.set(); sampler.join()
    rate, t_dev, _ = multi.whole_job_rate(args.steps * P, t_dev, "cuda")
    rate_e2e, t_e2e, _ = multi.whole_job_rate(args.steps * P, t_e2e, "cuda")
    if rank != 0:
        return
    N = susp.npts
    dfma_per_ves = 24 * N * N + 36 * N * N      # interpolant + derivative (4 x 6N x N), integration (6N x 6N)
    k_ms = statistics.mean(parts["redistribute"])
    clocks = sampler.summary()
    sm_max = clocks.get("sm_max_mhz") or 1965.0
    peak = SMS * FP64_LANES * sm_max * 1e6 / 1e12
    achieved = dfma_per_ves * susp.nves / (k_ms * 1e-3) / 1e12
    es = 4 if args.precision == "f32" else 8
    line = {"metric": "membrane points/s through redistribution + weights + elastic force", "value": rate,
            "unit": "points/s", "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
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
    if world == 1 and not args.no_cpu_baseline:
        Xo = np.asarray(susp.X, dtype=np_dtype).astype(np.float64)
        nv = min(susp.nves, 4000)
        t0 = time.perf_counter()
        Xe = oracle.redistribute(Xo[:nv]); oracle.weights(Xe); oracle.elastic_force(Xe, np.ones((nv, susp.npts)), 1.0)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": nv * susp.npts / dt, "unit": "points/s", "cores": oracle.num_threads(),
                                "kind": "oracle", "sample": f"first {nv} vesicles ({dt:.1f} s)"}
    print(json.dumps(line), flush=True)


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
    ap.add_argument("--order", type=int, default=0, help="expansion order of --path fmm (default 12 for f32, 38 for f64); with --path targets a value > 0 "
                         "selects vn_farfield_targets_fmm")
    ap.add_argument("--graph", action="store_true",
                    help="capture one step (all its evaluations) into a CUDA graph after the warm-up and time graph replays")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    args = ap.parse_args()
    if args.workload == 0:
        args.precision = "f64"          # config 0 is fp64 only

    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import paper_2606_25569_b200 as vn

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the product has no CPU path")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))
    vn.lib()                                           # fail loudly if the extension is missing

    tdtype = torch.float32 if args.precision == "f32" else torch.float64
    np_dtype = np.float32 if args.precision == "f32" else np.float64
    susp = make_workload(args.workload, rank)
    if args.path == "aux":
        return run_aux(args, susp, vn, torch, tdtype, np_dtype, rank, world, local_rank)
    seq_np = susp.X_sequence if susp.X_sequence else [susp.X]
    evals = len(seq_np)
    P = susp.nves * susp.npts
    pairs_eval = 512 * 512 * P if args.path == "targets" else susp.pairs
    pairs_step = evals * pairs_eval

    # ---- device-resident inputs (value) and pinned host inputs (e2e)
    seq_h = [torch.from_numpy(np.ascontiguousarray(x, dtype=np_dtype)).pin_memory() for x in seq_np]
    F_h = torch.from_numpy(np.ascontiguousarray(susp.F, dtype=np_dtype)).pin_memory()
    U_h = torch.empty_like(seq_h[0]).pin_memory()
    seq_d = [x.cuda() for x in seq_h]
    F_d = F_h.cuda()
    X_d = torch.empty_like(seq_d[0])
    W_d = torch.empty((susp.nves, susp.npts), dtype=tdtype, device="cuda")
    U_d = torch.empty_like(X_d)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device="cuda")

    fmm_order = args.order or (12 if args.precision == "f32" else 38)
    if args.path == "masked":                          # CSR buffers sized once (4 near vesicles per point is generous)
        near_ptr = torch.empty(P + 1, dtype=torch.int64, device="cuda")
        near_ves = torch.empty(4 * P, dtype=torch.int32, device="cuda")
    if args.path == "targets":
        Xt_h = torch.from_numpy(target_grid(susp, 512, np_dtype)).pin_memory()
        Xt_d = Xt_h.cuda()
        Ut_d = torch.empty_like(Xt_d)
        Ut_h = torch.empty_like(Xt_h).pin_memory()

    def evaluate():
        vn.vn_arclength_weights(X_d, out=W_d)          # a-1
        if args.path == "farfield":
            vn.vn_farfield(X_d, F_d, W_d, susp.mu, out=U_d)   # a-2 .. a-5
        elif args.path == "fmm":
            vn.vn_farfield_fmm(X_d, F_d, W_d, susp.mu, fmm_order, out=U_d)
        elif args.path == "masked":
            vn.vn_near_pairs(X_d, W_d, near_ptr, near_ves)
            vn.vn_farfield_masked(X_d, F_d, W_d, near_ptr, near_ves, susp.mu, out=U_d)
        else:
            vn.vn_farfield_targets(Xt_d, X_d, F_d, W_d, susp.mu, out=Ut_d, fmm_order=args.order)   # --order > 0: FMM

    def step_device():
        for c in range(evals):
            X_d.copy_(seq_d[c])                        # device-to-device, same stream
            evaluate()

    def step_host():
        for c in range(evals):
            if args.path == "farfield":
                vn.vn_farfield_host(seq_h[c], F_h, None, susp.mu, out=U_h)
            else:                                      # no host entry point for the NEXT rows: explicit copies
                X_d.copy_(seq_h[c], non_blocking=True)
                F_d.copy_(F_h, non_blocking=True)
                if args.path == "targets":
                    Xt_d.copy_(Xt_h, non_blocking=True)
                evaluate()
                if args.path == "targets":
                    Ut_h.copy_(Ut_d, non_blocking=True)
                else:
                    U_h.copy_(U_d, non_blocking=True)
                torch.cuda.synchronize()

    from paper_2606_25569_b200 import multi

    def barrier():
        multi.barrier()
        torch.cuda.synchronize()

    def timed(step_fn, steps, use_events):
        """K steps; L2 flushed between steps outside the timed intervals.  Returns seconds (sum)."""
        total = 0.0
        for _ in range(steps):
            flush.fill_(1)
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

    for _ in range(max(args.warmup, 3)):
        step_device()
    torch.cuda.synchronize()
    step_eager = step_device
    if args.graph:                                     # every call only enqueues stream-ordered work: capturable
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

    sampler = ClockSampler(nvml_index(local_rank))
    sampler.start()
    vn.vn_profile_enable(True)
    vn.vn_profile_read()
    n0 = vn.vn_launch_count()
    t_dev = timed(step_device, args.steps, True)
    launches = vn.vn_launch_count() - n0
    if args.graph:
        launches = launches_per_step * args.steps            # replayed from the graph, not re-enqueued by the host
    kernel_ms = vn.vn_profile_read()
    vn.vn_profile_enable(False)
    sampler.stop_flag.set()
    sampler.join()

    t_e2e = None
    if not args.no_e2e:
        for _ in range(3 if args.path == "farfield" else 1):
            step_host()
        t_e2e = timed(step_host, max(1, min(args.steps, 2)), False) / max(1, min(args.steps, 2)) * args.steps

    if args.path == "masked":
        torch.cuda.synchronize()
        n_near = int(near_ptr[P].item())
        if n_near > near_ves.numel():
            raise SystemExit(f"near relation has {n_near} pairs, buffer holds {near_ves.numel()}")
    # whole-job numbers: work summed over ranks, time = the slowest rank (paper_2606_25569_b200/multi.py)
    rate_dev, t_dev, _ = multi.whole_job_rate(args.steps * pairs_step, t_dev, "cuda")
    if t_e2e is not None:
        rate_e2e, t_e2e, _ = multi.whole_job_rate(args.steps * pairs_step, t_e2e, "cuda")

    if rank == 0:
        value = rate_dev / 1e9
        clocks = sampler.summary()
        peaks = measured_peaks()
        sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        lanes = FP32_LANES if args.precision == "f32" else FP64_LANES
        peak_lane = SMS * lanes * sm_max * 1e6 / 1e12                     # T lane-instr/s at max clock
        k_ms = statistics.mean(kernel_ms) if kernel_ms else None
        achieved = LANE_OPS_PER_PAIR * pairs_eval / (k_ms * 1e-3) / 1e12 if k_ms else None
        traffic = None                                   # dram bytes per launch from the committed ncu --set full capture
        try:
            import csv
            with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
                for row in csv.DictReader(fh):
                    if (row["workload"] == f"config{args.workload}" and row["precision"] == args.precision
                            and row.get("path", "farfield") == args.path):
                        traffic = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
        except Exception:
            pass
        roofline = {"bound": "alu",
                    "kernel": ("fmm kernels (P2M, M2M, M2L, L2L, L2P+P2P)" if args.path == "fmm" else
                               ("targets_%s_kernel" if args.path == "targets" else "farfield_%s_kernel") % args.precision),
                    "achieved": achieved, "peak": peak_lane,
                    "unit": "T lane-instr/s (%s pipe; 11 canonical instr per pair)" % ("FP32" if args.precision == "f32" else "FP64"),
                    "frac": achieved / peak_lane if achieved else None,
                    "peak_source": "derived: 148 SMs x %d lanes x %.0f MHz (guide unit counts, clocks.max.sm); "
                                   "MEASURED_PEAKS.json holds only HBM/bf16 peaks" % (lanes, sm_max),
                    "kernel_ms_avg": k_ms, "kernel_launches_timed": len(kernel_ms),
                    "kernel_ginteractions_per_s": pairs_eval / (k_ms * 1e-3) / 1e9 if k_ms else None,
                    "flop_frac": (FLOP_PER_PAIR * pairs_eval / (k_ms * 1e-3) / 1e12) / (2 * peak_lane) if k_ms else None,
                    "frac_at_sampled_clock": (achieved / (SMS * lanes * clocks["sm_mhz"] * 1e6 / 1e12)
                                              if achieved and clocks.get("sm_mhz") else None),
                    "hbm_algorithmic_bytes": 28 * P if args.precision == "f32" else 56 * P,
                    "traffic": traffic}
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": max(args.warmup, 3), "ms_per_step": t_dev / args.steps * 1e3, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": args.precision, "data": "synthetic",
                "config": workload_config(args, susp), "clocks": clocks, "gpu_launches": int(launches),
                "roofline": roofline}
        if t_e2e is not None:
            es = 4 if args.precision == "f32" else 8
            nt = 512 * 512
            line["e2e"] = {"value": rate_e2e / 1e9, "unit": UNIT,
                           "h2d_bytes_per_step": evals * 2 * es * (2 * P + (nt if args.path == "targets" else 0)),
                           "d2h_bytes_per_step": evals * 2 * es * (nt if args.path == "targets" else P),
                           "api": "vn_farfield_host (pinned host buffers; weights computed on device)"
                                  if args.path == "farfield" else
                                  "pinned host buffers -> device copies -> the path's C-ABI calls -> copy back, synchronised"}
        if args.path == "masked":
            line["config"]["near_pairs"] = n_near
        if args.path == "fmm" or (args.path == "targets" and args.order > 0):
            # an approximate O(P) algorithm does not execute the direct sum's interactions: no ALU roofline fraction
            # is claimed for it; `value` is the direct sum's pair count over the FMM's time ("equivalent" rate)
            line["config"]["order"] = fmm_order if args.path == "fmm" else args.order
            rl = line["roofline"]
            rl["kernel"] = "fmm kernels (P2M, M2M, M2L, L2L, L2P+P2P); kernel_ms_avg spans all of them"
            rl["equivalent_ginteractions_per_s"] = rl.pop("kernel_ginteractions_per_s", None)
            for k in ("achieved", "frac", "flop_frac", "frac_at_sampled_clock"):
                rl[k] = None
            rl["note"] = ("approximate algorithm (expansion order in config.order): no fraction of the pair kernels' "
                          "instruction roofline is claimed; see profiles/r1f_fmm_kernels_config4_f64_ncu.md for the "
                          "FP64-pipe occupancy of its two dominant kernels")
        if world == 1 and not args.no_cpu_baseline:
            v, cores, sample = oracle_rate(susp, np_dtype, 15.0, 4242, args.path)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        print(json.dumps(line), flush=True)

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
