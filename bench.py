#!/usr/bin/env python
"""bench.py -- far-field Stokeslet GInteractions/s on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload 0..4] [--precision f32|f64]
    python bench.py --impl reference ...        # the oracle, as it stands, on the host cores

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
    if rank == 0 or index == 0:
        return inputs.config(index)
    kw = dict(inputs._CONFIGS[index])
    return inputs.suspension(seed=inputs.BASE_SEED + index + 1000 * rank, **kw)


def oracle_rate(susp, np_dtype, seconds, rng_seed):
    """Times the oracle (as it stands) on a bounded random sample of targets x ALL sources of the
    same workload; returns (GInt/s, cores, description)."""
    import oracle
    X = np.asarray(susp.X, dtype=np_dtype).astype(np.float64)
    F = np.asarray(susp.F, dtype=np_dtype).astype(np.float64)
    W = oracle.weights(X)
    P = susp.nves * susp.npts
    per_target = P - susp.npts
    rng = np.random.Generator(np.random.PCG64(rng_seed))
    probe = rng.choice(P, size=min(P, 64 * oracle.num_threads()), replace=False)
    t0 = time.perf_counter()
    oracle.farfield_subset(X, F, W, probe, susp.mu)
    rate = len(probe) * per_target / (time.perf_counter() - t0)
    n = int(max(len(probe), min(P, rate * seconds / per_target)))
    idx = rng.choice(P, size=n, replace=False)
    t0 = time.perf_counter()
    oracle.farfield_subset(X, F, W, idx, susp.mu)
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
        r, cores, sample = oracle_rate(susp, np_dtype, per_step, 7000 + s)
        if s >= args.warmup:
            rates.append(r)
    value = statistics.mean(rates)
    P = susp.nves * susp.npts
    evals = 10 if args.workload == 4 else 1
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": evals * susp.pairs / (value * 1e9) * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(args, susp, "oracle on host cores; ms_per_step extrapolated from the sampled rate"),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle",
                             "sample": f"per step: {sample}"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def workload_config(args, susp, note=""):
    evals = 10 if args.workload == 4 else 1
    return {"workload": f"BASELINE.json configs[{args.workload}]: {susp.name}",
            "nves": susp.nves, "npts": susp.npts, "points": susp.nves * susp.npts,
            "pairs_per_evaluation": susp.pairs, "evaluations_per_step": evals,
            "precision": args.precision, "l2": "flushed between timed steps (256 MiB write); inputs < L2",
            "parallelism": f"{args.gpus} independent suspensions (one per GPU)" if args.gpus > 1 else "single GPU",
            "note": note}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", type=int, default=4, choices=[0, 1, 2, 3, 4])
    ap.add_argument("--precision", default="f32", choices=["f32", "f64"])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
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
    seq_np = susp.X_sequence if susp.X_sequence else [susp.X]
    evals = len(seq_np)
    P = susp.nves * susp.npts
    pairs_step = evals * susp.pairs

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

    def step_device():
        for c in range(evals):
            X_d.copy_(seq_d[c])                        # device-to-device, same stream
            vn.vn_arclength_weights(X_d, out=W_d)      # a-1
            vn.vn_farfield(X_d, F_d, W_d, susp.mu, out=U_d)   # a-2 .. a-5

    def step_host():
        for c in range(evals):
            vn.vn_farfield_host(seq_h[c], F_h, None, susp.mu, out=U_h)

    def barrier():
        if world > 1:
            dist.barrier()
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

    sampler = ClockSampler(nvml_index(local_rank))
    sampler.start()
    vn.vn_profile_enable(True)
    vn.vn_profile_read()
    n0 = vn.vn_launch_count()
    t_dev = timed(step_device, args.steps, True)
    launches = vn.vn_launch_count() - n0
    kernel_ms = vn.vn_profile_read()
    vn.vn_profile_enable(False)
    sampler.stop_flag.set()
    sampler.join()

    t_e2e = None
    if not args.no_e2e:
        for _ in range(3):
            vn.vn_farfield_host(seq_h[0], F_h, None, susp.mu, out=U_h)
        t_e2e = timed(step_host, max(1, min(args.steps, 2)), False) / max(1, min(args.steps, 2)) * args.steps

    def max_over_ranks(x):
        if world == 1:
            return x
        t = torch.tensor([x], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    t_dev = max_over_ranks(t_dev)
    if t_e2e is not None:
        t_e2e = max_over_ranks(t_e2e)

    if rank == 0:
        value = world * args.steps * pairs_step / t_dev / 1e9
        clocks = sampler.summary()
        peaks = measured_peaks()
        sm_max = clocks.get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        lanes = FP32_LANES if args.precision == "f32" else FP64_LANES
        peak_lane = SMS * lanes * sm_max * 1e6 / 1e12                     # T lane-instr/s at max clock
        k_ms = statistics.mean(kernel_ms) if kernel_ms else None
        achieved = LANE_OPS_PER_PAIR * susp.pairs / (k_ms * 1e-3) / 1e12 if k_ms else None
        traffic = None                                   # dram bytes per launch from the committed ncu --set full capture
        try:
            import csv
            with open(os.path.join(ROOT, "profiles", "traffic.csv")) as fh:
                for row in csv.DictReader(fh):
                    if row["workload"] == f"config{args.workload}" and row["precision"] == args.precision:
                        traffic = int(row["dram_read_bytes"]) + int(row["dram_write_bytes"])
        except Exception:
            pass
        roofline = {"bound": "alu", "kernel": "farfield_%s_kernel" % args.precision,
                    "achieved": achieved, "peak": peak_lane,
                    "unit": "T lane-instr/s (%s pipe; 11 canonical instr per pair)" % ("FP32" if args.precision == "f32" else "FP64"),
                    "frac": achieved / peak_lane if achieved else None,
                    "peak_source": "derived: 148 SMs x %d lanes x %.0f MHz (guide unit counts, clocks.max.sm); "
                                   "MEASURED_PEAKS.json holds only HBM/bf16 peaks" % (lanes, sm_max),
                    "kernel_ms_avg": k_ms, "kernel_launches_timed": len(kernel_ms),
                    "kernel_ginteractions_per_s": susp.pairs / (k_ms * 1e-3) / 1e9 if k_ms else None,
                    "flop_frac": (FLOP_PER_PAIR * susp.pairs / (k_ms * 1e-3) / 1e12) / (2 * peak_lane) if k_ms else None,
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
            line["e2e"] = {"value": world * args.steps * pairs_step / t_e2e / 1e9, "unit": UNIT,
                           "h2d_bytes_per_step": evals * 2 * (2 * es * P), "d2h_bytes_per_step": evals * 2 * es * P,
                           "api": "vn_farfield_host (pinned host buffers; weights computed on device)"}
        if world == 1 and not args.no_cpu_baseline:
            v, cores, sample = oracle_rate(susp, np_dtype, 15.0, 4242)
            line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        print(json.dumps(line), flush=True)

    if world > 1:
        dist.barrier()
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
