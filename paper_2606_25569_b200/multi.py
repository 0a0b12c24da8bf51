"""Host-side logic of the multi-GPU path: one process per GPU, every rank
evaluates its OWN suspension (independent problems, no data-path collective); the only exchanges
are a barrier and two tiny all-reduces for the timing (max over ranks) and the work (sum over
ranks).  Backend-agnostic: NCCL on GPUs, gloo in the CPU tests (world_size 2)."""
from __future__ import annotations


def shard_seed(base_seed: int, index: int, rank: int) -> int:
    """Seed of rank `rank`'s suspension: rank 0 keeps BASELINE.json's seed."""
    return base_seed + index + 1000 * rank


def _dist():
    import torch.distributed as dist
    return dist if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1 else None


def barrier() -> None:
    d = _dist()
    if d is not None:
        d.barrier()


def max_over_ranks(x: float, device="cpu") -> float:
    d = _dist()
    if d is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    d.all_reduce(t, op=d.ReduceOp.MAX)
    return float(t.item())


def sum_over_ranks(x: float, device="cpu") -> float:
    d = _dist()
    if d is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    d.all_reduce(t, op=d.ReduceOp.SUM)
    return float(t.item())


def whole_job_rate(units_this_rank: float, seconds_this_rank: float, device="cpu"):
    """(units of ALL ranks) / (slowest rank's time): the bench's `value`.  Returns (rate, t_max, units)."""
    t_max = max_over_ranks(seconds_this_rank, device)
    units = sum_over_ranks(units_this_rank, device)
    return units / t_max, t_max, units
