"""Host-side logic of the multi-GPU path: ONE suspension over N GPUs,
one process per GPU.

The pair kernel evaluates every unordered pair of points once and scatters into BOTH points' accumulators, so the
work cannot be cut by targets without giving up the symmetry (a target-sharded split evaluates every cross-shard
pair twice: 12.5 instead of 9.0 FP32 lane-instructions per interaction at N = 8).  It is cut by BLOCKS of the
pair walk instead:

    1. every rank owns a contiguous range of vesicles (its shard of X, F, W and of the result U);
    2. one all-gather makes all sources known everywhere           (20 B per point in fp32, 40 B in fp64);
    3. rank r runs blocks r, r + N, r + 2N, ... of the SAME grid the single-GPU call would run
       (vn_farfield_partial) and is left with raw 64-bit fixed-point accumulators for ALL points;
    4. one integer reduce-scatter (sum) hands every rank the summed accumulators of its own vesicles
                                                                    (16 B per point in fp32, 32 B in fp64);
    5. vn_farfield_finish scales and rounds the shard: U stays sharded.

Integer addition is associative, so the result is bit for bit the single-GPU result whatever N is, and the 2x saving
of the symmetric evaluation is kept.  At 8,000 x 128 (fp32): 20 MB gathered + 16 MB reduce-scattered per rank against
340 ms / N of arithmetic -- tens of microseconds on NVLink 5 / NVSwitch; the collectives are NCCL's (there is nothing
to overlap them with: step 2 must finish before, step 4 can only start after, the kernel).

`sharded_farfield` is written against two callables (the accumulate and the finish step) so that the CPU tests can
drive the same partition / gather / reduce logic with the oracle as the evaluator (tests/test_multi_gloo.py);
`sharded_farfield_gpu` binds it to the library.  Backend-agnostic: NCCL on GPUs, gloo in the tests (CPU tensors, or
CUDA tensors staged through host memory: tests/test_multi_gpu.py runs several ranks' real kernels on one GPU).
"""
from __future__ import annotations


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


# ------------------------------------------------------------------------------------------------ sharding
def shard_size(nves: int, world: int) -> int:
    """Vesicles per rank: ceil(nves / world); the last ranks may hold fewer (or none)."""
    return (nves + world - 1) // world


def shard_range(nves: int, world: int, rank: int):
    """[begin, end) of the vesicles rank `rank` owns."""
    s = shard_size(nves, world)
    return min(rank * s, nves), min((rank + 1) * s, nves)


def _staged(d, t):
    """gloo moves host memory only: a CUDA tensor goes through a host copy there (tests); NCCL takes it as it is."""
    return d.get_backend() == "gloo" and t.is_cuda


def all_gather_shards(local, nves: int, world: int):
    """local: this rank's shard [n_local, ...] -> the whole array [nves, ...] on every rank.  Shards are padded to
    the common size ceil(nves / world) for the collective and the padding is cut off again."""
    import torch
    d = _dist()
    if d is None:
        return local
    s = shard_size(nves, world)
    if local.shape[0] != s:
        pad = torch.zeros((s - local.shape[0],) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
        local = torch.cat([local, pad], 0)
    if _staged(d, local):
        host = torch.empty((world * s,) + tuple(local.shape[1:]), dtype=local.dtype)
        d.all_gather_into_tensor(host, local.contiguous().cpu())
        return host[:nves].to(local.device)
    full = torch.empty((world * s,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    d.all_gather_into_tensor(full, local.contiguous())
    return full[:nves]


def reduce_scatter_sum(full, nves: int, per_vesicle: int, world: int, rank: int):
    """full: integer accumulators of ALL vesicles [nves * per_vesicle] computed by this rank -> the sum over ranks of
    this rank's own vesicles [n_local * per_vesicle].  One reduce-scatter where the backend has it (NCCL); gloo has
    none, there it is an all-reduce followed by the slice (tests only)."""
    import torch
    d = _dist()
    b, e = shard_range(nves, world, rank)
    if d is None:
        return full[b * per_vesicle:e * per_vesicle]
    s = shard_size(nves, world)
    if d.get_backend() == "gloo":
        if full.is_cuda:
            host = full.cpu()
            d.all_reduce(host, op=d.ReduceOp.SUM)
            return host[b * per_vesicle:e * per_vesicle].to(full.device)
        d.all_reduce(full, op=d.ReduceOp.SUM)
        return full[b * per_vesicle:e * per_vesicle]
    if world * s != nves:
        full = torch.cat([full, torch.zeros((world * s - nves) * per_vesicle, dtype=full.dtype, device=full.device)])
    out = torch.empty(s * per_vesicle, dtype=full.dtype, device=full.device)
    d.reduce_scatter_tensor(out, full, op=d.ReduceOp.SUM)
    return out[:(e - b) * per_vesicle]


def sharded_farfield(X_loc, F_loc, W_loc, nves: int, accumulate, finish, rank: int = 0, world: int = 1):
    """Steps 2-5 above.  X_loc, F_loc [n_local, npts, 2], W_loc [n_local, npts]: this rank's vesicles.
    accumulate(X, F, W, part, nparts) -> (acc, aux): integer accumulators of ALL points (flat, a fixed number of
    words per point) from the blocks of part `part`; aux is passed on to finish.  finish(acc_shard, aux) -> U_loc."""
    npts = X_loc.shape[1]
    X = all_gather_shards(X_loc, nves, world)
    F = all_gather_shards(F_loc, nves, world)
    W = all_gather_shards(W_loc, nves, world)
    acc, aux = accumulate(X, F, W, rank, world)
    per_vesicle = acc.numel() // nves
    assert per_vesicle * nves == acc.numel() and per_vesicle % npts == 0
    acc_loc = reduce_scatter_sum(acc, nves, per_vesicle, world, rank)
    return finish(acc_loc, aux)


def sharded_farfield_gpu(vn, X_loc, F_loc, W_loc, nves: int, mu: float, rank: int, world: int):
    """The library's kernels behind `sharded_farfield`: U_loc [n_local, npts, 2] for this rank's vesicles."""
    npts = X_loc.shape[1]
    dtype = X_loc.dtype

    def accumulate(X, F, W, part, nparts):
        return vn.vn_farfield_partial(X.contiguous(), F.contiguous(), W.contiguous(), part, nparts)

    def finish(acc_loc, gmax):
        return vn.vn_farfield_finish(acc_loc.contiguous(), gmax, nves * npts, dtype, mu).view(-1, npts, 2)

    return sharded_farfield(X_loc, F_loc, W_loc, nves, accumulate, finish, rank, world)
