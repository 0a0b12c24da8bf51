"""The N > 1 path of bench.py on CPU: two gloo ranks, each with its own suspension (weak scaling,
no data-path collective), timing reduced as max over ranks and work as sum over ranks."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

from paper_2606_25569_b200 import inputs, multi


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        seed = multi.shard_seed(inputs.BASE_SEED, 1, rank)
        s = inputs.suspension(nves=6, npts=16, phi_area=0.1, aspect=1.0, seed=seed, nmodes=4)
        units = float(s.pairs) * (rank + 1)                   # unequal work: the sum must see both
        seconds = 0.5 + 0.25 * rank                           # unequal time: the max must win
        multi.barrier()
        rate, t_max, total = multi.whole_job_rate(units, seconds)
        out[rank] = (seed, float(s.X.sum()), rate, t_max, total, multi.max_over_ranks(rank), multi.sum_over_ranks(1.0))
    finally:
        dist.destroy_process_group()


def test_two_ranks_weak_scaling_reduction():
    world, port = 2, _free_port()
    with mp.get_context("spawn").Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == {0, 1}
    (seed0, sum0, rate0, tmax0, tot0, mx0, n0), (seed1, sum1, rate1, tmax1, tot1, mx1, n1) = res[0], res[1]
    assert seed0 == inputs.BASE_SEED + 1 and seed1 == seed0 + 1000      # rank 0 keeps BASELINE's seed
    assert sum0 != sum1                                                  # different suspensions
    pairs = 6 * 16 * (6 * 16 - 16)
    assert tot0 == tot1 == pairs * 3.0                                   # work: sum over ranks
    assert tmax0 == tmax1 == 0.75                                        # time: max over ranks
    assert rate0 == rate1 == pytest.approx(pairs * 3.0 / 0.75)
    assert mx0 == mx1 == 1.0 and n0 == n1 == 2.0


def test_single_process_is_identity():
    assert multi.max_over_ranks(1.5) == 1.5 and multi.sum_over_ranks(2.5) == 2.5
    assert multi.whole_job_rate(10.0, 2.0) == (5.0, 2.0, 10.0)
