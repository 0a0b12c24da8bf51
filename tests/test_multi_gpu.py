"""The N > 1 path with the REAL kernels: several processes, each a rank of a gloo group, share
ONE suspension; every rank calls vn_farfield_partial for its blocks of the pair walk on the one GPU of the box (the
ranks' kernels do not wait for one another: each runs to completion, the collectives go through host memory), the
integer accumulators are summed across ranks and vn_farfield_finish rounds each rank's shard.  The result must be
BITWISE the single-process vn_farfield (through partial + finish with one part): integer addition is associative.
tests/test_multi_gloo.py covers the same host logic on CPU with the oracle as the evaluator."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

import paper_2606_25569_b200 as vn
from paper_2606_25569_b200 import inputs, multi

pytestmark = pytest.mark.gpu


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _weights(X):
    """Trapezoid weights by the library itself (vn_arclength_weights): this file checks the sharding, not row a-1."""
    return vn.vn_arclength_weights(X)


def _worker(rank, world, port, index, dtype_name, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(0)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        dtype = getattr(torch, dtype_name)
        s = inputs.config(index)
        X = torch.from_numpy(np.ascontiguousarray(s.X)).to(dtype).cuda()
        F = torch.from_numpy(np.ascontiguousarray(s.F)).to(dtype).cuda()
        W = _weights(X)
        b, e = multi.shard_range(s.nves, world, rank)
        multi.barrier()
        U_loc = multi.sharded_farfield_gpu(vn, X[b:e].contiguous(), F[b:e].contiguous(), W[b:e].contiguous(),
                                           s.nves, s.mu, rank, world)
        torch.cuda.synchronize()
        res = {"range": (b, e), "U": U_loc.cpu().numpy()}
        if rank == 0:
            acc, gmax = vn.vn_farfield_partial(X, F, W, 0, 1)
            ref = vn.vn_farfield_finish(acc, gmax, s.nves * s.npts, dtype, s.mu)
            full = vn.vn_farfield(X, F, W, s.mu)
            torch.cuda.synchronize()
            res["ref"] = ref.cpu().numpy().reshape(s.nves, s.npts, 2)
            res["full"] = full.cpu().numpy().reshape(s.nves, s.npts, 2)
        out[rank] = res
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("index,dtype_name,world", [(1, "float32", 2), (1, "float64", 2), (2, "float32", 3)])
def test_ranks_sharing_one_suspension_reproduce_the_single_gpu_result_bitwise(index, dtype_name, world):
    port = _free_port()
    with mp.get_context("spawn").Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, index, dtype_name, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == set(range(world))
    nves, _ = inputs.config_shape(index)
    assert [res[r]["range"] for r in range(world)] == [multi.shard_range(nves, world, r) for r in range(world)]
    U = np.concatenate([res[r]["U"] for r in range(world)])
    assert U.shape == res[0]["ref"].shape
    assert np.all(np.isfinite(U))
    assert np.array_equal(U, res[0]["ref"])                 # partial (one part) + finish
    assert np.array_equal(U, res[0]["full"])                # and the one-call entry point (general path at these sizes)
