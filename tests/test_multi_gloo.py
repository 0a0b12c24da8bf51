"""The N > 1 path on CPU: two gloo ranks share ONE suspension.  The partition / all-gather /
integer reduce / finish logic of paper_2606_25569_b200.multi.sharded_farfield is driven with the ORACLE as the
evaluator of a block of the pair walk (vn_plan_farfield, host-only, says which blocks a part owns), quantised to
64-bit integers like the kernels' accumulators, and must reproduce the unsharded evaluation exactly -- integer
addition is associative -- and the oracle's own full sum up to the quantum."""
import os
import socket

import numpy as np
import pytest

torch = pytest.importorskip("torch")
import torch.multiprocessing as mp

import oracle
import paper_2606_25569_b200 as vn
from paper_2606_25569_b200 import inputs, multi

QUANTUM = 2.0 ** -36          # fixed-point unit of the test evaluator
NVES, NPTS = 70, 32           # 2,240 points: 3 super-tiles of 768 (fp64 plan), a ragged last one; 70 % 2 == 0 but 70 % 4 != 0
SLOTS = 3                     # resident blocks assumed by the plan: several chunks per super-tile


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _problem():
    return inputs.suspension(nves=NVES, npts=NPTS, phi_area=0.1, aspect=1.0, seed=inputs.BASE_SEED + 77, nmodes=4)


def block_entries(plan, part, nparts):
    """(target super-tile I, source tile, both directions) for every list entry of every block of `part`: the walk
    documented in include/vesnet_farfield.h (block b = (I, chunk c), b dealt round-robin to the parts)."""
    n_st, n_chunks, sub = plan["n_super_tiles"], plan["n_chunks"], plan["tiles_per_super_tile"]
    out = []
    for b in range(part, n_st * n_chunks, nparts):
        I, c = divmod(b, n_chunks)
        S = (n_st - 1) // 2 + (1 if n_st % 2 == 0 and I < n_st // 2 else 0)
        nu = sub * (S + 1)
        for u in range(nu * c // n_chunks, nu * (c + 1) // n_chunks):
            s, k = divmod(u, sub)
            out.append((I, ((I + s) % n_st) * sub + k, s >= 1))
    return out


def oracle_accumulate(X, F, W, part, nparts):
    """The evaluator: for every list entry of the part's blocks, the oracle's sum of the source tile's points over
    the targets of the super-tile (own vesicle excluded by the oracle itself) and, for an entry of another
    super-tile, the reverse direction too; every contribution is rounded to the quantum and added as an integer."""
    Xn, Fn, Wn = X.numpy(), F.numpy(), W.numpy()
    nves, npts, _ = Xn.shape
    P = nves * npts
    plan = vn.vn_plan_farfield(nves, npts, vn.VN_F64, SLOTS)      # the grid does not depend on the number of parts
    st, tile = plan["super_tile"], plan["tile"]
    acc = np.zeros((P, 2), dtype=np.int64)

    def add(targets, sources):
        if len(targets) == 0 or len(sources) == 0:
            return
        Fm = np.zeros_like(Fn).reshape(-1, 2)
        Fm[sources] = Fn.reshape(-1, 2)[sources]
        U = oracle.farfield_subset(Xn, Fm.reshape(Fn.shape), Wn, targets, 1.0)
        acc[targets] += np.rint(U / QUANTUM).astype(np.int64)

    for I, t, both in block_entries(plan, part, nparts):
        targets = np.arange(I * st, min((I + 1) * st, P))
        sources = np.arange(t * tile, min((t + 1) * tile, P))
        add(targets, sources)
        if both:
            add(sources, targets)
    return torch.from_numpy(acc.reshape(-1)), npts


def oracle_finish(acc_loc, npts):
    return torch.from_numpy(acc_loc.numpy().astype(np.float64) * QUANTUM).view(-1, npts, 2)


def _worker(rank, world, port, out):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        s = _problem()
        W = oracle.weights(s.X)
        b, e = multi.shard_range(s.nves, world, rank)
        X_loc, F_loc, W_loc = (torch.from_numpy(np.ascontiguousarray(a[b:e])) for a in (s.X, s.F, W))
        multi.barrier()
        U_loc = multi.sharded_farfield(X_loc, F_loc, W_loc, s.nves, oracle_accumulate, oracle_finish, rank, world)
        rate, t_max, total = multi.whole_job_rate(float(s.pairs) / world, 0.5 + 0.25 * rank)
        out[rank] = (b, e, U_loc.numpy(), rate, t_max, total)
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_one_suspension_over_several_ranks_is_exact(world):
    port = _free_port()
    with mp.get_context("spawn").Manager() as mgr:
        out = mgr.dict()
        mp.spawn(_worker, args=(world, port, out), nprocs=world, join=True)
        res = dict(out)
    assert set(res) == set(range(world))
    s = _problem()
    W = oracle.weights(s.X)
    # the ranks' ranges tile the vesicles in order (70 vesicles over 4 ranks: 18 + 18 + 18 + 16)
    assert [res[r][0] for r in range(world)] == [multi.shard_range(NVES, world, r)[0] for r in range(world)]
    assert res[0][0] == 0 and res[world - 1][1] == NVES and all(res[r][1] == res[r + 1][0] for r in range(world - 1))
    U_sharded = np.concatenate([res[r][2] for r in range(world)])
    # unsharded evaluation by the same evaluator in this process: nparts = 1
    acc, npts = oracle_accumulate(torch.from_numpy(s.X), torch.from_numpy(s.F), torch.from_numpy(W), 0, 1)
    U_single = oracle_finish(acc, npts).numpy()
    assert np.array_equal(U_sharded, U_single)                      # exact: integer sums do not depend on the split
    # and both are the oracle's sum up to the quantum per contribution
    ref = oracle.farfield(s.X, s.F, W, 1.0)
    n_contrib = -(-NVES * NPTS // 128) + 8
    assert np.abs(U_sharded - ref).max() <= n_contrib * QUANTUM
    # timing / work reductions of the bench: time = max over ranks, work = sum over ranks
    for r in range(world):
        assert res[r][4] == 0.5 + 0.25 * (world - 1) and res[r][5] == pytest.approx(float(s.pairs))
        assert res[r][3] == pytest.approx(float(s.pairs) / res[r][4])


def test_parts_partition_the_blocks():
    """Every block of the grid belongs to exactly one part, whatever the number of parts."""
    for nparts in (1, 2, 3, 8):
        plan = vn.vn_plan_farfield(NVES, NPTS, vn.VN_F64, SLOTS)
        every = sorted(e for p in range(nparts) for e in block_entries(plan, p, nparts))
        assert every == sorted(block_entries(plan, 0, 1))
        # the walk covers every (super-tile, tile) combination it should: own tiles once, foreign tiles from one side
        n_st, sub = plan["n_super_tiles"], plan["tiles_per_super_tile"]
        seen = {}
        for I, t, both in every:
            J = t // sub
            seen[(I, t)] = seen.get((I, t), 0) + 1
            assert both == (J != I)
        assert all(v == 1 for v in seen.values())
        pairs = {(min(I, t // sub), max(I, t // sub)) for I, t in seen}
        assert len(pairs) == n_st * (n_st + 1) // 2


def test_single_process_is_identity():
    assert multi.max_over_ranks(1.5) == 1.5 and multi.sum_over_ranks(2.5) == 2.5
    assert multi.whole_job_rate(10.0, 2.0) == (5.0, 2.0, 10.0)
    assert multi.shard_range(10, 1, 0) == (0, 10) and multi.shard_range(10, 4, 3) == (9, 10)
    assert multi.shard_range(2, 4, 3) == (2, 2)
    t = torch.arange(12)
    assert multi.all_gather_shards(t, 12, 1) is t
    assert torch.equal(multi.reduce_scatter_sum(t, 3, 4, 1, 0), t)
