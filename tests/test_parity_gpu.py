"""Parity of the CUDA path with the oracle (run on the B200 box: pytest -m gpu).

Every call goes through the C-ABI library via the thin binding.  Tolerances are north_star's:
relative L2 <= 1e-12 (fp64) and <= 2e-5 (fp32), measured against the oracle on the same seeded
inputs; for fp32 the oracle consumes the fp32-rounded inputs promoted to double, so the measured
error is arithmetic, not input quantisation."""
import numpy as np
import pytest

import oracle
import paper_2606_25569_b200 as vn
from paper_2606_25569_b200 import inputs

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

from parity_util import TOL, check, rel_l2

_cache = {}


def dev(a, dtype):
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).cuda()


def problem(index):
    """Config `index` with oracle weights (fp64), cached for the session."""
    if index not in _cache:
        s = inputs.config(index)
        _cache[index] = (s, oracle.weights(s.X))
    return _cache[index]


def gpu_farfield(X, F, W, mu, dtype):
    U = vn.vn_farfield(dev(X, dtype), dev(F, dtype), dev(W, dtype), mu)
    torch.cuda.synchronize()
    return U.cpu().numpy()


def oracle_inputs(X, F, W, dtype):
    """What the GPU sees, promoted to double."""
    return tuple(np.asarray(a, dtype=dtype).astype(np.float64) for a in (X, F, W))


def sample_targets(P, n, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    # always include the first and last points and both ends of a tile / vesicle boundary
    fixed = np.array([0, 1, 127, 128, P // 2, P - 129, P - 128, P - 1])
    return np.unique(np.concatenate([fixed, rng.choice(P, size=n, replace=False)]))


# ------------------------------------------------------------------------------------- full parity
@pytest.mark.parametrize("index,dtype", [(0, np.float64), (0, np.float32), (1, np.float64), (1, np.float32)])
def test_farfield_full_parity(index, dtype):
    s, W = problem(index)
    Xo, Fo, Wo = oracle_inputs(s.X, s.F, W, dtype)
    ref = oracle.farfield(Xo, Fo, Wo, s.mu)
    got = gpu_farfield(s.X, s.F, W, s.mu, dtype)
    check(got, ref, TOL[dtype], f"farfield config{index} {np.dtype(dtype).name} all targets")


# ------------------------------------------------------------------------------------- full-size configs, sampled targets
@pytest.mark.parametrize("index,dtype,nsample", [(2, np.float32, 8192), (2, np.float64, 8192),
                                                 (3, np.float32, 16384), (3, np.float64, 16384)])
def test_farfield_sampled_parity_large(index, dtype, nsample):
    s, W = problem(index)
    P = s.nves * s.npts
    idx = sample_targets(P, nsample, 260625569 + 100)
    Xo, Fo, Wo = oracle_inputs(s.X, s.F, W, dtype)
    ref = oracle.farfield_subset(Xo, Fo, Wo, idx, s.mu)
    got = gpu_farfield(s.X, s.F, W, s.mu, dtype).reshape(-1, 2)[idx]
    check(got, ref, TOL[dtype], f"farfield config{index} {np.dtype(dtype).name} sampled")


def test_config4_sequence_fp32():
    """8,000 x 128, ten consecutive evaluations on one stream reusing the device buffers (BASELINE.json configs[4]).
    ALL ten calls are compared on ALL 1.02 M targets with the fp64 GPU path on the same fp32-rounded inputs; the
    oracle checks calls 0, 4 and 9 on 16,384 sampled targets in both precisions, which ties
    the fp64 GPU path -- and through it every target of every call -- to the oracle."""
    s, W = problem(4)
    P = s.nves * s.npts
    idx = sample_targets(P, 16384, 260625569 + 100)
    seq = [dev(x, np.float32) for x in s.X_sequence]
    Xd = torch.empty_like(seq[0])
    Fd, Wd = dev(s.F, np.float32), dev(W, np.float32)
    Ud = torch.empty_like(Xd)
    outs = []
    for c in range(10):
        Xd.copy_(seq[c])
        vn.vn_farfield(Xd, Fd, Wd, s.mu, out=Ud)
        outs.append(Ud.clone())                    # stream-ordered copy of call c's result; no host synchronisation
    torch.cuda.synchronize()
    F64, W64 = Fd.double(), Wd.double()
    U64 = torch.empty((s.nves, s.npts, 2), dtype=torch.float64, device="cuda")
    for c in range(10):
        vn.vn_farfield(seq[c].double(), F64, W64, s.mu, out=U64)
        torch.cuda.synchronize()
        u64 = U64.cpu().numpy()
        check(outs[c].cpu().numpy(), u64, TOL[np.float32], f"config4 call {c}: fp32 GPU vs fp64 GPU, all targets")
        if c in (0, 4, 9):
            Xo, Fo, Wo = oracle_inputs(s.X_sequence[c], s.F, W, np.float32)
            ref = oracle.farfield_subset(Xo, Fo, Wo, idx, s.mu)
            check(outs[c].cpu().numpy().reshape(-1, 2)[idx], ref, TOL[np.float32], f"config4 call {c}: fp32 GPU vs oracle, sampled")
            check(u64.reshape(-1, 2)[idx], ref, TOL[np.float64], f"config4 call {c}: fp64 GPU vs oracle, sampled")
    assert not torch.equal(outs[0], outs[9])       # the positions really moved between calls


# ------------------------------------------------------------------------------------- edge shapes
def _blobs(rng, nves, npts):
    X = rng.normal(size=(nves, npts, 2)) * 0.3 + 4.0 * rng.normal(size=(nves, 1, 2))
    F = rng.normal(size=(nves, npts, 2))
    W = rng.uniform(0.5, 1.5, size=(nves, npts))
    return X, F, W


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("nves,npts", [(2, 1), (3, 2), (7, 3), (5, 31), (9, 32), (5, 33), (7, 100), (3, 129),
                                       (2, 257), (8, 128), (41, 25), (37, 128), (11, 1000), (1030, 1), (3, 2049)])
def test_edge_shapes(nves, npts, dtype):
    """Up to 1,024 points (8 x 128 is the last such shape, 41 x 25 = 1,025 the first beyond) vn_farfield is the
    single-launch kernel, above it the symmetric pair kernels; test_edge_shapes_general_path sends the small shapes
    through the pair kernels as well."""
    rng = np.random.Generator(np.random.PCG64(1000 * nves + npts))
    X, F, W = _blobs(rng, nves, npts)
    mu = 0.7
    Xo, Fo, Wo = oracle_inputs(X, F, W, dtype)
    ref = oracle.farfield(Xo, Fo, Wo, mu)
    got = gpu_farfield(X, F, W, mu, dtype)
    assert got.shape == ref.shape
    check(got, ref, TOL[dtype], f"edge shape {nves} x {npts} {np.dtype(dtype).name}")


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("nves,npts", [(2, 1), (3, 2), (7, 3), (5, 31), (9, 32), (5, 33), (7, 100), (3, 129), (2, 257), (8, 128)])
def test_edge_shapes_general_path(nves, npts, dtype):
    """vn_farfield_partial (part 0 of 1) + vn_farfield_finish IS the general path whatever the size."""
    rng = np.random.Generator(np.random.PCG64(1000 * nves + npts))
    X, F, W = _blobs(rng, nves, npts)
    mu = 0.7
    Xo, Fo, Wo = oracle_inputs(X, F, W, dtype)
    ref = oracle.farfield(Xo, Fo, Wo, mu)
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    acc, gmax = vn.vn_farfield_partial(Xd, Fd, Wd, 0, 1)
    got = vn.vn_farfield_finish(acc, gmax, nves * npts, Xd.dtype, mu)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, TOL[dtype], f"edge shape {nves} x {npts} {np.dtype(dtype).name}, general path")


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_small_path_is_deterministic_and_local(dtype):
    """The single-launch kernel: bitwise reproducible; a NaN density spoils the other vesicles' targets only
    (plain floating-point sums, no integer accumulators), a coincident pair only the two targets it touches."""
    s, W = problem(0)
    Xd, Fd, Wd = dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype)
    a = vn.vn_farfield(Xd, Fd, Wd, s.mu).clone()
    b = vn.vn_farfield(Xd, Fd, Wd, s.mu)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    Fn = s.F.copy(); Fn[3, 5, 0] = np.nan
    u = vn.vn_farfield(Xd, dev(Fn, dtype), Wd, s.mu).cpu().numpy()
    assert np.isfinite(u[3]).all() and np.isnan(u[[0, 1, 2, 4, 15]]).any(axis=(1, 2)).all()
    Xc = s.X.copy(); Xc[2, 7] = Xc[9, 1]
    u = vn.vn_farfield(dev(Xc, dtype), Fd, Wd, s.mu).cpu().numpy().reshape(-1, 2)
    bad = ~np.isfinite(u).all(1)
    assert set(np.flatnonzero(bad)) <= {2 * 32 + 7, 9 * 32 + 1}


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_single_vesicle_gives_zero(dtype):
    rng = np.random.Generator(np.random.PCG64(5))
    X, F, W = _blobs(rng, 1, 200)
    got = gpu_farfield(X, F, W, 1.0, dtype)
    assert np.all(got == 0.0)


def test_mu_and_output_overwrite():
    s, W = problem(0)
    Xd, Fd, Wd = dev(s.X, np.float64), dev(s.F, np.float64), dev(W, np.float64)
    out = torch.full_like(Xd, float("nan"))
    U1 = vn.vn_farfield(Xd, Fd, Wd, 1.0, out=out)
    U2 = vn.vn_farfield(Xd, Fd, Wd, 4.0)
    torch.cuda.synchronize()
    assert U1 is out and torch.isfinite(out).all()
    assert torch.allclose(U2 * 4.0, U1, rtol=1e-14, atol=0)


# ------------------------------------------------------------------------------------- weights (a-1)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("index", [0, 1, 3])
def test_arclength_weights_parity(index, dtype):
    s, _ = problem(index)
    Xo = np.asarray(s.X, dtype=dtype).astype(np.float64)
    ref = oracle.weights(Xo)
    got = vn.vn_arclength_weights(dev(s.X, dtype))
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, TOL[dtype], f"weights config{index} {np.dtype(dtype).name}", vec=1)


@pytest.mark.parametrize("npts", [1, 2, 3, 8, 31, 32, 33, 100, 129, 257, 1500])
def test_arclength_weights_edge_shapes(npts):
    rng = np.random.Generator(np.random.PCG64(npts))
    X = rng.normal(size=(5, npts, 2)) + 30.0
    ref = oracle.weights(X)
    got = vn.vn_arclength_weights(dev(X, np.float64))
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    if npts <= 2:
        assert np.abs(got).max() < 1e-12          # only the mean and the dropped Nyquist mode exist
    else:
        check(got, ref, 1e-12, f"weights npts={npts}", vec=1)


# ------------------------------------------------------------------------------------- whole path, host buffers
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_host_entry_point_whole_path(dtype):
    s, _ = problem(1)
    X = np.ascontiguousarray(s.X, dtype=dtype)
    F = np.ascontiguousarray(s.F, dtype=dtype)
    got = vn.vn_farfield_host(X, F, None, s.mu)                      # weights computed on the device
    Xo, Fo = X.astype(np.float64), F.astype(np.float64)
    idx = sample_targets(s.nves * s.npts, 2048, 3)
    ref = oracle.farfield_subset(Xo, Fo, oracle.weights(Xo), idx, s.mu)
    check(got.reshape(-1, 2)[idx], ref, TOL[dtype], f"host entry {np.dtype(dtype).name} (device weights)")
    # pinned torch tensors and caller-supplied weights
    Xp, Fp = torch.from_numpy(X).pin_memory(), torch.from_numpy(F).pin_memory()
    Wp = torch.from_numpy(oracle.weights(Xo).astype(dtype)).pin_memory()
    Up = torch.empty_like(Xp).pin_memory()
    vn.vn_farfield_host(Xp, Fp, Wp, s.mu, out=Up)
    check(Up.numpy().reshape(-1, 2)[idx], ref, TOL[dtype], f"host entry {np.dtype(dtype).name} (caller weights)")


# ------------------------------------------------------------------------------------- determinism, streams
def test_determinism_bitwise():
    s, W = problem(2)
    Xd, Fd, Wd = dev(s.X, np.float32), dev(s.F, np.float32), dev(W, np.float32)
    a = vn.vn_farfield(Xd, Fd, Wd).clone()
    b = vn.vn_farfield(Xd, Fd, Wd)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


def test_side_stream_behind_producer():
    """Enqueued on a non-default stream behind a producer kernel: no implicit device sync needed."""
    s, W = problem(1)
    Fd, Wd = dev(s.F, np.float64), dev(W, np.float64)
    Xh = dev(s.X, np.float64)
    ref = vn.vn_farfield(Xh, Fd, Wd)
    torch.cuda.synchronize()
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        Xd = torch.zeros_like(Xh)
        for _ in range(20):                       # producer chain on the side stream
            Xd = Xd * 0.5 + Xh * 0.5
        Xd = Xd * 0 + Xh                          # ends exactly at Xh
        got = vn.vn_farfield(Xd, Fd, Wd)
    side.synchronize()
    assert torch.equal(got, ref)


def test_launch_counter_moves():
    s, W = problem(0)
    n0 = vn.vn_launch_count()
    vn.vn_farfield(dev(s.X, np.float32), dev(s.F, np.float32), dev(W, np.float32))
    torch.cuda.synchronize()
    assert vn.vn_launch_count() >= n0 + 1          # 512 points: the single-launch kernel
    s1, W1 = problem(1)
    n1 = vn.vn_launch_count()
    vn.vn_farfield(dev(s1.X, np.float32), dev(s1.F, np.float32), dev(W1, np.float32))
    torch.cuda.synchronize()
    assert vn.vn_launch_count() >= n1 + 3          # pack, pair kernel, finish


# ------------------------------------------------------------------------------------- CUDA graphs
@pytest.mark.parametrize("path", ["farfield", "fmm"])
def test_sequence_is_graph_capturable(path):
    """Config 4's pattern (copy positions, weights, evaluation, several times on one stream) captured into a CUDA graph
    and replayed: every call only enqueues stream-ordered work (incl. its scratch), so the replay is bitwise the
    eager result."""
    s, W = problem(1)
    rng = np.random.Generator(np.random.PCG64(11))
    seq = [dev(s.X + 1e-3 * rng.standard_normal(s.X.shape), np.float32) for _ in range(3)]
    Fd = dev(s.F, np.float32)
    Xd, Wd, Ud = torch.empty_like(seq[0]), torch.empty((s.nves, s.npts), dtype=torch.float32, device="cuda"), torch.empty_like(seq[0])
    outs = [torch.empty_like(Ud) for _ in seq]

    def run():
        for x, o in zip(seq, outs):
            Xd.copy_(x)
            vn.vn_arclength_weights(Xd, out=Wd)
            if path == "farfield":
                vn.vn_farfield(Xd, Fd, Wd, s.mu, out=Ud)
            else:
                vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, 12, out=Ud)
            o.copy_(Ud)

    run()                                               # eager: also performs every lazy initialisation
    torch.cuda.synchronize()
    eager = [o.clone() for o in outs]
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    g = torch.cuda.CUDAGraph()
    with torch.cuda.stream(side):
        run()                                           # warm the side stream
        side.synchronize()
        with torch.cuda.graph(g, stream=side):
            run()
    for o in outs:
        o.zero_()
    g.replay()
    torch.cuda.synchronize()
    for a, b in zip(eager, outs):
        assert torch.equal(a, b)


# ------------------------------------------------------------------------------------- degenerate inputs (reading A5)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("call", ["farfield", "fmm"])
def test_coincident_points_and_nans_stay_local(call, dtype):
    """A coincident cross-vesicle pair (precondition violation) and a NaN density may spoil the targets they touch,
    nothing else: no hang, no fault, every other target keeps its value."""
    s, W = problem(1)
    X, F = s.X.copy(), s.F.copy()
    X[5, 7] = X[200, 3]                                   # point (5,7) now coincides with point (200,3)
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    fn = (lambda f: vn.vn_farfield(Xd, f, Wd, s.mu)) if call == "farfield" else (lambda f: vn.vn_farfield_fmm(Xd, f, Wd, s.mu, 14 if dtype == np.float32 else 38))
    got = fn(Fd).cpu().numpy()
    torch.cuda.synchronize()
    Xo, Fo, Wo = oracle_inputs(X, F, W, dtype)
    idx = np.setdiff1d(sample_targets(s.nves * s.npts, 1500, 17), [5 * s.npts + 7, 200 * s.npts + 3])
    ref = oracle.farfield_subset(Xo, Fo, Wo, idx, s.mu)
    check(got.reshape(-1, 2)[idx], ref, TOL[dtype], f"coincident pair elsewhere, {call} {np.dtype(dtype).name}",
          c_max=2.0 if call == "fmm" else 1.0)          # truncation error point-wise: tests/test_next_rows_gpu.py FMM_C
    # a NaN density at one source poisons every target of the other vesicles (that is the sum's meaning); the exact
    # path answers NaN everywhere (documented: its integer accumulators cannot carry NaN point by point)
    Fn = F.copy(); Fn[9, 0, 0] = np.nan
    gotn = fn(dev(Fn, dtype)).cpu().numpy()
    torch.cuda.synchronize()
    assert np.isnan(gotn[10]).all()
    if call == "farfield":
        assert np.isnan(gotn).all()


def test_two_streams_interleaved():
    """Calls enqueued alternately on two streams (different problems, different entry points): scratch is
    stream-ordered per call, so the results equal the ones computed one after the other."""
    s1, W1 = problem(1)
    s0, W0 = problem(0)
    a = [dev(s1.X, np.float32), dev(s1.F, np.float32), dev(W1, np.float32)]
    b = [dev(s0.X, np.float64), dev(s0.F, np.float64), dev(W0, np.float64)]
    ref_a = vn.vn_farfield(*a, s1.mu).clone()
    ref_b = vn.vn_farfield(*b, s0.mu).clone()
    ref_f = vn.vn_farfield_fmm(*a, s1.mu, 12).clone()
    torch.cuda.synchronize()
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs = []
    for _ in range(4):
        with torch.cuda.stream(st1):
            ua = vn.vn_farfield(*a, s1.mu)
            uf = vn.vn_farfield_fmm(*a, s1.mu, 12)
        with torch.cuda.stream(st2):
            ub = vn.vn_farfield(*b, s0.mu)
        outs.append((ua, ub, uf))
    torch.cuda.synchronize()
    for ua, ub, uf in outs:
        assert torch.equal(ua, ref_a) and torch.equal(ub, ref_b) and torch.equal(uf, ref_f)


# ------------------------------------------------------------------------------------- one suspension over several GPUs (section 8e)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("index,nparts", [(0, 2), (1, 2), (1, 3), (2, 8)])
def test_partial_accumulators_reproduce_farfield_bitwise(index, nparts, dtype):
    """The multi-GPU split on one device: the raw fixed-point accumulators of parts 0 .. nparts-1 (what each GPU
    would compute), added as integers (what the reduce-scatter does), finished on two vesicle ranges (what each
    GPU does with its shard) give bit for bit the result of vn_farfield."""
    s, W = problem(index)
    Xd, Fd, Wd = dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype)
    ref = vn.vn_farfield(Xd, Fd, Wd, s.mu)
    small = s.nves * s.npts <= 1024            # vn_farfield is then the single-launch kernel, not the pair kernels
    total, gmax0 = None, None
    for part in range(nparts):
        acc, gmax = vn.vn_farfield_partial(Xd, Fd, Wd, part, nparts)
        assert acc.abs().sum().item() != 0 or index == 0            # every part has work (config 0: a handful of blocks)
        total = acc.clone() if total is None else total + acc
        gmax0 = gmax.clone() if gmax0 is None else gmax0
        assert torch.equal(gmax, gmax0)                              # every device packs all sources: same scale
    P, words = s.nves * s.npts, vn.acc_words(Xd.dtype)
    k = (s.nves // 3) * s.npts                                       # two shards of different sizes
    lo = vn.vn_farfield_finish(total[:k * words], gmax0, P, Xd.dtype, s.mu)
    hi = vn.vn_farfield_finish(total[k * words:], gmax0, P, Xd.dtype, s.mu)
    torch.cuda.synchronize()
    # nparts = 1 is the single-device evaluation by the pair kernels
    acc, gmax = vn.vn_farfield_partial(Xd, Fd, Wd, 0, 1)
    assert torch.equal(acc, total)
    one = vn.vn_farfield_finish(acc, gmax, P, Xd.dtype, s.mu).view_as(ref)
    assert torch.equal(torch.cat([lo, hi]).view_as(ref), one)
    if small:
        check(one.cpu().numpy(), ref.cpu().numpy(), TOL[dtype], f"pair kernels vs single-launch kernel config{index} {np.dtype(dtype).name}")
    else:
        assert torch.equal(one, ref)


def test_sharded_farfield_single_process_equals_farfield():
    """multi.sharded_farfield_gpu with world = 1 (no process group) is the plain call."""
    from paper_2606_25569_b200 import multi
    s, W = problem(1)
    Xd, Fd, Wd = dev(s.X, np.float32), dev(s.F, np.float32), dev(W, np.float32)
    U = multi.sharded_farfield_gpu(vn, Xd, Fd, Wd, s.nves, s.mu, 0, 1)
    ref = vn.vn_farfield(Xd, Fd, Wd, s.mu)
    torch.cuda.synchronize()
    assert torch.equal(U, ref)


# ------------------------------------------------------------------------------------- ring self-check (stands in for racecheck / initcheck)
@pytest.mark.parametrize("dtype", [np.float32, np.float64])
@pytest.mark.parametrize("case", ["config1", "config2", "3x129", "7x100", "2x257", "11x1000", "1030x1", "3x2049"])
def test_ring_selfcheck_is_clean(case, dtype):
    """The verification build of the pair kernels compares every record a warp reads from the shared-memory ring with
    its original in global memory (a stage refilled too early or read too early would differ) on scratch that was
    filled with 0xFF bytes: zero mismatches, and bit for bit the result of the production kernel."""
    if case.startswith("config"):
        s, W = problem(int(case[-1]))
        X, F, mu = s.X, s.F, s.mu
    else:
        nves, npts = (int(t) for t in case.split("x"))
        rng = np.random.Generator(np.random.PCG64(1000 * nves + npts))
        X, F, W = _blobs(rng, nves, npts)
        mu = 0.7
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    U, bad = vn.vn_selfcheck(Xd, Fd, Wd, mu)
    assert bad == 0
    acc, gmax = vn.vn_farfield_partial(Xd, Fd, Wd, 0, 1)           # the production pair kernel, whatever the size
    ref = vn.vn_farfield_finish(acc, gmax, X.shape[0] * X.shape[1], Xd.dtype, mu).view_as(U)
    torch.cuda.synchronize()
    assert torch.equal(U, ref)


def test_prepared_calls_equal_the_plain_binding():
    """prepare_arclength_weights / prepare_farfield marshal once; every call must be the plain binding's result, on
    the current stream and on another one."""
    s, _ = problem(1)
    X = dev(s.X, np.float32)
    F = dev(s.F, np.float32)
    W = torch.empty(X.shape[:2], dtype=X.dtype, device=X.device)
    U = torch.empty_like(X)
    w = vn.prepare_arclength_weights(X, W)
    f = vn.prepare_farfield(X, F, W, U, s.mu)
    assert w() is W and f() is U
    torch.cuda.synchronize()
    W_ref = vn.vn_arclength_weights(X)
    U_ref = vn.vn_farfield(X, F, W_ref, s.mu)
    torch.cuda.synchronize()
    assert torch.equal(W, W_ref) and torch.equal(U, U_ref)
    side = torch.cuda.Stream()
    U.zero_()
    torch.cuda.synchronize()
    with torch.cuda.stream(side):
        w()
        f()
    side.synchronize()
    assert torch.equal(U, U_ref)
    with pytest.raises(ValueError):
        vn.prepare_farfield(X, F, W[:, :-1].contiguous(), U)
    U2 = torch.empty_like(X)
    m = vn.prepare_farfield_fmm(X, F, W, U2, s.mu, 14)
    assert m() is U2
    ref = vn.vn_farfield_fmm(X, F, W, s.mu, 14)
    torch.cuda.synchronize()
    assert torch.equal(U2, ref)
