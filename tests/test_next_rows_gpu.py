"""Parity of the NEXT rows (DESIGN.md f-1 near-field mask variant, f-2 elastic force, f-3 redistribution, f-4 free
targets, f-4b fast multipole evaluation) with the oracle
(run on the B200 box: pytest -m gpu).  Every call goes through the C-ABI library via the binding.

Index work (the near relation) must match the oracle exactly; the decision d^2 <= h^2 is taken in
double by the kernel and in long double by the oracle on the same stored values, and every test
checks that no pair sits within 1e-9 (relative) of the threshold, so that the comparison is
meaningful.  Floating point: rel-L2 <= 1e-12 (fp64), <= 2e-5 (fp32) as for vn_farfield."""
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


def stored(a, dtype):
    """What the GPU sees, promoted to double."""
    return np.asarray(a, dtype=dtype).astype(np.float64)


def crowded(index, shrink):
    """Config `index` with the vesicle centres pulled together by `shrink` (shapes unchanged): gaps
    fall below the arclength spacing, so many points get near vesicles."""
    key = (index, shrink)
    if key not in _cache:
        s = inputs.config(index)
        c = s.X.mean(1, keepdims=True)
        X = (s.X - c) + c * shrink
        _cache[key] = (X, s.F, oracle.weights(X), s.mu)
    return _cache[key]


def three_circles(npts=16):
    """Three unit circles on a triangle of side 2.05: points facing the middle are near TWO vesicles."""
    al = 2 * np.pi * np.arange(npts) / npts
    body = np.stack([np.cos(al), np.sin(al)], -1)
    cen = np.array([[0.0, 0.0], [2.05, 0.0], [1.025, 1.7753]])
    X = body[None] + cen[:, None, :]
    rng = np.random.Generator(np.random.PCG64(77))
    F = rng.normal(size=X.shape)
    return X, F, oracle.weights(X), 0.9


def csr_to_dense(ptr, ves, nves):
    P = len(ptr) - 1
    dense = np.zeros((P, nves), dtype=np.uint8)
    rows = np.repeat(np.arange(P), np.diff(ptr))
    dense[rows, ves] = 1
    return dense


def margin_ok(X, W, near_rows, idx):
    """No (target, vesicle) pair within 1e-9 relative of the threshold d^2 = h^2."""
    nves, npts, _ = X.shape
    P = X.reshape(-1, 2)
    h2 = W.max(1) ** 2
    for q, t in enumerate(idx):
        cand = np.flatnonzero(near_rows[q])
        for vp in cand:
            d2 = ((P[t] - X[vp]) ** 2).sum(1).min()
            if abs(d2 - h2[vp]) <= 1e-9 * h2[vp]:
                return False
    return True


def gpu_near(X, W, dtype):
    ptr, ves = vn.vn_near_pairs(dev(X, dtype), dev(W, dtype))
    torch.cuda.synchronize()
    return ptr.cpu().numpy(), ves.cpu().numpy()


# ------------------------------------------------------------------------------------- near relation (index work: exact)
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("case", ["three_circles", "config0", "config1", "crowded1"])
def test_near_pairs_exact(case, dtype):
    if case == "three_circles":
        X, F, W, mu = three_circles()
    elif case == "config0":
        s = inputs.config(0); X, W = s.X, oracle.weights(s.X)
    elif case == "config1":
        s = inputs.config(1); X, W = s.X, oracle.weights(s.X)
    else:
        X, F, W, mu = crowded(1, 0.94)
    Xo, Wo = stored(X, dtype), stored(W, dtype)
    ref = oracle.near_mask(Xo, Wo)
    nves, npts, _ = X.shape
    assert margin_ok(Xo, Wo, ref, np.arange(nves * npts))
    ptr, ves = gpu_near(X, W, dtype)
    assert ptr[0] == 0 and ptr[-1] == len(ves) == ref.sum() and np.all(np.diff(ptr) >= 0)
    got = csr_to_dense(ptr, ves, nves)
    assert np.array_equal(got, ref)
    for t in np.flatnonzero(np.diff(ptr) > 1):                 # ascending vesicle order inside a row
        assert np.all(np.diff(ves[ptr[t]:ptr[t + 1]]) > 0)
    if case == "three_circles":
        assert np.diff(ptr).max() == 2
    if case == "crowded1":
        assert ref.sum() > 300
    print(f"{case} {np.dtype(dtype).name}: {ref.sum()} near pairs")


def test_near_pairs_capacity_and_count_only():
    X, F, W, mu = crowded(1, 0.94)
    Xd, Wd = dev(X, np.float64), dev(W, np.float64)
    P = X.shape[0] * X.shape[1]
    ptr_full, ves_full = vn.vn_near_pairs(Xd, Wd)
    n = ves_full.numel()
    # a too-small buffer: the pointer array is still complete, only the first `capacity` entries are written
    small = torch.full((n + 16,), -7, dtype=torch.int32, device="cuda")
    ptr = torch.empty(P + 1, dtype=torch.int64, device="cuda")
    rc = vn.lib().vn_near_pairs(Xd.data_ptr(), Wd.data_ptr(), X.shape[0], X.shape[1], ptr.data_ptr(),
                                small.data_ptr(), n // 2, vn.VN_F64, None)
    torch.cuda.synchronize()
    assert rc == vn.VN_OK and torch.equal(ptr, ptr_full)
    assert torch.equal(small[:n // 2], ves_full[:n // 2]) and bool((small[n // 2:] == -7).all())


@pytest.mark.parametrize("nves,npts", [(2, 1), (5, 3), (9, 31), (4, 129), (3, 300), (130, 7), (300, 2)])
def test_near_pairs_edge_shapes(nves, npts):
    rng = np.random.Generator(np.random.PCG64(31 * nves + npts))
    X = rng.normal(size=(nves, npts, 2)) * 0.3 + 1.5 * rng.normal(size=(nves, 1, 2))
    W = rng.uniform(0.02, 0.25, size=(nves, npts))
    ref = oracle.near_mask(X, W)
    assert margin_ok(X, W, ref, np.arange(nves * npts))
    ptr, ves = gpu_near(X, W, np.float64)
    assert np.array_equal(csr_to_dense(ptr, ves, nves), ref)
    assert ref.sum() > 0 or nves * npts < 1000          # the larger cases all contain near pairs


def test_near_pairs_large_sampled():
    """Config 3 (2,000 x 128): the oracle checks 2,048 sampled rows; the total count is checked against
    the relation's own CSR invariants."""
    s = inputs.config(3)
    W = oracle.weights(s.X)
    P = s.nves * s.npts
    rng = np.random.Generator(np.random.PCG64(260625569 + 200))
    ptr, ves = gpu_near(s.X, W, np.float32)
    Xo, Wo = stored(s.X, np.float32), stored(W, np.float32)
    hot = np.flatnonzero(np.diff(ptr) > 0)
    idx = np.unique(np.concatenate([rng.choice(P, size=1536, replace=False), hot[:512]]))
    ref = oracle.near_mask_subset(Xo, Wo, idx)
    assert margin_ok(Xo, Wo, ref, idx)
    got = csr_to_dense(ptr, ves, s.nves)[idx] if P * s.nves <= 1 << 29 else None
    if got is None:
        got = np.zeros_like(ref)
        for q, t in enumerate(idx):
            got[q, ves[ptr[t]:ptr[t + 1]]] = 1
    assert np.array_equal(got, ref)
    assert ves.min() >= 0 and ves.max() < s.nves and np.all(ves != np.repeat(np.arange(P), np.diff(ptr)) // s.npts)
    print(f"config3: {len(ves)} near pairs, {len(hot)} points with a near vesicle")


# ------------------------------------------------------------------------------------- masked sum
@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("case", ["three_circles", "crowded1"])
def test_farfield_masked_full_parity(case, dtype):
    X, F, W, mu = three_circles() if case == "three_circles" else crowded(1, 0.94)
    Xo, Fo, Wo = stored(X, dtype), stored(F, dtype), stored(W, dtype)
    near = oracle.near_mask(Xo, Wo)
    ref = oracle.farfield_masked(Xo, Fo, Wo, near, mu)
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    ptr, ves = vn.vn_near_pairs(Xd, Wd)
    got = vn.vn_farfield_masked(Xd, Fd, Wd, ptr, ves, mu)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    rows = near.sum(1) > 0                                           # the corrected targets on their own
    check(got, ref, TOL[dtype], f"masked {case} {np.dtype(dtype).name}")
    check(got.reshape(-1, 2)[rows], ref.reshape(-1, 2)[rows], TOL[dtype], f"masked {case} {np.dtype(dtype).name}, corrected rows only")
    # the mask matters: the unmasked sum differs on those rows by far more than the tolerance
    full = oracle.farfield(Xo, Fo, Wo, mu).reshape(-1, 2)
    assert rel_l2(full[rows], ref.reshape(-1, 2)[rows]) > 1e3 * TOL[dtype]


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_farfield_masked_empty_relation_equals_plain(dtype):
    s = inputs.config(0)
    W = oracle.weights(s.X)
    Xd, Fd, Wd = dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype)
    ptr, ves = vn.vn_near_pairs(Xd, Wd)
    assert ves.numel() == 0
    a = vn.vn_farfield_masked(Xd, Fd, Wd, ptr, ves, s.mu)
    acc, gmax = vn.vn_farfield_partial(Xd, Fd, Wd, 0, 1)         # the pair kernels (512 points: vn_farfield itself takes
    b = vn.vn_farfield_finish(acc, gmax, s.nves * s.npts, Xd.dtype, s.mu).view_as(a)   # the single-launch kernel)
    torch.cuda.synchronize()
    assert torch.equal(a, b)
    check(a.cpu().numpy(), vn.vn_farfield(Xd, Fd, Wd, s.mu).cpu().numpy(), TOL[dtype], f"masked with an empty relation vs vn_farfield {np.dtype(dtype).name}")


@pytest.mark.parametrize("dtype", [np.float32, np.float64])
def test_farfield_masked_large_sampled(dtype):
    """Config 3 pulled together by 3 %: thousands of near pairs; oracle on sampled targets, half of
    them rows that carry a correction."""
    X, F, W, mu = crowded(3, 0.97)
    nves, npts, _ = X.shape
    P = nves * npts
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    ptr, ves = vn.vn_near_pairs(Xd, Wd)
    got = vn.vn_farfield_masked(Xd, Fd, Wd, ptr, ves, mu)
    torch.cuda.synchronize()
    ptr_h = ptr.cpu().numpy()
    hot = np.flatnonzero(np.diff(ptr_h) > 0)
    rng = np.random.Generator(np.random.PCG64(260625569 + 300))
    idx = np.unique(np.concatenate([rng.choice(P, size=1024, replace=False),
                                    rng.choice(hot, size=min(1024, len(hot)), replace=False)]))
    Xo, Fo, Wo = stored(X, dtype), stored(F, dtype), stored(W, dtype)
    rows = oracle.near_mask_subset(Xo, Wo, idx)
    ref = oracle.farfield_masked_subset(Xo, Fo, Wo, idx, rows, mu)
    check(got.cpu().numpy().reshape(-1, 2)[idx], ref, TOL[dtype], f"masked config3 x0.97 {np.dtype(dtype).name}, {len(hot)} corrected points, sampled")
    assert len(hot) > 1000


def test_farfield_masked_deterministic():
    X, F, W, mu = crowded(1, 0.94)
    Xd, Fd, Wd = dev(X, np.float32), dev(F, np.float32), dev(W, np.float32)
    ptr, ves = vn.vn_near_pairs(Xd, Wd)
    a = vn.vn_farfield_masked(Xd, Fd, Wd, ptr, ves, mu).clone()
    b = vn.vn_farfield_masked(Xd, Fd, Wd, ptr, ves, mu)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


# ------------------------------------------------------------------------------------- free targets
def grid_targets(X, n, seed, keep_away=0.25):
    """Random points of the suspension's bounding box that stay `keep_away` from every membrane point."""
    from scipy.spatial import cKDTree
    P = X.reshape(-1, 2)
    rng = np.random.Generator(np.random.PCG64(seed))
    lo, hi = P.min(0) - 1.0, P.max(0) + 1.0
    xt = rng.uniform(lo, hi, size=(3 * n, 2))
    d, _ = cKDTree(P).query(xt)
    return xt[d >= keep_away][:n]


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("index,nt", [(0, 1), (0, 777), (1, 5000)])
def test_farfield_targets_parity(index, nt, dtype):
    s = inputs.config(index)
    W = oracle.weights(s.X)
    xt = grid_targets(s.X, nt, 900 + index)
    assert len(xt) == nt
    ref = oracle.farfield_targets(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), stored(xt, dtype), s.mu)
    got = vn.vn_farfield_targets(dev(xt, dtype), dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, TOL[dtype], f"targets config{index} nt={nt} {np.dtype(dtype).name}")


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_farfield_targets_large_sampled(dtype):
    """Config 3 sources, 100,000 free targets (several target blocks and a ragged tail), oracle on 1,500 of them."""
    s = inputs.config(3)
    W = oracle.weights(s.X)
    xt = grid_targets(s.X, 100_000, 903)
    got = vn.vn_farfield_targets(dev(xt, dtype), dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu)
    torch.cuda.synchronize()
    rng = np.random.Generator(np.random.PCG64(904))
    idx = np.unique(np.concatenate([[0, 1023, 1024, len(xt) - 1], rng.choice(len(xt), size=1500, replace=False)]))
    ref = oracle.farfield_targets(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), stored(xt, dtype)[idx], s.mu)
    check(got.cpu().numpy()[idx], ref, TOL[dtype], f"targets config3 nt={len(xt)} {np.dtype(dtype).name}, sampled")


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_farfield_targets_on_a_membrane_free_vesicle_equals_farfield(dtype):
    """Targets = the points of a force-free extra vesicle: vn_farfield's value there (own vesicle
    excluded, and it carries no force anyway) equals the free-target value."""
    s = inputs.config(0)
    X = np.concatenate([s.X, s.X[:1] + np.array([1.5, 1.5])])     # a 17th ellipse between grid rows
    F = np.concatenate([s.F, np.zeros_like(s.F[:1])])
    W = oracle.weights(X)
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    a = vn.vn_farfield(Xd, Fd, Wd, s.mu)[-1]
    # sources for the free-target call: the 16 force-carrying vesicles only (a target must not coincide
    # with a source point)
    b = vn.vn_farfield_targets(Xd[-1].clone(), Xd[:-1].contiguous(), Fd[:-1].contiguous(), Wd[:-1].contiguous(), s.mu)
    torch.cuda.synchronize()
    check(b.cpu().numpy(), a.cpu().numpy(), TOL[dtype], f"targets on a force-free vesicle vs farfield {np.dtype(dtype).name}")


def test_farfield_targets_empty():
    s = inputs.config(0)
    W = oracle.weights(s.X)
    xt = torch.empty((0, 2), dtype=torch.float64, device="cuda")
    out = vn.vn_farfield_targets(xt, dev(s.X, np.float64), dev(s.F, np.float64), dev(W, np.float64), s.mu)
    assert out.shape == (0, 2)


# ------------------------------------------------------------------------------------- elastic force (row f-2)
def force_tol(X, sig, kb, dtype):
    """Empirical conditioning of f = -kappa_b X_ssss + (sigma X_s)_s at this input (the operator is a fourth spectral
    derivative, so north_star's 1e-12 -- stated for vn_farfield -- does not apply unchanged): the ORACLE is evaluated
    on X and on X with every vesicle-centred coordinate multiplied by (1 + 2 eps r), r = +-1 at random,
    eps = 2^-53; the relative L2 change is what one rounding of the input costs.  The kernel differentiates
    differences to the vesicle's first point in double, i.e. it rounds numbers of the vesicle's size, hence the
    centred perturbation.  Allowed: 8 x that change (+ 1e-14 for tiny npts; + 2^-23 for rounding the result to
    float).  At npts = 128 this is about 2e-11 (the bound used in round 1, 64 eps (npts/2)^4, was 2.4e-7)."""
    Xo, so = stored(X, dtype), stored(sig, dtype)
    rng = np.random.Generator(np.random.PCG64(12345))
    c = Xo.mean(1, keepdims=True)
    Xp = c + (Xo - c) * (1.0 + 2.0 ** -52 * rng.choice([-1.0, 1.0], size=Xo.shape))
    est = rel_l2(oracle.elastic_force(Xp, so, kb), oracle.elastic_force(Xo, so, kb))
    return 8.0 * est + 1e-14 + (2.0 ** -23 if dtype == np.float32 else 0.0)


def tension(nves, npts, seed):
    rng = np.random.Generator(np.random.PCG64(seed))
    al = 2 * np.pi * np.arange(npts) / npts
    sig = np.ones((nves, npts))
    for k in range(1, 9):
        sig += rng.normal(size=(nves, 1)) / k ** 2 * np.cos(k * al + rng.uniform(0, 2 * np.pi, size=(nves, 1)))
    return sig


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("index", [0, 1])
def test_elastic_force_parity(index, dtype):
    s = inputs.config(index)
    sig = tension(s.nves, s.npts, 40 + index)
    kb = 0.7
    ref = oracle.elastic_force(stored(s.X, dtype), stored(sig, dtype), kb)
    got = vn.vn_elastic_force(dev(s.X, dtype), dev(sig, dtype), kb)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, force_tol(s.X, sig, kb, dtype), f"elastic force config{index} {np.dtype(dtype).name}", c_max=4.0)


@pytest.mark.parametrize("npts", [3, 8, 31, 32, 33, 100, 129, 257, 1024])
def test_elastic_force_edge_shapes(npts):
    rng = np.random.Generator(np.random.PCG64(npts))
    al = 2 * np.pi * np.arange(npts) / npts
    r = 1.0 + 0.2 * np.cos(2 * al + rng.uniform(0, 6.28, size=(5, 1)))
    X = np.stack([r * np.cos(al), 0.7 * r * np.sin(al)], -1) + 10.0 * rng.normal(size=(5, 1, 2))
    sig = tension(5, npts, npts)
    ref = oracle.elastic_force(X, sig, 1.3)
    got = vn.vn_elastic_force(dev(X, np.float64), dev(sig, np.float64), 1.3)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, force_tol(X, sig, 1.3, np.float64), f"elastic force npts={npts}", c_max=4.0)


def test_elastic_force_rejects_long_vesicles_and_feeds_farfield():
    s = inputs.config(0)
    with pytest.raises(vn.VesnetError):
        vn.vn_elastic_force(torch.zeros((1, 1025, 2), device="cuda"), torch.zeros((1, 1025), device="cuda"))
    # the producer feeds the consumer on one stream: F = elastic force, U = far field of F
    Xd = dev(s.X, np.float64)
    sig = dev(tension(s.nves, s.npts, 7), np.float64)
    Wd = vn.vn_arclength_weights(Xd)
    Fd = vn.vn_elastic_force(Xd, sig, 0.5)
    Ud = vn.vn_farfield(Xd, Fd, Wd, s.mu)
    torch.cuda.synchronize()
    Fo = oracle.elastic_force(s.X, sig.cpu().numpy(), 0.5)
    ref = oracle.farfield(s.X, Fo, oracle.weights(s.X), s.mu)
    check(Ud.cpu().numpy(), ref, 8.0 * force_tol(s.X, sig.cpu().numpy(), 0.5, np.float64), "elastic force -> farfield chain config0")


# ------------------------------------------------------------------------------------- equal-arclength redistribution (row f-3)
def shape_err(got, ref):
    """Error relative to the size of the vesicles (not to their position in the box)."""
    c = ref.mean(1, keepdims=True)
    return float(np.linalg.norm(got - ref) / np.linalg.norm(ref - c))


def shape_err_max(got, ref):
    """Largest point-wise displacement over the rms radius of the vesicles."""
    c = ref.mean(1, keepdims=True)
    return float(np.sqrt(((got - ref) ** 2).sum(-1)).max() / np.sqrt(((ref - c) ** 2).sum(-1).mean()))


def redistribute_tol(X, dtype):
    """fp64: 1e-12.  fp32: the result is rounded to float at box coordinates, 2^-24 max|X| per coordinate,
    measured here against the vesicle size; at least north_star's 2e-5."""
    if dtype == np.float64:
        return 1e-12
    size = np.sqrt(((X - X.mean(1, keepdims=True)) ** 2).sum(-1).mean())
    return max(2e-5, 2.0 ** -24 * np.abs(X).max() / size)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("index", [0, 1, 3])
def test_redistribute_parity(index, dtype):
    s = inputs.config(index)
    X = s.X if index < 3 else s.X[:500]                         # the oracle is O((6N)^2) per vesicle
    ref = oracle.redistribute(stored(X, dtype))
    got = vn.vn_redistribute_arclength(dev(X, dtype))
    torch.cuda.synchronize()
    err = shape_err(got.cpu().numpy().astype(np.float64), ref)
    err_max = shape_err_max(got.cpu().numpy().astype(np.float64), ref)
    W0, W1 = oracle.weights(stored(X, dtype)), oracle.weights(got.cpu().numpy().astype(np.float64))
    print(f"redistribute config{index} {np.dtype(dtype).name}: shape-relative L2 {err:.3e} (tolerance {redistribute_tol(X, dtype):.1e}); "
          f"max/min spacing {np.max(W0.max(1) / W0.min(1)):.3f} -> {np.max(W1.max(1) / W1.min(1)):.4f}")
    print(f"redistribute config{index} {np.dtype(dtype).name}: point-wise max {err_max:.3e}")
    assert err <= redistribute_tol(X, dtype) and err_max <= 4.0 * redistribute_tol(X, dtype)


@pytest.mark.parametrize("npts", [3, 4, 5, 8, 31, 33, 100, 129, 257, 512])
def test_redistribute_edge_shapes(npts):
    rng = np.random.Generator(np.random.PCG64(npts))
    al = 2 * np.pi * np.arange(npts) / npts
    be = al + 0.3 * np.sin(al + rng.uniform(0, 6.28, size=(4, 1)))
    r = 1.0 + (0.2 if npts >= 8 else 0.0) * np.cos(2 * be)
    X = np.stack([r * np.cos(be), 0.7 * r * np.sin(be)], -1) + 10.0 * rng.normal(size=(4, 1, 2))
    ref = oracle.redistribute(X)
    got = vn.vn_redistribute_arclength(dev(X, np.float64))
    torch.cuda.synchronize()
    assert shape_err(got.cpu().numpy(), ref) <= 1e-12 and shape_err_max(got.cpu().numpy(), ref) <= 4e-12


def test_redistribute_rejects_bad_sizes_and_chains():
    with pytest.raises(vn.VesnetError):
        vn.vn_redistribute_arclength(torch.zeros((1, 2, 2), device="cuda", dtype=torch.float64))
    with pytest.raises(vn.VesnetError):
        vn.vn_redistribute_arclength(torch.zeros((1, 513, 2), device="cuda", dtype=torch.float64))
    # redistribute -> weights -> far field on one stream equals the oracle's chain
    s = inputs.config(0)
    Xd = vn.vn_redistribute_arclength(dev(s.X, np.float64))
    Wd = vn.vn_arclength_weights(Xd)
    Ud = vn.vn_farfield(Xd, dev(s.F, np.float64), Wd, s.mu)
    torch.cuda.synchronize()
    Xo = oracle.redistribute(s.X)
    ref = oracle.farfield(Xo, s.F, oracle.weights(Xo), s.mu)
    check(Ud.cpu().numpy(), ref, 1e-12, "redistribute -> weights -> farfield chain config0")


# ------------------------------------------------------------------------------------- fast multipole method (row f-4, second half)
# vn_farfield_fmm approximates the exact sum; the oracle is still the plain direct sum.  The tolerance follows the
# truncation error of the expansions, about 0.45^p relative: p = 12 for the fp32 bar (2e-5),
# p = 38 for the fp64 bar (1e-12).  Point-wise (max-rel) the truncation error is held to FMM_C x the tolerance: the
# error of a truncated expansion is largest for the targets closest to the corner of their box, a handful of points,
# so it exceeds the L2 average by a factor of about 15 that the exact path does not have (measured at p = 12:
# rel-L2 5.6e-6, max-rel 8.4e-5 at 2,000 x 128).  The default order for fp32 storage is therefore 14, not 12: 0.45^2
# brings the point-wise error to 1.7e-5 (measured maxima: DESIGN.md section 7).
FMM_C = 2.0
@pytest.mark.parametrize("index,dtype,order", [(0, np.float64, 38), (0, np.float32, 14), (1, np.float64, 38),
                                                (1, np.float32, 14), (1, np.float64, 14)])
def test_fmm_full_parity(index, dtype, order):
    s = inputs.config(index)
    W = oracle.weights(s.X)
    ref = oracle.farfield(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), s.mu)
    got = vn.vn_farfield_fmm(dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu, order)
    torch.cuda.synchronize()
    tol = TOL[dtype] if not (dtype == np.float64 and order < 30) else 2e-5
    check(got.cpu().numpy(), ref, tol, f"fmm config{index} {np.dtype(dtype).name} p={order}", c_max=FMM_C)


@pytest.mark.parametrize("index,dtype,order,nsample", [(3, np.float32, 14, 3072), (3, np.float64, 38, 3072),
                                                      (4, np.float32, 14, 1024)])
def test_fmm_sampled_parity_large(index, dtype, order, nsample):
    s = inputs.config(index)
    W = oracle.weights(s.X)
    P = s.nves * s.npts
    rng = np.random.Generator(np.random.PCG64(260625569 + 400))
    idx = np.unique(np.concatenate([[0, 127, 128, P - 1], rng.choice(P, size=nsample, replace=False)]))
    ref = oracle.farfield_subset(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), idx, s.mu)
    got = vn.vn_farfield_fmm(dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu, order)
    torch.cuda.synchronize()
    check(got.cpu().numpy().reshape(-1, 2)[idx], ref, TOL[dtype], f"fmm config{index} {np.dtype(dtype).name} p={order} sampled", c_max=FMM_C)


def test_fmm_converges_with_order_and_agrees_with_exact_path():
    s = inputs.config(2)
    W = oracle.weights(s.X)
    Xd, Fd, Wd = dev(s.X, np.float64), dev(s.F, np.float64), dev(W, np.float64)
    exact = vn.vn_farfield(Xd, Fd, Wd, s.mu)
    errs = []
    for order in (4, 8, 16, 24, 32):
        got = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, order)
        torch.cuda.synchronize()
        errs.append(rel_l2(got.cpu().numpy(), exact.cpu().numpy()))
    print("fmm vs exact GPU path, config2, p = 4, 8, 16, 24, 32:", " ".join(f"{e:.2e}" for e in errs))
    assert all(b < 0.05 * a for a, b in zip(errs, errs[1:])) and errs[-1] < 1e-10
    # bitwise reproducible
    a = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, 12).clone()
    b = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, 12)
    torch.cuda.synchronize()
    assert torch.equal(a, b)


@pytest.mark.parametrize("nves,npts", [(2, 1), (3, 2), (7, 3), (5, 33), (3, 129), (37, 128), (11, 1000), (1030, 1), (3, 2049)])
def test_fmm_edge_shapes(nves, npts):
    rng = np.random.Generator(np.random.PCG64(1000 * nves + npts))
    X = rng.normal(size=(nves, npts, 2)) * 0.3 + 4.0 * rng.normal(size=(nves, 1, 2))
    F = rng.normal(size=(nves, npts, 2))
    W = rng.uniform(0.5, 1.5, size=(nves, npts))
    ref = oracle.farfield(X, F, W, 0.7)
    got = vn.vn_farfield_fmm(dev(X, np.float64), dev(F, np.float64), dev(W, np.float64), 0.7, 40)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    check(got, ref, 1e-11, f"fmm edge shape {nves} x {npts}", c_max=FMM_C)


@pytest.mark.parametrize("order", [14, 15])
@pytest.mark.parametrize("nves,npts", [(2, 1), (3, 2), (7, 3), (5, 33), (3, 129), (37, 128), (11, 1000), (1030, 1), (3, 2049), (300, 64)])
def test_fmm_edge_shapes_single_precision(nves, npts, order):
    """The kernels only the fp32 calls run (packed direct part, half-warp P2M / M2L: q = order + 1 <= 16) on the same
    ragged shapes, at the default order and at the largest order of that path (q = 16: every lane of a half-warp
    carries a coefficient).  A structural test -- an indexing fault gives errors of order one --, so the bound is
    the fp32 tolerance times 5: random clouds put points of different vesicles closer than a suspension does."""
    rng = np.random.Generator(np.random.PCG64(1000 * nves + npts))
    X = rng.normal(size=(nves, npts, 2)) * 0.3 + 4.0 * rng.normal(size=(nves, 1, 2))
    F = rng.normal(size=(nves, npts, 2))
    W = rng.uniform(0.5, 1.5, size=(nves, npts))
    ref = oracle.farfield(stored(X, np.float32), stored(F, np.float32), stored(W, np.float32), 0.7)
    got = vn.vn_farfield_fmm(dev(X, np.float32), dev(F, np.float32), dev(W, np.float32), 0.7, order)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, 5 * TOL[np.float32], f"fmm fp32 edge shape {nves} x {npts} p={order}", c_max=FMM_C)


def test_fmm_orders_across_the_kernel_switch_single_precision():
    """Orders 13 .. 18 at config 1 in fp32: q = order + 1 <= 16 runs the half-warp kernels, above that the general ones;
    all of them must sit at the fp32 bar against the exact fp32 path, and low orders must be visibly worse."""
    s = inputs.config(1)
    W = oracle.weights(s.X)
    Xd, Fd, Wd = dev(s.X, np.float32), dev(s.F, np.float32), dev(W, np.float32)
    exact = vn.vn_farfield(Xd, Fd, Wd, s.mu).cpu().numpy()
    errs = {}
    for order in (2, 6, 13, 14, 15, 16, 17, 18):
        got = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, order)
        torch.cuda.synchronize()
        errs[order] = rel_l2(got.cpu().numpy(), exact)
    print("fmm fp32 vs exact fp32 path, config1:", " ".join(f"p={o}: {e:.2e}" for o, e in errs.items()))
    assert errs[2] > errs[6] > errs[13] and errs[2] > 1e-3
    assert all(errs[o] <= TOL[np.float32] for o in (14, 15, 16, 17, 18))


@pytest.mark.parametrize("dtype,order", [(np.float32, 14), (np.float64, 38)])
def test_fmm_calls_on_two_streams_at_once(dtype, order):
    """The multi-level M2M / L2L launches hold a grid barrier, i.e. need all their blocks resident at once; they are
    launched with the cooperative attribute, so two evaluations in flight on two streams must neither deadlock nor
    disturb each other (at p = 38 one such grid fills the device)."""
    s = inputs.config(2)
    W = oracle.weights(s.X)
    Xd, Fd, Wd = dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype)
    F2 = Fd.flip(0).contiguous()
    ref1 = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, order).clone()
    ref2 = vn.vn_farfield_fmm(Xd, F2, Wd, s.mu, order).clone()
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    out1, out2 = torch.empty_like(ref1), torch.empty_like(ref2)
    for _ in range(5):
        with torch.cuda.stream(s1):
            vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, order, out=out1)
        with torch.cuda.stream(s2):
            vn.vn_farfield_fmm(Xd, F2, Wd, s.mu, order, out=out2)
    torch.cuda.synchronize()
    assert torch.equal(out1, ref1) and torch.equal(out2, ref2)


def test_fmm_single_vesicle_gives_zero():
    rng = np.random.Generator(np.random.PCG64(5))
    X = rng.normal(size=(1, 700, 2)); F = rng.normal(size=(1, 700, 2)); W = rng.uniform(0.5, 1.5, size=(1, 700))
    got = vn.vn_farfield_fmm(dev(X, np.float64), dev(F, np.float64), dev(W, np.float64), 1.0, 30)
    torch.cuda.synchronize()
    # everything the expansions add is taken out again by the own-vesicle correction: zero up to truncation
    scale = np.abs(oracle.farfield_targets(X, F, W, X[0, :1] + 50.0)).max()
    assert np.abs(got.cpu().numpy()).max() <= 1e-9 * max(scale, 1.0) * 700


@pytest.mark.parametrize("dtype,order", [(np.float64, 38), (np.float32, 14)])
def test_fmm_masked_parity(dtype, order):
    """The paper's DirectSingleLayerIntegral in O(P): FMM + near-field mask against the masked oracle."""
    X, F, W, mu = crowded(1, 0.94)
    Xo, Fo, Wo = stored(X, dtype), stored(F, dtype), stored(W, dtype)
    near = oracle.near_mask(Xo, Wo)
    ref = oracle.farfield_masked(Xo, Fo, Wo, near, mu)
    Xd, Fd, Wd = dev(X, dtype), dev(F, dtype), dev(W, dtype)
    ptr, ves = vn.vn_near_pairs(Xd, Wd)
    got = vn.vn_farfield_fmm(Xd, Fd, Wd, mu, order, near_ptr=ptr, near_ves=ves)
    torch.cuda.synchronize()
    rows = near.sum(1) > 0
    check(got.cpu().numpy(), ref, TOL[dtype], f"fmm masked crowded1 {np.dtype(dtype).name} p={order}", c_max=FMM_C)
    check(got.cpu().numpy().reshape(-1, 2)[rows], ref.reshape(-1, 2)[rows], TOL[dtype],
          f"fmm masked crowded1 {np.dtype(dtype).name} p={order}, corrected rows", c_max=FMM_C)


@pytest.mark.parametrize("dtype,order", [(np.float64, 38), (np.float32, 14)])
@pytest.mark.parametrize("index,nt", [(0, 777), (1, 5000), (3, 100_000)])
def test_fmm_targets_parity(index, nt, dtype, order):
    s = inputs.config(index)
    W = oracle.weights(s.X)
    xt = grid_targets(s.X, nt, 900 + index)
    rng = np.random.Generator(np.random.PCG64(905))
    idx = np.arange(len(xt)) if len(xt) <= 5000 else np.unique(np.concatenate([[0, len(xt) - 1], rng.choice(len(xt), size=1500, replace=False)]))
    ref = oracle.farfield_targets(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), stored(xt, dtype)[idx], s.mu)
    got = vn.vn_farfield_targets(dev(xt, dtype), dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu, fmm_order=order)
    torch.cuda.synchronize()
    check(got.cpu().numpy()[idx], ref, TOL[dtype], f"fmm targets config{index} nt={len(xt)} {np.dtype(dtype).name} p={order}", c_max=FMM_C)


@pytest.mark.parametrize("layout", ["two_clusters", "line", "one_far_outlier"])
def test_fmm_nonuniform_layouts(layout):
    """Strongly non-uniform point distributions cost time (crowded leaves), never accuracy."""
    rng = np.random.Generator(np.random.PCG64({"two_clusters": 501, "line": 502, "one_far_outlier": 503}[layout]))
    nves, npts = 60, 64
    al = 2 * np.pi * np.arange(npts) / npts
    body = np.stack([np.cos(al), 0.5 * np.sin(al)], -1) * 0.3
    if layout == "two_clusters":
        cen = np.concatenate([rng.normal(size=(30, 2)) * 2.0, rng.normal(size=(30, 2)) * 2.0 + np.array([400.0, 250.0])])
    elif layout == "line":
        cen = np.stack([np.arange(nves) * 0.9, np.zeros(nves)], -1)
    else:
        cen = rng.normal(size=(nves, 2)) * 3.0
        cen[-1] = (5000.0, -3000.0)
    X = body[None] + cen[:, None, :]
    F = rng.normal(size=X.shape)
    W = oracle.weights(X)
    ref = oracle.farfield(X, F, W, 1.0)
    got = vn.vn_farfield_fmm(dev(X, np.float64), dev(F, np.float64), dev(W, np.float64), 1.0, 40)
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, 1e-11, f"fmm {layout}", c_max=FMM_C)


def test_fmm_four_million_points():
    """2 x 2 copies of config 4 side by side (32,000 vesicles, 4.1 M points): far beyond what the direct kernels are
    for (5.7 s per evaluation); the oracle checks 256 sampled targets."""
    s = inputs.config(4)
    Lx, Ly = s.box
    X = np.concatenate([s.X + np.array([i * (Lx + 1.0), j * (Ly + 1.0)]) for i in range(2) for j in range(2)])
    F = np.concatenate([s.F] * 4)
    W = oracle.weights(s.X)
    W = np.concatenate([W] * 4)
    nves, npts, _ = X.shape
    rng = np.random.Generator(np.random.PCG64(260625569 + 500))
    idx = rng.choice(nves * npts, size=256, replace=False)
    ref = oracle.farfield_subset(stored(X, np.float32), stored(F, np.float32), stored(W, np.float32), idx, s.mu)
    Xd, Fd, Wd = dev(X, np.float32), dev(F, np.float32), dev(W, np.float32)
    got = vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, 14)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(3):
        vn.vn_farfield_fmm(Xd, Fd, Wd, s.mu, 14, out=got)
    e1.record()
    e1.synchronize()
    print(f"fmm 32000 x 128 (4.1 M points) float32 p=14: {e0.elapsed_time(e1) / 3:.2f} ms per evaluation")
    check(got.cpu().numpy().reshape(-1, 2)[idx], ref, TOL[np.float32], "fmm 32000 x 128 float32 p=14 sampled", c_max=FMM_C)


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_fmm_default_order_meets_the_tolerance(dtype):
    s = inputs.config(1)
    W = oracle.weights(s.X)
    ref = oracle.farfield(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), s.mu)
    got = vn.vn_farfield_fmm(dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu, 0)     # order 0 = default for the precision
    torch.cuda.synchronize()
    check(got.cpu().numpy(), ref, TOL[dtype], f"fmm default order {np.dtype(dtype).name}", c_max=FMM_C)


@pytest.mark.parametrize("shift", [(1.0e4, -3.0e4), (-2.0e5, 1.0e5)])
def test_fmm_is_translation_invariant(shift):
    """The expansions work in the root square's frame, so a suspension far from the origin keeps the accuracy it
    has at the origin (the exact path is translation invariant by construction; in absolute coordinates the terms
    conj(zeta) g and z conj(Phi') would each be |z| / |r| times larger than their sum)."""
    s = inputs.config(1)
    W = oracle.weights(s.X)
    Xs = s.X + np.asarray(shift)
    ref = oracle.farfield(Xs, s.F, W, s.mu)                       # the oracle on the SHIFTED points
    got = vn.vn_farfield_fmm(dev(Xs, np.float64), dev(s.F, np.float64), dev(W, np.float64), s.mu, 38)
    got0 = vn.vn_farfield_fmm(dev(s.X, np.float64), dev(s.F, np.float64), dev(W, np.float64), s.mu, 38)
    torch.cuda.synchronize()
    e_shift, _ = check(got.cpu().numpy(), ref, 1e-12, f"fmm config1 shifted by {shift}", c_max=FMM_C)
    e_zero = rel_l2(got0.cpu().numpy(), oracle.farfield(s.X, s.F, W, s.mu))
    # moving into the root square's frame rounds once more (an ulp of the box size against gaps of 0.05): the shifted
    # run may lose a digit against the run at the origin, not the six digits |z| / |r| = 1e5 / 0.05 would cost
    print(f"fmm at the origin {e_zero:.2e}, shifted {e_shift:.2e}")
    assert e_shift <= 1e-13
    # the exact path, for comparison
    ex = vn.vn_farfield(dev(Xs, np.float64), dev(s.F, np.float64), dev(W, np.float64), s.mu)
    torch.cuda.synchronize()
    check(ex.cpu().numpy(), ref, 1e-12, f"farfield config1 shifted by {shift}")


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
def test_farfield_targets_bad_distance_stays_local(dtype):
    """A free target on top of a membrane point (precondition violation, r = 0) may spoil its own value, nothing else:
    in particular not the target that shares its packed register in the fp32 kernel (128 indices away), whose
    reciprocal is shared with it (t = rcp(a b))."""
    s = inputs.config(1)
    W = oracle.weights(s.X)
    xt = grid_targets(s.X, 2000, 911)
    hit = [300, 1700]
    xt[hit[0]] = s.X[7, 5]
    xt[hit[1]] = s.X[200, 100]
    xo = stored(xt, dtype)
    xo[hit[0]] = stored(s.X, dtype)[7, 5]                       # exactly the stored source point in the storage precision too
    xo[hit[1]] = stored(s.X, dtype)[200, 100]
    got = vn.vn_farfield_targets(dev(xo, dtype), dev(s.X, dtype), dev(s.F, dtype), dev(W, dtype), s.mu)
    torch.cuda.synchronize()
    got = got.cpu().numpy()
    keep = np.setdiff1d(np.arange(len(xt)), hit)
    assert {428, 1828} <= set(keep)                             # the register partners of the two bad targets
    ref = oracle.farfield_targets(stored(s.X, dtype), stored(s.F, dtype), stored(W, dtype), xo[keep], s.mu)
    check(got[keep], ref, TOL[dtype], f"targets with two coincident targets elsewhere {np.dtype(dtype).name}")
