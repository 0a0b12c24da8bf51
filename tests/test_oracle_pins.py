"""Pins for the oracle (CPU only).  Each test fixes the oracle against something other
than itself: a closed form, a continuous integral computed by mpmath (tests/golden/),
an identity of the Stokes kernel, a library routine (numpy.fft), or a brute-force pair
loop written independently here.  A dropped term, wrong sign, transposed index or wrong
exclusion set fails at least one of them (see test_wrong_kernels_are_caught)."""
import math
import os

import numpy as np
import pytest

import oracle

FOURPI = 4.0 * math.pi


def _load(golden_dir, name):
    rows = []
    with open(os.path.join(golden_dir, name)) as fh:
        for line in fh:
            if line.startswith("#") or not line.strip():
                continue
            rows.append([float(t) for t in line.split()])
    return np.array(rows)


def _rot(th):
    return np.array([[math.cos(th), -math.sin(th)], [math.sin(th), math.cos(th)]])


def _ellipse(a, b, n, th=0.0, c=(0.0, 0.0)):
    al = 2 * np.pi * np.arange(n) / n
    P = np.stack([a * np.cos(al), b * np.sin(al)], -1) @ _rot(th).T + np.asarray(c)
    return P, al


def _random_problem(rng, nves, npts, spread=3.0):
    """Well separated blobs of random points (not curves: the sum does not care)."""
    X = rng.normal(size=(nves, npts, 2)) * 0.3 + spread * rng.normal(size=(nves, 1, 2))
    F = rng.normal(size=(nves, npts, 2))
    W = rng.uniform(0.5, 1.5, size=(nves, npts))
    return X, F, W


# ----------------------------------------------------------------------------- kernel values
def test_point_stokeslet_closed_form(golden_dir):
    """eq 2.9 for one source: nves=2, npts=1, second vesicle carries no force."""
    for x, y, gx, gy, ex, ey in _load(golden_dir, "point_stokeslet.txt"):
        X = np.array([[[0.0, 0.0]], [[x, y]]])
        F = np.array([[[gx, gy]], [[0.0, 0.0]]])
        W = np.ones((2, 1))
        U = oracle.farfield(X, F, W, mu=1.0)
        assert np.allclose(FOURPI * U[1, 0], [ex, ey], rtol=0, atol=2e-15)
        assert np.all(U[0, 0] == 0.0)           # the only other vesicle has zero density


def test_mu_scaling_and_prefactor():
    rng = np.random.default_rng(1)
    X, F, W = _random_problem(rng, 3, 5)
    U1 = oracle.farfield(X, F, W, mu=1.0)
    U2 = oracle.farfield(X, F, W, mu=2.5)
    assert np.allclose(U2 * 2.5, U1, rtol=1e-15, atol=0)


# ----------------------------------------------------------------------------- whole operator vs exact integrals
def test_constant_density_on_circle(golden_dir):
    """Trapezoid sum vs closed form / mpmath quadrature of eq 2.8."""
    N = 64
    for R, ex, ey, x, y, cx, cy, qx, qy in _load(golden_dir, "circle_constant_density.txt"):
        src, _ = _ellipse(R, R, N)
        X = np.stack([src, np.tile([[x, y]], (N, 1))])
        F = np.stack([np.tile([[ex, ey]], (N, 1)), np.zeros((N, 2))])
        W = np.stack([np.full(N, 2 * np.pi * R / N), np.ones(N)])
        U = oracle.farfield(X, F, W)
        assert np.allclose(FOURPI * U[1, 0], [cx, cy], rtol=0, atol=5e-15)
        assert abs(cx - qx) < 1e-20 and abs(cy - qy) < 1e-20


def test_smooth_density_on_rotated_ellipse_uses_oracle_weights(golden_dir):
    """General density, general shape: oracle.weights + oracle.farfield together reproduce
    the continuous integral (spectral convergence for far targets)."""
    N = 128
    src, al = _ellipse(1.0, 0.4, N, th=0.35, c=(0.2, -0.1))
    f = np.stack([0.5 + np.cos(2 * al) - 0.3 * np.sin(al),
                  -0.2 + 0.7 * np.sin(3 * al) + 0.4 * np.cos(al)], -1)
    rows = _load(golden_dir, "ellipse_smooth_density.txt")
    tg = np.zeros((N, 2)); tg[:] = rows[0, :2]; tg[:len(rows)] = rows[:, :2]
    X = np.stack([src, tg])
    F = np.stack([f, np.zeros((N, 2))])
    W = oracle.weights(X)
    W[1] = 1.0
    U = oracle.farfield(X, F, W)
    assert np.allclose(FOURPI * U[1, :len(rows)], rows[:, 2:4], rtol=0, atol=3e-14)


@pytest.mark.parametrize("a,b", [(1.0, 1.0), (1.0, 0.4)])
def test_single_layer_of_normal_vanishes_outside(a, b):
    """S[n](x) = 0 outside a closed curve (Stokeslet is divergence free).  With the paper's
    printed '+log' and no identity the residual is O(0.1): this pins reading A1."""
    N = 128
    src, al = _ellipse(a, b, N, th=0.6, c=(0.3, 0.2))
    tx, ty = -a * np.sin(al), b * np.cos(al)                     # dX/dalpha in the body frame
    sa = np.sqrt(tx ** 2 + ty ** 2)
    nrm = np.stack([ty / sa, -tx / sa], -1) @ _rot(0.6).T        # outward unit normal
    tg, _ = _ellipse(a + 1.0, b + 1.0, N, th=0.6, c=(0.3, 0.2))   # targets at distance >= 1
    X = np.stack([src, tg]); F = np.stack([nrm, np.zeros((N, 2))])
    W = np.stack([sa * 2 * np.pi / N, np.ones(N)])
    U = oracle.farfield(X, F, W)
    assert np.abs(U[1]).max() < 1e-15


def test_single_layer_of_normal_spectral_decay_N32():
    """N=32: residual decays with distance like the trapezoid rule's (R/rho)^N."""
    N = 32
    src, al = _ellipse(1.0, 1.0, N)
    res = []
    for d in (0.5, 1.0, 2.0):
        tg, _ = _ellipse(1.0 + d, 1.0 + d, N)
        X = np.stack([src, tg]); F = np.stack([src.copy(), np.zeros((N, 2))])
        W = np.stack([np.full(N, 2 * np.pi / N), np.ones(N)])
        res.append(np.abs(oracle.farfield(X, F, W)[1]).max())
    assert 1e-8 < res[0] < 1e-5 and res[1] < 1e-9 and res[2] < 1e-14


# ----------------------------------------------------------------------------- identities
def test_scaling_identity_pins_log_and_exclusion():
    """X -> sX, W -> sW  =>  U -> s [ U - ln(s)/(4 pi mu) (G_tot - G_own) ],  G_v = sum_j F W."""
    rng = np.random.default_rng(2)
    X, F, W = _random_problem(rng, 4, 6)
    s, mu = 1.7, 0.9
    U = oracle.farfield(X, F, W, mu)
    Us = oracle.farfield(s * X, F, s * W, mu)
    G = (F * W[..., None]).sum(1)                                 # [nves, 2]
    corr = (G.sum(0)[None, :] - G)[:, None, :]                    # other vesicles only
    assert np.allclose(Us, s * (U - math.log(s) / (FOURPI * mu) * corr), rtol=0, atol=1e-14)


def test_adjoint_identity():
    """<a, S g> = <S a, g> with W = 1: G(r) = G(-r) = G^T and a symmetric exclusion set."""
    rng = np.random.default_rng(3)
    X, _, _ = _random_problem(rng, 5, 7)
    a = rng.normal(size=X.shape); g = rng.normal(size=X.shape)
    W = np.ones(X.shape[:2])
    lhs = (a * oracle.farfield(X, g, W)).sum()
    rhs = (oracle.farfield(X, a, W) * g).sum()
    assert abs(lhs - rhs) < 1e-13 * max(1.0, abs(lhs))


def test_brute_force_symmetric_pair_sum():
    """Independent loop over unordered cross-vesicle pairs, K built once per pair and
    scattered both ways (different loop structure, numpy float64)."""
    rng = np.random.default_rng(4)
    nves, npts = 4, 5
    X, F, W = _random_problem(rng, nves, npts)
    g = (F * W[..., None]).reshape(-1, 2); P = X.reshape(-1, 2)
    ves = np.repeat(np.arange(nves), npts)
    U = np.zeros_like(P)
    for i in range(len(P)):
        for j in range(i + 1, len(P)):
            if ves[i] == ves[j]:
                continue
            r = P[i] - P[j]
            K = -0.5 * math.log(r @ r) * np.eye(2) + np.outer(r, r) / (r @ r)
            U[i] += K @ g[j]
            U[j] += K @ g[i]
    U /= FOURPI
    assert np.allclose(oracle.farfield(X, F, W).reshape(-1, 2), U, rtol=0, atol=1e-14)


def test_translation_rotation_linearity_superposition():
    rng = np.random.default_rng(5)
    X, F, W = _random_problem(rng, 4, 6)
    U = oracle.farfield(X, F, W)
    # translation: only differences enter
    assert np.allclose(oracle.farfield(X + np.array([3.0, -2.0]), F, W), U, rtol=0, atol=1e-14)
    # rotation equivariance
    R = _rot(0.83)
    assert np.allclose(oracle.farfield(X @ R.T, F @ R.T, W), U @ R.T, rtol=0, atol=1e-14)
    # linearity in F and dependence on F, W only through F*W
    F2 = rng.normal(size=F.shape)
    assert np.allclose(oracle.farfield(X, 2 * F - 3 * F2, W),
                       2 * U - 3 * oracle.farfield(X, F2, W), rtol=0, atol=1e-13)
    assert np.allclose(oracle.farfield(X, F * W[..., None], np.ones_like(W)), U, rtol=0, atol=1e-14)
    # superposition over source vesicles: U = sum over "only vesicle s carries force"
    acc = np.zeros_like(U)
    for s in range(X.shape[0]):
        Fs = np.zeros_like(F); Fs[s] = F[s]
        Us = oracle.farfield(X, Fs, W)
        assert np.all(Us[s] == 0.0)                               # a vesicle never acts on itself
        acc += Us
    assert np.allclose(acc, U, rtol=0, atol=1e-14)


def test_permutation_equivariance():
    rng = np.random.default_rng(6)
    X, F, W = _random_problem(rng, 5, 4)
    U = oracle.farfield(X, F, W)
    pv = rng.permutation(5)
    assert np.allclose(oracle.farfield(X[pv], F[pv], W[pv]), U[pv], rtol=0, atol=1e-14)
    pp = rng.permutation(4)
    assert np.allclose(oracle.farfield(X[:, pp], F[:, pp], W[:, pp]), U[:, pp], rtol=0, atol=1e-14)


def test_single_vesicle_is_zero_and_errors():
    rng = np.random.default_rng(7)
    X, F, W = _random_problem(rng, 1, 9)
    assert np.all(oracle.farfield(X, F, W) == 0.0)
    with pytest.raises(ValueError):
        oracle.farfield(X, F, W, mu=0.0)


def test_subset_and_free_targets_agree_with_full():
    rng = np.random.default_rng(8)
    X, F, W = _random_problem(rng, 4, 6)
    U = oracle.farfield(X, F, W, mu=1.3).reshape(-1, 2)
    idx = np.array([0, 7, 23, 11])
    assert np.array_equal(oracle.farfield_subset(X, F, W, idx, mu=1.3), U[idx])
    # free targets see every vesicle: U_free(x) = sum over all; check against superposition of
    # a 5-vesicle problem whose extra vesicle holds the targets and no force
    xt = rng.normal(size=(6, 2)) * 5
    X5 = np.concatenate([X, xt[None]], 0); F5 = np.concatenate([F, np.zeros((1, 6, 2))], 0)
    W5 = np.concatenate([W, np.ones((1, 6))], 0)
    assert np.allclose(oracle.farfield_targets(X, F, W, xt, mu=1.3),
                       oracle.farfield(X5, F5, W5, mu=1.3)[4], rtol=0, atol=1e-15)


def test_wrong_kernels_are_caught():
    """The pins are sharp: the paper's printed kernel (+log, no I) and a transposed dyad
    both violate S[n] = 0 by O(0.1) on the same input where the oracle gives < 1e-15."""
    N = 128
    src, al = _ellipse(1.0, 0.4, N)
    tx, ty = -np.sin(al), 0.4 * np.cos(al)
    sa = np.hypot(tx, ty)
    g = np.stack([ty / sa, -tx / sa], -1) * (sa * 2 * np.pi / N)[:, None]
    x = np.array([1.5, 1.2])
    r = x - src; r2 = (r ** 2).sum(1)
    printed = (0.5 * np.log(r2)[:, None] * g + ((r * g).sum(1) / r2)[:, None] * r).sum(0)
    nodyad = (-0.5 * np.log(r2)[:, None] * g).sum(0)
    assert np.abs(printed).max() > 0.05 and np.abs(nodyad).max() > 0.05


# ----------------------------------------------------------------------------- weights
def test_weights_circle_and_ellipse_pointwise(golden_dir):
    for N in (32, 33, 128):
        for (a, b, th, c) in [(0.8, 0.8, 0.0, (0, 0)), (1.0, 0.4, 0.9, (2.0, -1.0))]:
            P, al = _ellipse(a, b, N, th, c)
            W = oracle.weights(P[None])[0]
            exact = (2 * np.pi / N) * np.sqrt(a * a * np.sin(al) ** 2 + b * b * np.cos(al) ** 2)
            assert np.allclose(W, exact, rtol=0, atol=2e-15)
    per = _load(golden_dir, "ellipse_perimeter.txt")[0, 0]
    P, _ = _ellipse(1.0, 0.4, 128)
    assert abs(oracle.weights(P[None]).sum() - per) < 1e-14
    P, _ = _ellipse(1.0, 0.4, 32)
    assert 1e-9 < abs(oracle.weights(P[None]).sum() - per) < 1e-6      # N=32: -4.7e-8 (not yet converged)


@pytest.mark.parametrize("N", [1, 2, 3, 8, 31, 32, 33, 100, 128, 129])
def test_weights_match_numpy_fft(N):
    """Library routine: derivative via numpy.fft with the Nyquist mode zeroed (reading A4)."""
    rng = np.random.default_rng(100 + N)
    X = rng.normal(size=(3, N, 2))
    k = np.fft.fftfreq(N, 1.0 / N)
    if N % 2 == 0:
        k[N // 2] = 0.0
    d = np.fft.ifft(1j * k[None, :, None] * np.fft.fft(X, axis=1), axis=1).real
    W, dX = oracle.weights(X, return_derivative=True)
    assert np.allclose(dX, d, rtol=0, atol=1e-12 * max(1, N))
    assert np.allclose(W, (2 * np.pi / N) * np.hypot(d[..., 0], d[..., 1]), rtol=0, atol=1e-12 * max(1, N))


def test_weights_invariances_and_circulant_form():
    rng = np.random.default_rng(9)
    N = 16
    X = rng.normal(size=(2, N, 2))
    W = oracle.weights(X)
    assert np.allclose(oracle.weights(X @ _rot(1.1).T + 4.0), W, rtol=0, atol=1e-14)
    assert np.allclose(oracle.weights(2.5 * X), 2.5 * W, rtol=0, atol=1e-14)
    # circulant differentiation matrix D_jk = 1/2 (-1)^(j-k) cot((j-k) pi / N), even N (textbook form)
    j = np.arange(N)[:, None]; k = np.arange(N)[None, :]
    with np.errstate(divide="ignore"):
        D = 0.5 * (-1.0) ** (j - k) / np.tan((j - k) * np.pi / N)
    D[np.arange(N), np.arange(N)] = 0.0
    d = np.einsum("jk,vkc->vjc", D, X)
    assert np.allclose(W, (2 * np.pi / N) * np.hypot(d[..., 0], d[..., 1]), rtol=0, atol=1e-13)


# ----------------------------------------------------------------------------- near-field mask variant
def test_near_mask_and_masked_sum():
    """Two ellipses 0.03 apart (closer than the arclength spacing) and one far away."""
    N = 32
    A, _ = _ellipse(1.0, 0.4, N, c=(0.0, 0.0))
    B, _ = _ellipse(1.0, 0.4, N, c=(0.0, 0.83))          # gap 0.03 at the minor-axis tips
    C, _ = _ellipse(1.0, 0.4, N, c=(6.0, 0.0))
    X = np.stack([A, B, C])
    W = oracle.weights(X)
    rng = np.random.default_rng(10)
    F = rng.normal(size=X.shape)
    near = oracle.near_mask(X, W)
    h = W.max(1)
    # brute-force definition: dist(point, vesicle) <= arclength spacing of that vesicle
    P = X.reshape(-1, 2)
    for t in range(3 * N):
        for vp in range(3):
            d = np.sqrt(((P[t] - X[vp]) ** 2).sum(1)).min()
            assert near[t, vp] == (1 if (vp != t // N and d <= h[vp]) else 0)
    assert near[:N, 1].any() and near[N:2 * N, 0].any() and not near[:, 2].any() and not near[2 * N:].any()
    # masked sum = full sum minus the masked vesicles' contributions (superposition)
    U = oracle.farfield(X, F, W)
    Um = oracle.farfield_masked(X, F, W, near)
    FB = np.zeros_like(F); FB[1] = F[1]
    UB = oracle.farfield(X, FB, W)                       # vesicle B's contribution everywhere
    rows = near[:N, 1].astype(bool)
    assert np.allclose(Um[0][rows], (U[0] - UB[0])[rows], rtol=0, atol=1e-13)
    assert np.allclose(Um[0][~rows], U[0][~rows], rtol=0, atol=0)
    assert np.array_equal(Um[2], U[2])
    # subset variants are the same rows
    idx = np.array([0, 5, N - 1, N, N + 7, 2 * N, 3 * N - 1])
    rows_sub = oracle.near_mask_subset(X, W, idx)
    assert np.array_equal(rows_sub, near[idx])
    assert np.array_equal(oracle.farfield_masked_subset(X, F, W, idx, rows_sub), Um.reshape(-1, 2)[idx])
    # the relation is not symmetric in general (h belongs to the SOURCE vesicle): shrink B's weights
    W2 = W.copy(); W2[1] *= 0.1
    near2 = oracle.near_mask(X, W2)
    assert near2[N:2 * N, 0].any() and not near2[:N, 1].any()


# ----------------------------------------------------------------------------- elastic force (row f-2)
def _circle(R, N, c=(0.0, 0.0), warp=0.0):
    al = 2 * np.pi * np.arange(N) / N
    be = al + warp * np.sin(al)                      # warp != 0: same circle, points not equispaced in arclength
    return np.asarray(c) + R * np.stack([np.cos(be), np.sin(be)], -1), be


def test_elastic_force_circle_closed_form():
    """Circle of radius R about c: X_ss = -(X-c)/R^2, X_ssss = (X-c)/R^4, so with constant tension
    f = -kappa_b (X-c)/R^4 - sigma (X-c)/R^2 (eq 2.7).  A sign error in either term, a
    missing 1/|X_alpha| or a wrong derivative count fails this."""
    for N in (16, 32, 64):
        X, _ = _circle(0.7, N)
        F = oracle.elastic_force(X[None], np.full((1, N), 1.3), 0.4)[0]
        ref = -0.4 * X / 0.7 ** 4 - 1.3 * X / 0.7 ** 2
        assert np.abs(F - ref).max() <= 1e-16 * (N / 2) ** 4 * 64


def test_elastic_force_warped_circle_variable_tension():
    """Arclength derivatives do not depend on the parametrisation: a circle sampled at beta = alpha +
    0.3 sin(alpha) with sigma = 1.3 + 0.5 cos(beta) has (sigma X_s)_s = sigma_s X_s + sigma X_ss,
    sigma_s = -0.5 sin(beta)/R, X_s = (-sin beta, cos beta).  Error falls spectrally with N."""
    R, kb = 0.7, 0.4
    errs = []
    for N in (12, 16, 32):
        X, be = _circle(R, N, warp=0.3)
        sig = 1.3 + 0.5 * np.cos(be)
        Xs = np.stack([-np.sin(be), np.cos(be)], -1)
        ref = -kb * X / R ** 4 + (-0.5 * np.sin(be) / R)[:, None] * Xs - sig[:, None] * X / R ** 2
        errs.append(np.abs(oracle.elastic_force(X[None], sig[None], kb)[0] - ref).max())
    assert errs[0] > 1e-5 and errs[1] < 0.2 * errs[0] and errs[2] < 1e-10, errs


def test_elastic_force_ellipse_tension_is_curvature_times_normal():
    """kappa_b = 0, sigma = const on an ellipse sampled uniformly in the parameter (NOT in arclength):
    f = sigma X_ss = -sigma * curvature * outward normal, curvature = ab/(a^2 sin^2 + b^2 cos^2)^(3/2)."""
    a, b, N = 1.0, 0.6, 128
    t = 2 * np.pi * np.arange(N) / N
    th = 0.4
    R = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    X = np.stack([a * np.cos(t), b * np.sin(t)], -1) @ R.T
    q = np.sqrt(a * a * np.sin(t) ** 2 + b * b * np.cos(t) ** 2)
    n = np.stack([b * np.cos(t), a * np.sin(t)], -1) / q[:, None] @ R.T
    ref = -2.5 * (a * b / q ** 3)[:, None] * n
    F = oracle.elastic_force(X[None], np.full((1, N), 2.5), 0.0)[0]
    assert np.abs(F - ref).max() <= 1e-10


def _random_vesicles(seed, nves, N):
    rng = np.random.default_rng(seed)
    al = 2 * np.pi * np.arange(N) / N
    r = 1.0 + sum(rng.uniform(0, 0.1 / k, (nves, 1)) * np.cos(k * al + rng.uniform(0, 2 * np.pi, (nves, 1))) for k in (2, 3, 4))
    X = np.stack([r * np.cos(al), 0.6 * r * np.sin(al)], -1) + rng.normal(size=(nves, 1, 2))
    sig = 1.0 + sum(rng.normal(size=(nves, 1)) / k ** 2 * np.cos(k * al + rng.uniform(0, 2 * np.pi, (nves, 1))) for k in (1, 2, 3))
    return X, sig


def test_elastic_force_total_force_vanishes_and_symmetries():
    N = 32
    X, sig = _random_vesicles(5, 4, N)
    kb = 0.3
    F = oracle.elastic_force(X, sig, kb)
    W = oracle.weights(X)
    # sum_j f_j w_j = (2 pi/N) sum_j d/dalpha(...)_j = 0 exactly: a membrane exerts no net force
    assert np.abs((F * W[..., None]).sum(1)).max() <= 1e-11
    # net torque vanishes to spectral accuracy
    tq = ((X[..., 0] * F[..., 1] - X[..., 1] * F[..., 0]) * W).sum(1)
    assert np.abs(tq).max() <= 1e-6
    # translation invariance, rotation equivariance
    assert np.allclose(oracle.elastic_force(X + np.array([7.0, -3.0]), sig, kb), F, rtol=0, atol=1e-9)
    th = 1.1
    R = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    assert np.allclose(oracle.elastic_force(X @ R.T, sig, kb), F @ R.T, rtol=0, atol=1e-9)
    # linear in (kappa_b, sigma); bending scales like a^-3, tension like a^-1 under X -> a X
    Fb = oracle.elastic_force(X, 0 * sig, 1.0)
    Ft = oracle.elastic_force(X, sig, 0.0)
    assert np.allclose(F, kb * Fb + Ft, rtol=0, atol=1e-10)
    a = 1.7
    assert np.allclose(oracle.elastic_force(a * X, sig, kb), kb * Fb / a ** 3 + Ft / a, rtol=0, atol=1e-9)
    # each vesicle on its own
    assert np.array_equal(oracle.elastic_force(X[2:3], sig[2:3], kb)[0], F[2])
    # reversing the orientation of the curve changes nothing (even number of arclength derivatives)
    rev = np.concatenate([[0], np.arange(N - 1, 0, -1)])
    assert np.allclose(oracle.elastic_force(X[:, rev], sig[:, rev], kb)[:, rev], F, rtol=0, atol=1e-9)


def test_elastic_force_matches_numpy_fft_route():
    """Independent route: numpy's FFT for every derivative (library routine, double)."""
    N = 32
    X, sig = _random_vesicles(6, 3, N)
    k = np.fft.fftfreq(N, 1.0 / N)
    k[N // 2] = 0.0                                                     # reading A4
    D = lambda f: np.real(np.fft.ifft(1j * k[None, :, None] * np.fft.fft(f, axis=1), axis=1))
    dX = D(X)
    sa = np.sqrt((dX ** 2).sum(-1, keepdims=True))
    Xs = dX / sa
    Xssss = D(D(D(Xs) / sa) / sa) / sa
    ref = -0.8 * Xssss + D(sig[..., None] * Xs) / sa
    F = oracle.elastic_force(X, sig, 0.8)
    assert np.abs(F - ref).max() <= 1e-16 * (N / 2) ** 4 * 64 * np.abs(ref).max()


# ----------------------------------------------------------------------------- equal-arclength redistribution (row f-3)
def _np_redistribute(X):
    """Independent route through numpy's FFT, searchsorted and interp (library routines, double)."""
    nves, N, _ = X.shape
    M = 6 * N
    out = np.empty_like(X)
    k = np.fft.fftfreq(N, 1.0 / N)
    for v in range(nves):
        Xh = np.fft.fft(X[v], axis=0) / N
        pad = np.zeros((M, 2), dtype=complex)
        K = (N - 1) // 2
        pad[:K + 1] = Xh[:K + 1]
        pad[M - K:] = Xh[N - K:]
        dpad = pad * (1j * np.fft.fftfreq(M, 1.0 / M))[:, None]          # Nyquist mode not in it (reading A4)
        if N % 2 == 0:                                                    # cos(N alpha / 2): split over +-N/2
            pad[N // 2] = Xh[N // 2] / 2
            pad[M - N // 2] = Xh[N // 2] / 2
        Xu = np.real(np.fft.ifft(pad, axis=0)) * M
        dXu = np.real(np.fft.ifft(dpad, axis=0)) * M
        sa = np.sqrt((dXu ** 2).sum(1))
        sh = np.fft.fft(sa) / M
        kk = np.fft.fftfreq(M, 1.0 / M)
        ih = np.zeros(M, dtype=complex)
        nz = (kk != 0) & (np.abs(kk) != M // 2)
        ih[nz] = sh[nz] / (1j * kk[nz])
        prim = np.real(np.fft.ifft(ih)) * M
        al = 2 * np.pi * np.arange(M) / M
        l = np.real(sh[0]) * al + prim - prim[0]
        L = 2 * np.pi * np.real(sh[0])
        l = np.append(l, L)
        lt = np.arange(N) * L / N
        Xc = np.vstack([Xu, Xu[:1]])
        out[v, :, 0] = np.interp(lt, l, Xc[:, 0])
        out[v, :, 1] = np.interp(lt, l, Xc[:, 1])
    return out


def test_redistribute_fixed_point_and_warped_circle():
    """A circle sampled equally in arclength is a fixed point.  The same circle sampled at beta = alpha +
    0.4 sin(alpha) comes back equispaced in angle (the piecewise-linear error of the 6x-upsampled
    polygon is O((2 pi / 6N)^2)), on the chords of that polygon, with point 0 exactly where it was."""
    N, R = 32, 0.8
    al = 2 * np.pi * np.arange(N) / N
    X = R * np.stack([np.cos(al), np.sin(al)], -1)[None] + np.array([1.0, 2.0])
    assert np.abs(oracle.redistribute(X) - X).max() <= 2e-15
    be = al + 0.4 * np.sin(al)
    Xw = R * np.stack([np.cos(be), np.sin(be)], -1)[None]
    Y = oracle.redistribute(Xw)[0]
    assert np.abs(Y[0] - Xw[0, 0]).max() <= 1e-16
    ang = np.unwrap(np.arctan2(Y[:, 1], Y[:, 0]))
    assert np.abs(ang - al).max() <= 5e-6
    rad = np.hypot(Y[:, 0], Y[:, 1])
    sag = R * (1 - np.cos(1.4 * np.pi / (6 * N)))            # largest chord sag: fine spacing stretched by <= 1.4
    assert np.all(rad <= R + 1e-12) and np.all(rad >= R - sag * 1.01)
    # reversed orientation gives the mirrored answer; a wrong sign in the integration would not
    rev = np.concatenate([[0], np.arange(N - 1, 0, -1)])
    assert np.allclose(oracle.redistribute(Xw[:, rev])[0][rev], Y, rtol=0, atol=1e-13)


def test_redistribute_matches_numpy_route_and_equalises_spacing():
    for N in (31, 32, 64):
        X, _ = _random_vesicles(11 + N, 3, N)
        # make the sampling uneven in arclength on purpose
        al = 2 * np.pi * np.arange(N) / N
        be = al + 0.5 * np.sin(al + 0.3)
        kk = np.arange(-(N // 2) + 1, N // 2)
        Xh = np.array([[np.exp(-1j * k * al) @ X[v] / N for k in kk] for v in range(3)])
        Xw = np.real(np.einsum("jk,vkc->vjc", np.exp(1j * np.outer(be, kk)), Xh))
        Y = oracle.redistribute(Xw)
        assert np.abs(Y - _np_redistribute(Xw)).max() <= 1e-12
        W0, W1 = oracle.weights(Xw), oracle.weights(Y)
        assert (W0.max(1) / W0.min(1)).min() > 2.0                       # uneven before
        if N >= 32:
            assert (W1.max(1) / W1.min(1)).max() < 1.05                  # even after
        # the perimeter is preserved up to the chord sag
        assert np.allclose(W1.sum(1), W0.sum(1), rtol=2e-3)


def test_redistribute_equivariances():
    N = 32
    X, _ = _random_vesicles(21, 3, N)
    Y = oracle.redistribute(X)
    th = 0.7
    R = np.array([[np.cos(th), -np.sin(th)], [np.sin(th), np.cos(th)]])
    assert np.allclose(oracle.redistribute(X + np.array([5.0, -9.0])), Y + np.array([5.0, -9.0]), rtol=0, atol=1e-13)
    assert np.allclose(oracle.redistribute(X @ R.T), Y @ R.T, rtol=0, atol=1e-13)
    assert np.allclose(oracle.redistribute(2.5 * X), 2.5 * Y, rtol=0, atol=1e-13)
    assert np.array_equal(oracle.redistribute(X[1:2])[0], Y[1])
    # cyclic relabelling of the input points: the new point 0 follows the old point 0, the curve does not change,
    # so the new points are the same polygon's equal-arclength points started elsewhere -- still equispaced
    W = oracle.weights(oracle.redistribute(np.roll(X, 5, axis=1)))
    assert (W.max(1) / W.min(1)).max() < 1.05
    # almost idempotent: a second pass moves the points by much less than the first
    d1 = np.abs(Y - X).max()
    d2 = np.abs(oracle.redistribute(Y) - Y).max()
    assert d2 < 2e-2 * d1


# ----------------------------------------------------------------------------- complex form (the identity behind row f-4b)
def test_complex_potential_form_of_the_stokeslet_sum():
    """With z = x + i y, g = gx + i gy:  sum_j K(z - zeta_j) g_j = -(Re Phi1 + i Re Phi2) + (z/2) conj(Phi1' + i Phi2')
    - (1/2) conj(psi),  Phi_m = sum g_{m,j} log(z - zeta_j),  psi = sum [conj(zeta_j) g_j / (z - zeta_j) - conj(g_j)].
    An independent statement of the same sum (two logarithmic potentials and a Cauchy sum, evaluated by brute force
    with numpy's complex arithmetic): it pins the oracle once more and is the identity vn_farfield_fmm expands."""
    rng = np.random.default_rng(42)
    nves, N = 5, 12
    X = rng.normal(size=(nves, N, 2)) * 0.4 + 3.0 * rng.normal(size=(nves, 1, 2))
    F = rng.normal(size=(nves, N, 2))
    W = rng.uniform(0.5, 1.5, size=(nves, N))
    xt = rng.normal(size=(9, 2)) * 4.0 + np.array([15.0, -2.0])
    zeta = (X[..., 0] + 1j * X[..., 1]).ravel()
    g = ((F[..., 0] + 1j * F[..., 1]) * W).ravel()
    z = xt[:, 0] + 1j * xt[:, 1]
    dz = z[:, None] - zeta[None, :]
    Phi1 = (g.real[None, :] * np.log(dz)).sum(1)
    Phi2 = (g.imag[None, :] * np.log(dz)).sum(1)
    dPhi = ((g.real + 1j * g.imag)[None, :] / dz).sum(1)                 # Phi1' + i Phi2'
    psi = (np.conj(zeta)[None, :] * g[None, :] / dz - np.conj(g)[None, :]).sum(1)
    u = -(Phi1.real + 1j * Phi2.real) + 0.5 * z * np.conj(dPhi) - 0.5 * np.conj(psi)
    ref = oracle.farfield_targets(X, F, W, xt, mu=1.0) * 4 * np.pi
    assert np.abs(u - (ref[:, 0] + 1j * ref[:, 1])).max() <= 1e-13


# ----------------------------------------------------------------------------- sharp pins (round 2)
def test_near_mask_threshold_is_sharp_and_inclusive():
    """PAPER.md:144 "less than OR EQUAL TO the arclength spacing", :248 |d| <= h.  All coordinates are dyadic
    rationals, so d^2 and h^2 are exact doubles and the decision at d = h is not a rounding accident:
    h = 5/16; targets on the axis at h(1 - 1e-6), h, h(1 + 1e-6), 0.95 h, 1.05 h and on the 3-4-5 diagonal
    (3/16, 4/16) with d = 5/16 = h exactly, each next to its own source point (the sources are 10 apart)."""
    h = 0.3125
    offs = [(h * (1 - 1e-6), 0.0, 1), (h, 0.0, 1), (h * (1 + 1e-6), 0.0, 0), (0.95 * h, 0.0, 1), (1.05 * h, 0.0, 0),
            (0.1875, 0.25, 1), (0.0, -h, 1), (-0.1875, -0.25, 1), (0.1875 + 2.0 ** -20, 0.25, 0),
            (0.1875 - 2.0 ** -20, 0.25, 1)]
    n = len(offs)
    B = np.stack([10.0 * np.arange(n), np.zeros(n)], -1)                # source vesicle: spacing h
    A = B + np.array([(dx, dy) for dx, dy, _ in offs])                  # target vesicle: tiny spacing of its own
    X = np.stack([A, B])
    W = np.stack([np.full(n, 2.0 ** -10), np.full(n, h)])
    W[1, 3] = 0.25 * h                                                  # h is the LARGEST weight of the vesicle (N1)
    near = oracle.near_mask(X, W)
    want = np.array([e for _, _, e in offs], dtype=np.uint8)
    assert np.array_equal(near[:n, 1], want)
    assert not near[:n, 0].any() and not near[n:, 1].any()              # never the own vesicle
    assert not near[n:, 0].any()                                        # A's own spacing 2^-10: B is not near A
    assert np.array_equal(oracle.near_mask_subset(X, W, np.arange(2 * n)), near)
    # the spacing is the SOURCE vesicle's: give A the spacing h and B a tiny one, the relation flips
    near2 = oracle.near_mask(X, W[::-1].copy())
    assert np.array_equal(near2[n:, 0][[0, 1, 3, 5, 6, 7, 9]], np.ones(7, dtype=np.uint8)) and not near2[:n, 1].any()


def test_redistribute_integrates_every_mode_of_the_fine_spectrum():
    """Reading R2: the arclength is the term-by-term integral of the Fourier series of |X_alpha| on the fine grid,
    modes k = 1 .. M/2 - 1.  A strong ripple at the coarse grid's highest matched mode (N/2 - 1) puts energy
    6e-7 / 7e-6 (coefficient / k) into the fine grid's top mode M/2 - 1, so dropping any mode up to the last one
    moves the arclengths by far more than the 1e-12 this is compared at (numpy FFT / interp route)."""
    for N, amp in ((12, 0.2), (16, 0.2)):
        M = 6 * N
        al = 2 * np.pi * np.arange(N) / N
        r = 1 + amp * np.cos((N // 2 - 1) * al + 0.3)
        X = np.stack([r * np.cos(al), 0.7 * r * np.sin(al)], -1)[None] + np.array([0.5, -0.25])
        # the premise: |shat_k| / k at the top mode is large against the tolerance
        Xh = np.fft.fft(X[0], axis=0) / N
        pad = np.zeros((M, 2), dtype=complex)
        K = (N - 1) // 2
        pad[:K + 1] = Xh[:K + 1]
        pad[M - K:] = Xh[N - K:]
        dXu = np.real(np.fft.ifft(pad * (1j * np.fft.fftfreq(M, 1.0 / M))[:, None], axis=0)) * M
        sh = np.fft.fft(np.sqrt((dXu ** 2).sum(1))) / M
        assert abs(sh[M // 2 - 1]) / (M // 2 - 1) > 1e-7
        assert np.abs(oracle.redistribute(X) - _np_redistribute(X)).max() <= 1e-12


def test_speed_baseline_agrees_with_the_oracle():
    """oracle/baseline_f64.c (plain double, vectorised; the CPU SPEED baseline bench.py times) is the same sum as
    the long-double oracle: 1e-13 relative L2 and point-wise, on a suspension-like input and on random blobs.
    It is never compared with the CUDA path; this pin only keeps the timed code honest."""
    rng = np.random.default_rng(77)
    X, F, W = _random_problem(rng, 9, 37)
    idx = np.arange(9 * 37)
    ref = oracle.farfield_subset(X, F, W, idx, mu=0.8)
    got = oracle.baseline_farfield_subset(X, F, W, idx, mu=0.8)
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-13
    assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()
    assert np.array_equal(oracle.baseline_farfield_subset(X, F, W, idx[5:9], mu=0.8), got[5:9])
    A, _ = _ellipse(1.0, 0.4, 128, th=0.3)
    B, _ = _ellipse(1.0, 0.4, 128, th=1.1, c=(2.4, 0.3))
    X = np.stack([A, B]); F = rng.normal(size=X.shape); W = oracle.weights(X)
    ref = oracle.farfield(X, F, W).reshape(-1, 2)
    got = oracle.baseline_farfield_subset(X, F, W, np.arange(256))
    assert np.linalg.norm(got - ref) / np.linalg.norm(ref) <= 1e-13
