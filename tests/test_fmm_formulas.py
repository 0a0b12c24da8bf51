"""CPU check of the FMM's translation formulas (numpy restatement in tests/fmm_numpy.py) against the oracle: the
truncation error falls geometrically with the order and reaches rounding level."""
import numpy as np

import oracle
from fmm_numpy import fmm


def test_numpy_fmm_converges_to_the_oracle():
    rng = np.random.default_rng(3)
    nves, npts = 40, 16
    al = 2 * np.pi * np.arange(npts) / npts
    body = 0.35 * np.stack([np.cos(al), 0.6 * np.sin(al)], -1)
    X = body[None] + rng.uniform(0, 12, size=(nves, 1, 2))
    F = rng.normal(size=X.shape)
    W = oracle.weights(X)
    ref = oracle.farfield(X, F, W, 1.0).reshape(-1, 2) * 4 * np.pi
    ref = ref[:, 0] + 1j * ref[:, 1]
    G = (F * W[..., None]).reshape(-1, 2)
    ves = np.repeat(np.arange(nves), npts)
    errs = []
    for p in (6, 12, 24, 40):
        u = fmm(X.reshape(-1, 2), G, ves, 3, p)
        errs.append(np.linalg.norm(u - ref) / np.linalg.norm(ref))
    assert errs[0] < 1e-2 and errs[1] < 1e-2 * errs[0] * 10 and errs[2] < 1e-8 and errs[3] < 1e-13, errs
    assert all(b < a for a, b in zip(errs, errs[1:]))
