"""Shared comparison helpers of the GPU parity tests.

Two measures, both asserted wherever the CUDA path is compared with the oracle:
  rel-L2     ||got - ref||_2 / ||ref||_2 over the whole array          (north_star's metric and tolerances)
  max-rel    max_i |got_i - ref_i| / max_i |ref_i|, i over POINTS       (|.| the Euclidean norm of the 2-vector)
A single norm hides local faults -- one target of 32,768 wrong by 1e-3 moves the fp32 rel-L2 by 4e-6, a fifth of
its tolerance -- and a tile-boundary or ragged-tail bug is exactly a few-targets bug.  max-rel is held to
C_MAX x the rel-L2 tolerance; C_MAX = 1 (measured maxima are recorded in DESIGN.md section 7: the point-wise
error of a correct run sits at or below its rel-L2 because the largest velocities carry the norm)."""
import json
import os

import numpy as np

TOL = {np.float64: 1e-12, np.float32: 2e-5}
C_MAX = 1.0
_LOG = os.environ.get("VN_PARITY_LOG")          # optional: one JSON line per comparison (measured values for DESIGN.md)


def rel_l2(a, b):
    a = np.asarray(a, dtype=np.float64).ravel()
    b = np.asarray(b, dtype=np.float64).ravel()
    return float(np.linalg.norm(a - b) / np.linalg.norm(b))


def max_rel(a, b, vec=2):
    """Largest point-wise error over the largest point-wise magnitude of the reference."""
    a = np.asarray(a, dtype=np.float64)
    b = np.asarray(b, dtype=np.float64)
    if vec > 1:
        a, b = a.reshape(-1, vec), b.reshape(-1, vec)
        d, m = np.sqrt(((a - b) ** 2).sum(1)), np.sqrt((b ** 2).sum(1))
    else:
        d, m = np.abs(a - b).ravel(), np.abs(b).ravel()
    return float(d.max() / m.max())


def check(got, ref, tol, label="", vec=2, c_max=C_MAX):
    """Asserts rel-L2 <= tol and max-rel <= c_max * tol; returns (rel-L2, max-rel)."""
    got = np.asarray(got, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    assert got.shape == ref.shape or got.size == ref.size, (got.shape, ref.shape)
    assert np.all(np.isfinite(got)), f"{label}: non-finite values"
    e2, em = rel_l2(got, ref), max_rel(got, ref, vec)
    print(f"{label}: rel-L2 {e2:.3e}, max-rel {em:.3e} (tolerance {tol:.1e}, x{c_max:g} point-wise, {ref.size // max(vec, 1)} points)")
    if _LOG:
        with open(_LOG, "a") as fh:
            fh.write(json.dumps({"case": label, "rel_l2": e2, "max_rel": em, "tol": tol, "points": ref.size // max(vec, 1)}) + "\n")
    assert e2 <= tol, f"{label}: rel-L2 {e2:.3e} > {tol:.1e}"
    assert em <= c_max * tol, f"{label}: max-rel {em:.3e} > {c_max * tol:.1e}"
    return e2, em
