"""TEST INFRASTRUCTURE, NOT THE PRODUCT.

ctypes wrapper around ``oracle_vesnet.c`` -- the plain long-double CPU statement of
VesNet's far-field single-layer sum (PAPER.md:129-136 eqs 2.8/2.9, :173 trapezoid rule,
:140-144 who contributes, :163-169 spectral derivative).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl reference``
legs may import this package.  It imports nothing from ``paper_2606_25569_b200`` and
that package imports nothing from here.

All arrays are float64 numpy arrays on the host; results are float64.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import zlib

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "oracle_vesnet.c")
_LIB = os.path.join(_HERE, "liboracle_vesnet.so")
_lib = None
_BASE_SRC = os.path.join(_HERE, "baseline_f64.c")
_BASE_LIB = os.path.join(_HERE, "libbaseline_f64.so")
_BASE_FLAGS = ["-O3", "-march=native", "-ffast-math", "-fopenmp"]
_base = None


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no FMA contraction, OpenMP over targets only)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


def _cpu_stamp() -> str:
    """Identifies the instruction set of this machine (-march=native binaries must not travel between machines)."""
    try:
        with open("/proc/cpuinfo") as fh:
            for line in fh:
                if line.startswith("flags"):
                    return str(zlib.crc32(line.split(":", 1)[1].strip().encode()))
    except OSError:
        pass
    return "unknown"


def build_baseline(force: bool = False) -> str:
    """Compile baseline_f64.c, the plain-double SPEED baseline (not the parity oracle; see its header).
    -march=native: rebuilt whenever the library was made on a machine with another instruction set (the in-tree .so
    travels to the GPU box with the snapshot), and always on the machine that times it (bench.py passes force=True)."""
    stamp_file = _BASE_LIB + ".cpu"
    stamp = _cpu_stamp()
    old = open(stamp_file).read().strip() if os.path.exists(stamp_file) else ""
    if (force or old != stamp or not os.path.exists(_BASE_LIB)
            or os.path.getmtime(_BASE_LIB) < os.path.getmtime(_BASE_SRC)):
        subprocess.run(["gcc"] + _BASE_FLAGS + ["-fPIC", "-shared", "-o", _BASE_LIB, _BASE_SRC, "-lm"], check=True)
        with open(stamp_file, "w") as fh:
            fh.write(stamp)
    return _BASE_LIB


def baseline_flags() -> str:
    return "gcc " + " ".join(_BASE_FLAGS)


def baseline_farfield_subset(X, F, W, idx, mu=1.0, rebuild=False):
    """The direct sum in plain double at the flat point indices ``idx`` -> [len(idx), 2] (speed baseline)."""
    global _base
    if _base is None or rebuild:
        lib = ctypes.CDLL(build_baseline(force=rebuild))
        d = ctypes.POINTER(ctypes.c_double)
        lib.baseline_num_threads.restype = ctypes.c_int
        lib.baseline_farfield_subset.argtypes = [d, d, d, ctypes.c_int64, ctypes.c_int64, ctypes.c_double,
                                                 ctypes.POINTER(ctypes.c_int64), ctypes.c_int64, d]
        _base = lib
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    Us = np.empty((idx.size, 2), dtype=np.float64)
    rc = _base.baseline_farfield_subset(_p(X), _p(F), _p(W), nves, npts, float(mu),
                                        idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), idx.size, _p(Us))
    if rc:
        raise ValueError(f"baseline_farfield_subset rc={rc}")
    return Us


def _load():
    global _lib
    if _lib is None:
        build()
        lib = ctypes.CDLL(_LIB)
        d = ctypes.POINTER(ctypes.c_double)
        i64 = ctypes.c_int64
        u8 = ctypes.POINTER(ctypes.c_ubyte)
        lib.oracle_num_threads.restype = ctypes.c_int
        lib.oracle_farfield.argtypes = [d, d, d, i64, i64, ctypes.c_double, d]
        lib.oracle_farfield_subset.argtypes = [d, d, d, i64, i64, ctypes.c_double,
                                               ctypes.POINTER(i64), i64, d]
        lib.oracle_farfield_targets.argtypes = [d, d, d, i64, i64, ctypes.c_double, d, i64, d]
        lib.oracle_weights.argtypes = [d, i64, i64, d, d]
        lib.oracle_near_mask.argtypes = [d, d, i64, i64, u8]
        lib.oracle_farfield_masked.argtypes = [d, d, d, i64, i64, ctypes.c_double, u8, d]
        lib.oracle_near_mask_subset.argtypes = [d, d, i64, i64, ctypes.POINTER(i64), i64, u8]
        lib.oracle_farfield_masked_subset.argtypes = [d, d, d, i64, i64, ctypes.c_double,
                                                      ctypes.POINTER(i64), i64, u8, d]
        lib.oracle_elastic_force.argtypes = [d, d, i64, i64, ctypes.c_double, d]
        lib.oracle_redistribute.argtypes = [d, i64, i64, d]
        _lib = lib
    return _lib


def _c(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if shape is not None and a.shape != tuple(shape):
        raise ValueError(f"expected shape {shape}, got {a.shape}")
    return a


def _p(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def num_threads() -> int:
    return int(_load().oracle_num_threads())


def farfield(X, F, W, mu=1.0):
    """U[nves,npts,2]: eq 2.8/2.9 by the trapezoid rule over every other vesicle."""
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    U = np.empty_like(X)
    rc = _load().oracle_farfield(_p(X), _p(F), _p(W), nves, npts, float(mu), _p(U))
    if rc:
        raise ValueError(f"oracle_farfield rc={rc}")
    return U


def farfield_subset(X, F, W, idx, mu=1.0):
    """U at the flat point indices ``idx`` only -> [len(idx), 2]."""
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    Us = np.empty((idx.size, 2), dtype=np.float64)
    rc = _load().oracle_farfield_subset(_p(X), _p(F), _p(W), nves, npts, float(mu),
                                        idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)),
                                        idx.size, _p(Us))
    if rc:
        raise ValueError(f"oracle_farfield_subset rc={rc}")
    return Us


def farfield_targets(X, F, W, xt, mu=1.0):
    """Velocity at free points xt[nt,2] induced by all vesicles -> [nt,2]."""
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    xt = _c(xt)
    Ut = np.empty_like(xt)
    rc = _load().oracle_farfield_targets(_p(X), _p(F), _p(W), nves, npts, float(mu),
                                         _p(xt), xt.shape[0], _p(Ut))
    if rc:
        raise ValueError(f"oracle_farfield_targets rc={rc}")
    return Ut


def weights(X, return_derivative=False):
    """W[nves,npts] = (2 pi/N) |dX/dalpha| by explicit DFT -> ik -> inverse DFT."""
    X = _c(X); nves, npts, _ = X.shape
    W = np.empty((nves, npts), dtype=np.float64)
    dX = np.empty_like(X) if return_derivative else None
    rc = _load().oracle_weights(_p(X), nves, npts, _p(W), _p(dX) if dX is not None else None)
    if rc:
        raise ValueError(f"oracle_weights rc={rc}")
    return (W, dX) if return_derivative else W


def near_mask(X, W):
    """near[P, nves] (uint8): vesicle vp within its arclength spacing of point t."""
    X = _c(X); nves, npts, _ = X.shape
    W = _c(W, (nves, npts))
    near = np.empty((nves * npts, nves), dtype=np.uint8)
    rc = _load().oracle_near_mask(_p(X), _p(W), nves, npts,
                                  near.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)))
    if rc:
        raise ValueError(f"oracle_near_mask rc={rc}")
    return near


def farfield_masked(X, F, W, near, mu=1.0):
    """Direct sum with near vesicles' contribution set to zero."""
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    near = np.ascontiguousarray(near, dtype=np.uint8)
    if near.shape != (nves * npts, nves):
        raise ValueError("near mask shape")
    U = np.empty_like(X)
    rc = _load().oracle_farfield_masked(_p(X), _p(F), _p(W), nves, npts, float(mu),
                                        near.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)), _p(U))
    if rc:
        raise ValueError(f"oracle_farfield_masked rc={rc}")
    return U


def near_mask_subset(X, W, idx):
    """Rows ``idx`` of the near mask -> [len(idx), nves] (uint8)."""
    X = _c(X); nves, npts, _ = X.shape
    W = _c(W, (nves, npts))
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    near = np.empty((idx.size, nves), dtype=np.uint8)
    rc = _load().oracle_near_mask_subset(_p(X), _p(W), nves, npts,
                                         idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), idx.size,
                                         near.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)))
    if rc:
        raise ValueError(f"oracle_near_mask_subset rc={rc}")
    return near


def farfield_masked_subset(X, F, W, idx, near_rows, mu=1.0):
    """Masked direct sum at the flat point indices ``idx``; near_rows: [len(idx), nves]."""
    X = _c(X); nves, npts, _ = X.shape
    F = _c(F, X.shape); W = _c(W, (nves, npts))
    idx = np.ascontiguousarray(idx, dtype=np.int64)
    near_rows = np.ascontiguousarray(near_rows, dtype=np.uint8)
    if near_rows.shape != (idx.size, nves):
        raise ValueError("near_rows shape")
    Us = np.empty((idx.size, 2), dtype=np.float64)
    rc = _load().oracle_farfield_masked_subset(_p(X), _p(F), _p(W), nves, npts, float(mu),
                                               idx.ctypes.data_as(ctypes.POINTER(ctypes.c_int64)), idx.size,
                                               near_rows.ctypes.data_as(ctypes.POINTER(ctypes.c_ubyte)), _p(Us))
    if rc:
        raise ValueError(f"oracle_farfield_masked_subset rc={rc}")
    return Us


def elastic_force(X, sigma, kappa_b=1.0):
    """f = -kappa_b X_ssss + (sigma X_s)_s (eq 2.7), spectral arclength derivatives -> [nves,npts,2]."""
    X = _c(X); nves, npts, _ = X.shape
    sigma = _c(sigma, (nves, npts))
    F = np.empty_like(X)
    rc = _load().oracle_elastic_force(_p(X), _p(sigma), nves, npts, float(kappa_b), _p(F))
    if rc:
        raise ValueError(f"oracle_elastic_force rc={rc}")
    return F


def redistribute(X):
    """Points of every vesicle redistributed equally in arclength (sec 4.2) -> [nves,npts,2]."""
    X = _c(X); nves, npts, _ = X.shape
    Xn = np.empty_like(X)
    rc = _load().oracle_redistribute(_p(X), nves, npts, _p(Xn))
    if rc:
        raise ValueError(f"oracle_redistribute rc={rc}")
    return Xn
