"""Builds libvesnet_farfield.so in-tree with nvcc for sm_100a (no other target, no fallback).

    python -m paper_2606_25569_b200.build [--force] [-v]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libvesnet_farfield.so")
SOURCES = ["vn_api.cu", "vn_farfield_f32.cu", "vn_farfield_f64.cu", "vn_weights.cu", "vn_near.cu", "vn_force.cu", "vn_redistribute.cu", "vn_fmm.cu", "vn_peaks.cu", "vn_farfield_small.cu"]
HEADERS = [os.path.join(CSRC, "vn_common.cuh"), os.path.join(CSRC, "vn_log64.cuh"),
           os.path.join(os.path.dirname(HERE), "include", "vesnet_farfield.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc() -> str:
    cand = os.environ.get("NVCC")
    if cand:
        return cand
    return "/usr/local/cuda/bin/nvcc" if os.path.exists("/usr/local/cuda/bin/nvcc") else "nvcc"


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES] + HEADERS + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        cmd = [_nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
