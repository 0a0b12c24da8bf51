"""The C-ABI library loads on a CPU-only box, exports every symbol the header declares, and
rejects bad arguments before touching CUDA (no compute calls here)."""
import ctypes
import os
import re

import paper_2606_25569_b200 as vn

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    text = open(os.path.join(ROOT, "include", "vesnet_farfield.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(vn_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    from paper_2606_25569_b200 import build
    build.build()
    L = vn.lib()
    names = _declared()
    assert {"vn_farfield", "vn_arclength_weights", "vn_farfield_host", "vn_status_string",
            "vn_version", "vn_launch_count", "vn_near_pairs", "vn_farfield_masked",
            "vn_farfield_targets", "vn_elastic_force", "vn_redistribute_arclength", "vn_farfield_fmm", "vn_farfield_targets_fmm", "vn_plan_farfield"} <= set(names)
    for n in names:
        assert hasattr(L, n), n
    # the header's encoding, major*10000 + minor*100 + patch, and the header's own constant
    header = open(os.path.join(ROOT, "include", "vesnet_farfield.h")).read()
    assert vn.vn_version() == int(re.search(r"#define\s+VN_VERSION\s+(\d+)", header).group(1)) == 201
    assert "vn_pipe_peaks" in names and "vn_farfield_noalloc_f32" in names and "vn_noalloc_max_points" in names
    assert L.vn_status_string(0) == b"ok" and b"invalid" in L.vn_status_string(1)


def test_argument_validation_needs_no_gpu():
    L = vn.lib()
    buf = (ctypes.c_double * 64)()
    p = ctypes.addressof(buf)
    q = p + 256 if False else ctypes.addressof((ctypes.c_double * 64)())
    INV = vn.VN_ERR_INVALID_ARG
    assert L.vn_farfield(None, p, p, 2, 4, 1.0, q, vn.VN_F64, None) == INV          # null
    assert L.vn_farfield(p, p, p, 0, 4, 1.0, q, vn.VN_F64, None) == INV             # nves < 1
    assert L.vn_farfield(p, p, p, 2, 0, 1.0, q, vn.VN_F64, None) == INV             # npts < 1
    assert L.vn_farfield(p, p, p, 1 << 20, 1 << 12, 1.0, q, vn.VN_F32, None) == INV  # >= 2^31 points
    assert L.vn_farfield(p, p, p, 2, 4, 0.0, q, vn.VN_F64, None) == INV             # mu <= 0
    assert L.vn_farfield(p, p, p, 2, 4, float("nan"), q, vn.VN_F64, None) == INV    # mu not finite
    assert L.vn_farfield(p, p, p, 2, 4, 1.0, q, 7, None) == INV                     # bad enum
    assert L.vn_farfield(p + 4, p, p, 2, 4, 1.0, q, vn.VN_F32, None) == INV         # misaligned pair
    assert L.vn_farfield(p, p, p, 2, 4, 1.0, p, vn.VN_F64, None) == INV             # U aliases X
    assert L.vn_arclength_weights(None, 2, 4, q, vn.VN_F64, None) == INV
    # no-allocation entry point: the size limit of its static scratch is checked before any CUDA call
    cap = L.vn_noalloc_max_points()
    assert cap == 262144
    assert L.vn_farfield_noalloc_f32(p, p, p, cap // 128 + 1, 128, 1.0, q, None) == vn.VN_ERR_TOO_LARGE
    assert L.vn_farfield_noalloc_f32(p, p, p, 1, cap + 1, 1.0, q, None) == vn.VN_ERR_TOO_LARGE
    assert L.vn_farfield_noalloc_f32(None, p, p, 2, 4, 1.0, q, None) == INV
    assert L.vn_farfield_noalloc_f32(p, p, p, 2, 4, -1.0, q, None) == INV
    assert L.vn_farfield_noalloc_f32(p, p, p, 2, 4, 1.0, p, None) == INV              # U aliases X
    assert b"static scratch" in L.vn_status_string(vn.VN_ERR_TOO_LARGE)
    assert L.vn_arclength_weights(p, 2, -1, q, vn.VN_F64, None) == INV
    # NEXT rows
    assert L.vn_near_pairs(p, None, 2, 4, q, None, 0, vn.VN_F64, None) == INV          # null W
    assert L.vn_near_pairs(p, p, 2, 4, None, None, 0, vn.VN_F64, None) == INV          # null near_ptr
    assert L.vn_near_pairs(p, p, 2, 4, q, None, 5, vn.VN_F64, None) == INV             # capacity without buffer
    assert L.vn_near_pairs(p, p, 2, 4, q, q, -1, vn.VN_F64, None) == INV               # negative capacity
    assert L.vn_near_pairs(p, p, 2, 4, q + 4, None, 0, vn.VN_F64, None) == INV         # misaligned near_ptr
    assert L.vn_farfield_masked(p, p, p, 2, 4, 1.0, None, None, q, vn.VN_F64, None) == INV
    assert L.vn_farfield_masked(p, p, p, 2, 4, -2.0, q, None, q, vn.VN_F64, None) == INV
    assert L.vn_farfield_targets(None, 3, p, p, p, 2, 4, 1.0, q, vn.VN_F64, None) == INV
    assert L.vn_farfield_targets(q, -1, p, p, p, 2, 4, 1.0, q, vn.VN_F64, None) == INV
    assert L.vn_farfield_targets(q, 3, p, p, p, 2, 4, 1.0, q, vn.VN_F64, None) == INV   # Ut aliases Xt
    assert L.vn_farfield_targets(None, 0, p, p, p, 2, 4, 1.0, None, vn.VN_F64, None) == vn.VN_OK   # nt == 0: nothing to do
    assert L.vn_elastic_force(p, None, 2, 4, 1.0, q, vn.VN_F64, None) == INV            # null sigma
    assert L.vn_elastic_force(p, p, 2, 1025, 1.0, q, vn.VN_F64, None) == INV            # npts > 1024
    assert L.vn_elastic_force(p, p, 2, 4, float("inf"), q, vn.VN_F64, None) == INV      # kappa_b not finite
    assert L.vn_redistribute_arclength(None, 2, 4, q, vn.VN_F64, None) == INV
    assert L.vn_redistribute_arclength(p, 2, 2, q, vn.VN_F64, None) == INV               # npts < 3
    assert L.vn_redistribute_arclength(p, 2, 513, q, vn.VN_F64, None) == INV             # npts > 512
    assert L.vn_redistribute_arclength(p, 2, 4, p, vn.VN_F64, None) == INV               # in place
    assert L.vn_farfield_fmm(p, p, None, 2, 4, 1.0, 12, None, None, q, vn.VN_F64, None) == INV       # null W
    assert L.vn_farfield_fmm(p, p, p, 2, 4, 1.0, 1, None, None, q, vn.VN_F64, None) == INV          # order < 2
    assert L.vn_farfield_fmm(p, p, p, 2, 4, 1.0, 49, None, None, q, vn.VN_F64, None) == INV         # order > 48
    assert L.vn_farfield_fmm(p, p, p, 2, 4, 1.0, 12, None, None, p, vn.VN_F64, None) == INV         # U aliases X
    assert L.vn_farfield_targets_fmm(q, 3, p, p, p, 2, 4, 1.0, 60, q, vn.VN_F64, None) == INV   # order > 48
    assert L.vn_farfield_targets_fmm(None, 0, p, p, p, 2, 4, 1.0, 12, None, vn.VN_F64, None) == vn.VN_OK
    assert L.vn_farfield_host(p, None, None, 2, 4, 1.0, q, vn.VN_F64) == INV
    assert L.vn_pipe_peaks(None, None) == INV
    assert L.vn_farfield_host(p, p, None, 2, 4, -1.0, q, vn.VN_F64) == INV


def test_partial_and_finish_argument_validation():
    L = vn.lib()
    buf = (ctypes.c_double * 64)()
    p = ctypes.addressof(buf)
    q = ctypes.addressof((ctypes.c_double * 64)())
    g = ctypes.addressof((ctypes.c_double * 2)())
    INV = vn.VN_ERR_INVALID_ARG
    assert L.vn_farfield_partial(p, p, p, 2, 4, 2, 2, q, g, vn.VN_F32, None) == INV        # part >= nparts
    assert L.vn_farfield_partial(p, p, p, 2, 4, -1, 2, q, g, vn.VN_F32, None) == INV       # part < 0
    assert L.vn_farfield_partial(p, p, p, 2, 4, 0, 0, q, g, vn.VN_F32, None) == INV        # nparts < 1
    assert L.vn_farfield_partial(p, p, p, 2, 4, 0, 1, None, g, vn.VN_F32, None) == INV     # null acc
    assert L.vn_farfield_partial(p, p, p, 2, 4, 0, 1, q, None, vn.VN_F32, None) == INV     # null gmax
    assert L.vn_farfield_partial(p, p, p, 2, 4, 0, 1, p, g, vn.VN_F32, None) == INV        # acc aliases X
    assert L.vn_farfield_finish(q, g, 8, 9, 1.0, p, vn.VN_F32, None) == INV                # count > total
    assert L.vn_farfield_finish(q, g, 8, -1, 1.0, p, vn.VN_F32, None) == INV
    assert L.vn_farfield_finish(q, g, 8, 4, 0.0, p, vn.VN_F32, None) == INV                # mu
    assert L.vn_farfield_finish(q, g, 8, 4, 1.0, None, vn.VN_F32, None) == INV             # null U
    assert L.vn_farfield_finish(None, g, 8, 0, 1.0, None, vn.VN_F32, None) == vn.VN_OK     # count == 0: nothing to do
