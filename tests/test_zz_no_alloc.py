"""vn_farfield_noalloc_f32 (include/vesnet_farfield.h): the fp32 general path with its scratch in a static device
array of the library instead of the stream-ordered allocator, for callers that may not allocate.  Checked against the
existing path (vn_farfield) on the same inputs, within the fp32 tolerance of the parity tests and -- the kernels and
the grid are the same and the accumulation is integer -- bit for bit, on calls IN A ROW that share the array: a
larger suspension, a smaller one (stale contents of the array beyond it must not matter), the first one again.

Collected last on purpose (the suite runs with pytest -x); passes alone in a fresh process and after the others."""
import ctypes

import numpy as np
import pytest

import paper_2606_25569_b200 as vn
from paper_2606_25569_b200 import inputs

pytestmark = pytest.mark.gpu
torch = pytest.importorskip("torch")

from parity_util import TOL, check


def _device_problem(s):
    X = torch.from_numpy(np.ascontiguousarray(s.X, dtype=np.float32)).cuda()
    F = torch.from_numpy(np.ascontiguousarray(s.F, dtype=np.float32)).cuda()
    return X, F, vn.vn_arclength_weights(X)


def test_noalloc_matches_vn_farfield_on_calls_in_a_row():
    big = inputs.config(1)                                                       # general path: > 1,024 points
    small = inputs.suspension(nves=40, npts=64, phi_area=0.2, aspect=1.0, seed=inputs.BASE_SEED + 901, nmodes=8)
    assert 1024 < small.nves * small.npts < big.nves * big.npts <= vn.vn_noalloc_max_points()
    probs = [(big, _device_problem(big)), (small, _device_problem(small))]
    refs = [vn.vn_farfield(X, F, W, s.mu) for s, (X, F, W) in probs]
    outs = [torch.full_like(X, float("nan")) for _, (X, _, _) in probs] + [torch.full_like(probs[0][1][0], float("nan"))]
    torch.cuda.synchronize()
    launches = vn.vn_launch_count()
    # three calls back to back on one stream, no synchronisation in between: big, small, big again
    order = [0, 1, 0]
    for k, which in enumerate(order):
        s, (X, F, W) = probs[which]
        vn.vn_farfield_noalloc_f32(X, F, W, outs[k], s.mu)
    torch.cuda.synchronize()
    assert vn.vn_launch_count() - launches == 3 * 3                            # pack, pair kernel, finish: ours ran
    for k, which in enumerate(order):
        got, ref = outs[k].cpu().numpy(), refs[which].cpu().numpy()
        check(got, ref, TOL[np.float32], f"noalloc call {k} vs vn_farfield")
        assert np.array_equal(got, ref)                                         # same kernels, same grid, integer sums


def test_noalloc_rejects_what_the_static_scratch_cannot_hold():
    cap = vn.vn_noalloc_max_points()
    assert cap == 1 << 18
    # sizes are checked before any pointer is used: dummy device tensors of the wrong size never reach a kernel
    t = torch.zeros(64, dtype=torch.float32, device="cuda")
    p = ctypes.c_void_p(t.data_ptr())
    q = ctypes.c_void_p(t.data_ptr() + 128)
    L = vn.lib()
    assert L.vn_farfield_noalloc_f32(p, p, p, cap // 128 + 1, 128, 1.0, q, None) == vn.VN_ERR_TOO_LARGE
    assert L.vn_farfield_noalloc_f32(p, p, p, 8000, 128, 1.0, q, None) == vn.VN_ERR_TOO_LARGE      # configs[4]
    assert b"262,144" in L.vn_status_string(vn.VN_ERR_TOO_LARGE)
    with pytest.raises(vn.VesnetError, match="static scratch"):
        raise vn.VesnetError(vn.VN_ERR_TOO_LARGE, "vn_farfield_noalloc_f32")
    # exactly at the limit the call is accepted and agrees with vn_farfield (2,048 x 128 points)
    s = inputs.suspension(nves=cap // 128, npts=128, phi_area=0.15, aspect=1.0, seed=inputs.BASE_SEED + 902, nmodes=8)
    X, F, W = _device_problem(s)
    out = torch.full_like(X, float("nan"))
    vn.vn_farfield_noalloc_f32(X, F, W, out, s.mu)
    ref = vn.vn_farfield(X, F, W, s.mu)
    torch.cuda.synchronize()
    check(out.cpu().numpy(), ref.cpu().numpy(), TOL[np.float32], "noalloc at the limit vs vn_farfield")
    assert torch.equal(out, ref)
