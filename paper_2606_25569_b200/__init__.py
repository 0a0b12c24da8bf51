"""paper_2606_25569_b200 -- B200-native far-field module of VesNet (arxiv/paper_2606_25569).

Thin Python binding over the C-ABI library ``libvesnet_farfield.so`` (include/vesnet_farfield.h).
The functions below carry the same names as the C entry points and do argument marshalling only:
every step of the path (weights, packing, pair sum, reduction, scaling) runs in the library's
sm_100a kernels.  PyTorch is used for device memory and streams, nothing else.  There is no CPU
or PyTorch fallback: if the library is missing or the device is not a B200-class GPU the call
raises.

    W = vn_arclength_weights(X)                 # X: [nves, npts, 2] cuda tensor, fp32 or fp64
    U = vn_farfield(X, F, W, mu=1.0)            # U: [nves, npts, 2]
    U = vn_farfield_host(X, F, None, mu=1.0)    # host (numpy / pinned torch) buffers, whole path
    ptr, ves = vn_near_pairs(X, W)              # near-field relation (CSR)
    U = vn_farfield_masked(X, F, W, ptr, ves)   # the paper's DirectSingleLayerIntegral
    Ut = vn_farfield_targets(Xt, X, F, W)       # velocity at free points Xt[nt, 2]
    F = vn_elastic_force(X, sigma, kappa_b)     # eq 2.7, the density the sums above consume
    Xe = vn_redistribute_arclength(X)           # points equispaced in arclength, sec 4.2
    U = vn_farfield_fmm(X, F, W, order=12)      # the same sum in O(P) by a fast multipole method (approximate)

`inputs` (seeded synthetic suspensions) is importable without the library.
"""
from __future__ import annotations

import ctypes
import os

VN_F32, VN_F64 = 0, 1
VN_OK, VN_ERR_INVALID_ARG, VN_ERR_UNSUPPORTED, VN_ERR_CUDA, VN_ERR_TOO_LARGE = 0, 1, 2, 3, 4

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libvesnet_farfield.so")
_lib = None


class VesnetError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        msg = lib().vn_status_string(status).decode()
        super().__init__(f"{where}: {msg} (vn_status {status})")


def lib():
    """Load the C-ABI library (built in-tree by ``python -m paper_2606_25569_b200.build``)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_25569_b200.build` "
                              "(nvcc, sm_100a). There is no fallback path.")
        L = ctypes.CDLL(LIB_PATH)
        vp, i64, dbl, ci = ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_int
        L.vn_farfield.argtypes = [vp, vp, vp, i64, i64, dbl, vp, ci, vp]
        L.vn_farfield.restype = ci
        L.vn_arclength_weights.argtypes = [vp, i64, i64, vp, ci, vp]
        L.vn_arclength_weights.restype = ci
        L.vn_farfield_host.argtypes = [vp, vp, vp, i64, i64, dbl, vp, ci]
        L.vn_farfield_host.restype = ci
        L.vn_near_pairs.argtypes = [vp, vp, i64, i64, vp, vp, i64, ci, vp]
        L.vn_near_pairs.restype = ci
        L.vn_farfield_masked.argtypes = [vp, vp, vp, i64, i64, dbl, vp, vp, vp, ci, vp]
        L.vn_farfield_masked.restype = ci
        L.vn_farfield_targets.argtypes = [vp, i64, vp, vp, vp, i64, i64, dbl, vp, ci, vp]
        L.vn_farfield_targets.restype = ci
        L.vn_elastic_force.argtypes = [vp, vp, i64, i64, dbl, vp, ci, vp]
        L.vn_elastic_force.restype = ci
        L.vn_redistribute_arclength.argtypes = [vp, i64, i64, vp, ci, vp]
        L.vn_redistribute_arclength.restype = ci
        L.vn_farfield_fmm.argtypes = [vp, vp, vp, i64, i64, dbl, ci, vp, vp, vp, ci, vp]
        L.vn_farfield_fmm.restype = ci
        L.vn_farfield_targets_fmm.argtypes = [vp, i64, vp, vp, vp, i64, i64, dbl, ci, vp, ci, vp]
        L.vn_farfield_targets_fmm.restype = ci
        L.vn_plan_farfield.argtypes = [i64, i64, ci, ctypes.c_int32, ctypes.POINTER(ctypes.c_int32)]
        L.vn_plan_farfield.restype = ci
        L.vn_profile_enable.argtypes = [ci]
        L.vn_profile_enable.restype = ci
        L.vn_profile_read.argtypes = [ctypes.POINTER(dbl), i64]
        L.vn_profile_read.restype = i64
        L.vn_launch_count.argtypes = []
        L.vn_launch_count.restype = i64
        L.vn_status_string.argtypes = [ci]
        L.vn_status_string.restype = ctypes.c_char_p
        L.vn_farfield_partial.argtypes = [vp, vp, vp, i64, i64, ctypes.c_int32, ctypes.c_int32, vp, vp, ci, vp]
        L.vn_farfield_partial.restype = ci
        L.vn_farfield_finish.argtypes = [vp, vp, i64, i64, dbl, vp, ci, vp]
        L.vn_farfield_finish.restype = ci
        L.vn_selfcheck.argtypes = [vp, vp, vp, i64, i64, dbl, vp, ci, vp, ctypes.POINTER(i64)]
        L.vn_selfcheck.restype = ci
        L.vn_pipe_peaks.argtypes = [ctypes.POINTER(dbl), vp]
        L.vn_pipe_peaks.restype = ci
        L.vn_farfield_noalloc_f32.argtypes = [vp, vp, vp, i64, i64, dbl, vp, vp]
        L.vn_farfield_noalloc_f32.restype = ci
        L.vn_noalloc_max_points.argtypes = []
        L.vn_noalloc_max_points.restype = i64
        L.vn_version.argtypes = []
        L.vn_version.restype = ci
        _lib = L
    return _lib


def _prec(t):
    import torch
    if t.dtype == torch.float32:
        return VN_F32
    if t.dtype == torch.float64:
        return VN_F64
    raise TypeError(f"dtype must be float32 or float64, got {t.dtype}")


def _check_dev(name, t, shape=None, dtype=None):
    if not t.is_cuda:
        raise ValueError(f"{name} must be a CUDA tensor (device calls take device pointers)")
    if not t.is_contiguous():
        raise ValueError(f"{name} must be contiguous")
    if shape is not None and tuple(t.shape) != tuple(shape):
        raise ValueError(f"{name}: expected shape {tuple(shape)}, got {tuple(t.shape)}")
    if dtype is not None and t.dtype != dtype:
        raise TypeError(f"{name}: expected dtype {dtype}, got {t.dtype}")


def _stream_ptr(stream):
    """cudaStream_t of `stream`, or of torch's current stream on the current device (the bindings make the tensors'
    device current first).  The raw-handle query costs 0.3 us where building a torch.cuda.Stream object costs 3."""
    import torch
    if stream is not None:
        return ctypes.c_void_p(stream.cuda_stream)
    raw = getattr(torch._C, "_cuda_getCurrentRawStream", None)
    if raw is not None:
        return ctypes.c_void_p(raw(torch.cuda.current_device()))
    return ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)


class _NoGuard:
    def __enter__(self):
        return None

    def __exit__(self, *exc):
        return False


_NO_GUARD = _NoGuard()


def _on(device):
    """Context that makes `device` current for the call -- nothing at all when it already is (every call of a
    single-GPU process; torch.cuda.device() costs 3 us to enter and leave, a tenth of a small problem's step)."""
    import torch
    return _NO_GUARD if device.index == torch.cuda.current_device() else torch.cuda.device(device)


def vn_farfield(X, F, W, mu: float = 1.0, out=None, stream=None):
    """U = far-field single-layer potential (device tensors; enqueues on the current stream)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    with _on(X.device):
        rc = lib().vn_farfield(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu),
                               out.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield")
    return out


def _raw_stream_fn():
    try:
        import torch
        return getattr(torch._C, "_cuda_getCurrentRawStream", None)
    except Exception:
        return None


_RAW_STREAM = _raw_stream_fn()


class PreparedCall:
    """A device entry point with its arguments checked and marshalled ONCE, for loops that call it again and again on
    the same buffers (a time stepper: PAPER.md Alg. 4 evaluates the sum twice per step on the same arrays).  Calling
    the object enqueues the work on torch's current stream (or the one given) of the tensors' device; the tensors are
    kept alive by the object.  Per call this costs one ctypes call (about 3 us) instead of the checks of the plain
    binding (about 10 us more), which is what a 512-point problem's 14 us kernel is measured against."""
    __slots__ = ("_fn", "_args", "_name", "_device", "_keep")

    def __init__(self, name, fn, args, device, keep):
        self._name, self._fn, self._args, self._device, self._keep = name, fn, tuple(args), device, keep

    def __call__(self, stream=None):
        import torch
        index = self._device.index
        if stream is None and torch.cuda.current_device() == index and _RAW_STREAM is not None:
            rc = self._fn(*self._args, _RAW_STREAM(index))          # the common case: one device query, one stream query
        else:
            with _on(self._device):
                rc = self._fn(*self._args, _stream_ptr(stream))
        if rc != VN_OK:
            raise VesnetError(rc, self._name)
        return self._keep[-1]


def prepare_arclength_weights(X, out) -> PreparedCall:
    """vn_arclength_weights(X, out=out) as a PreparedCall (returns `out` when called)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("out", out, (nves, npts), X.dtype)
    return PreparedCall("vn_arclength_weights", lib().vn_arclength_weights,
                        (X.data_ptr(), nves, npts, out.data_ptr(), _prec(X)), X.device, (X, out))


def prepare_farfield(X, F, W, out, mu: float = 1.0) -> PreparedCall:
    """vn_farfield(X, F, W, mu, out=out) as a PreparedCall (returns `out` when called)."""
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    _check_dev("out", out, X.shape, X.dtype)
    return PreparedCall("vn_farfield", lib().vn_farfield,
                        (X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu), out.data_ptr(), _prec(X)),
                        X.device, (X, F, W, out))


def prepare_farfield_fmm(X, F, W, out, mu: float = 1.0, order: int = 0) -> PreparedCall:
    """vn_farfield_fmm(X, F, W, mu, order, out=out) (plain sum, no near-field relation) as a PreparedCall."""
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    _check_dev("out", out, X.shape, X.dtype)
    return PreparedCall("vn_farfield_fmm", lib().vn_farfield_fmm,
                        (X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu), int(order), None, None,
                         out.data_ptr(), _prec(X)), X.device, (X, F, W, out))


def vn_noalloc_max_points() -> int:
    """Most points (nves * npts) vn_farfield_noalloc_f32 takes: the capacity of the library's static scratch."""
    return int(lib().vn_noalloc_max_points())


def vn_farfield_noalloc_f32(X, F, W, out, mu: float = 1.0, stream=None):
    """vn_farfield in single precision without any allocation (static scratch inside the library; see the header for
    the limit and the sharing rule).  `out` [nves, npts, 2] float32 is the caller's and required: the binding
    allocates nothing either.  Raises VesnetError(VN_ERR_TOO_LARGE) above vn_noalloc_max_points() points."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X, None, torch.float32)
    _check_dev("F", F, X.shape, torch.float32)
    _check_dev("W", W, (nves, npts), torch.float32)
    _check_dev("out", out, X.shape, torch.float32)
    with _on(X.device):
        rc = lib().vn_farfield_noalloc_f32(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu),
                                           out.data_ptr(), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_noalloc_f32")
    return out


def acc_words(dtype) -> int:
    """64-bit accumulator words per point of vn_farfield_partial: 2 for float32, 4 for float64."""
    import torch
    return 2 if dtype == torch.float32 else 4


def vn_farfield_partial(X, F, W, part: int, nparts: int, acc=None, gmax=None, stream=None):
    """Raw fixed-point accumulators of the blocks of part `part` of `nparts` (device tensors).
    Returns (acc int64 [nves*npts*words], gmax int64 [1])."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    n = nves * npts * acc_words(X.dtype)
    if acc is None:
        acc = torch.empty(n, dtype=torch.int64, device=X.device)
    if gmax is None:
        gmax = torch.empty(1, dtype=torch.int64, device=X.device)
    _check_dev("acc", acc, (n,), torch.int64)
    _check_dev("gmax", gmax, (1,), torch.int64)
    with _on(X.device):
        rc = lib().vn_farfield_partial(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, int(part), int(nparts),
                                       acc.data_ptr(), gmax.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_partial")
    return acc, gmax


def vn_farfield_finish(acc, gmax, npoints_total: int, dtype, mu: float = 1.0, out=None, stream=None):
    """U[count, 2] from a contiguous range of summed accumulators (count = acc.numel() / words per point)."""
    import torch
    _check_dev("acc", acc, None, torch.int64)
    _check_dev("gmax", gmax, (1,), torch.int64)
    count = acc.numel() // acc_words(dtype)
    if out is None:
        out = torch.empty((count, 2), dtype=dtype, device=acc.device)
    _check_dev("out", out, None, dtype)
    if out.numel() != 2 * count:
        raise ValueError("out must hold count x 2 values")
    with _on(acc.device):
        rc = lib().vn_farfield_finish(acc.data_ptr() if count else None, gmax.data_ptr(), int(npoints_total), count,
                                      float(mu), out.data_ptr() if count else None,
                                      VN_F32 if dtype == torch.float32 else VN_F64, _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_finish")
    return out


def vn_farfield_fmm(X, F, W, mu: float = 1.0, order: int = 0, out=None, stream=None, near_ptr=None, near_ves=None):
    """The far-field sum by the fast multipole method with `order` expansion terms (approximate, O(P); 0 = the
    default for the precision: 14 for float32, 38 for float64);
    with the CSR relation of vn_near_pairs the near vesicles' contributions are zeroed as in vn_farfield_masked."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    with _on(X.device):
        if near_ptr is not None:
            _check_dev("near_ptr", near_ptr, (nves * npts + 1,), torch.int64)
            _check_dev("near_ves", near_ves, None, torch.int32)
        rc = lib().vn_farfield_fmm(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu), int(order),
                                   None if near_ptr is None else near_ptr.data_ptr(),
                                   None if near_ptr is None or near_ves.numel() == 0 else near_ves.data_ptr(),
                                   out.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_fmm")
    return out


def vn_arclength_weights(X, out=None, stream=None):
    """W[v, j] = (2 pi / npts) |dX_v/dalpha| (device tensors; enqueues on the current stream)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    if out is None:
        out = torch.empty((nves, npts), dtype=X.dtype, device=X.device)
    _check_dev("out", out, (nves, npts), X.dtype)
    with _on(X.device):
        rc = lib().vn_arclength_weights(X.data_ptr(), nves, npts, out.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_arclength_weights")
    return out


def vn_near_pairs(X, W, near_ptr=None, near_ves=None, stream=None):
    """Near-field relation in CSR form (device tensors).  With near_ves=None the binding makes the
    count-only call, reads near_ptr[P] (one host synchronisation), allocates near_ves of exactly
    that size and calls again; pass both tensors to stay asynchronous.  Returns (near_ptr, near_ves)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("W", W, (nves, npts), X.dtype)
    P = nves * npts
    if near_ptr is None:
        near_ptr = torch.empty(P + 1, dtype=torch.int64, device=X.device)
    _check_dev("near_ptr", near_ptr, (P + 1,), torch.int64)
    L = lib()
    with _on(X.device):
        if near_ves is None:
            rc = L.vn_near_pairs(X.data_ptr(), W.data_ptr(), nves, npts, near_ptr.data_ptr(), None, 0,
                                 _prec(X), _stream_ptr(stream))
            if rc != VN_OK:
                raise VesnetError(rc, "vn_near_pairs")
            near_ves = torch.empty(int(near_ptr[P].item()), dtype=torch.int32, device=X.device)
            if near_ves.numel() == 0:
                return near_ptr, near_ves                  # the count-only call has filled near_ptr
        _check_dev("near_ves", near_ves, None, torch.int32)
        # a caller-supplied empty near_ves still gets the count-only call, so that near_ptr is always written
        rc = L.vn_near_pairs(X.data_ptr(), W.data_ptr(), nves, npts, near_ptr.data_ptr(),
                             near_ves.data_ptr() if near_ves.numel() else None, near_ves.numel(), _prec(X),
                             _stream_ptr(stream))
        if rc != VN_OK:
            raise VesnetError(rc, "vn_near_pairs")
    return near_ptr, near_ves


def vn_farfield_masked(X, F, W, near_ptr, near_ves, mu: float = 1.0, out=None, stream=None):
    """The paper's DirectSingleLayerIntegral: vn_farfield with the near vesicles' contribution zeroed."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    _check_dev("near_ptr", near_ptr, (nves * npts + 1,), torch.int64)
    _check_dev("near_ves", near_ves, None, torch.int32)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    with _on(X.device):
        rc = lib().vn_farfield_masked(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu),
                                      near_ptr.data_ptr(), near_ves.data_ptr() if near_ves.numel() else None,
                                      out.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_masked")
    return out


def vn_farfield_targets(Xt, X, F, W, mu: float = 1.0, out=None, stream=None, fmm_order: int = 0):
    """Velocity at free points Xt[nt, 2] induced by all vesicles (device tensors); fmm_order > 0 selects
    vn_farfield_targets_fmm with that expansion order (approximate, O(P + nt))."""
    import torch
    nves, npts, two = X.shape
    if two != 2 or Xt.dim() != 2 or Xt.shape[1] != 2:
        raise ValueError("X must be [nves, npts, 2] and Xt [nt, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    _check_dev("Xt", Xt, None, X.dtype)
    if out is None:
        out = torch.empty_like(Xt)
    _check_dev("out", out, Xt.shape, X.dtype)
    with _on(X.device):
        pt, po = (Xt.data_ptr(), out.data_ptr()) if Xt.numel() else (None, None)
        if fmm_order > 0:
            rc = lib().vn_farfield_targets_fmm(pt, Xt.shape[0], X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts,
                                               float(mu), int(fmm_order), po, _prec(X), _stream_ptr(stream))
        else:
            rc = lib().vn_farfield_targets(pt, Xt.shape[0], X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts,
                                           float(mu), po, _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_targets")
    return out


def vn_elastic_force(X, sigma, kappa_b: float = 1.0, out=None, stream=None):
    """F = -kappa_b X_ssss + (sigma X_s)_s (eq 2.7) for every vesicle (device tensors)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("sigma", sigma, (nves, npts), X.dtype)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    with _on(X.device):
        rc = lib().vn_elastic_force(X.data_ptr(), sigma.data_ptr(), nves, npts, float(kappa_b), out.data_ptr(),
                                    _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_elastic_force")
    return out


def vn_redistribute_arclength(X, out=None, stream=None):
    """Points of every vesicle redistributed equally in arclength (sec 4.2; device tensors)."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    with _on(X.device):
        rc = lib().vn_redistribute_arclength(X.data_ptr(), nves, npts, out.data_ptr(), _prec(X), _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_redistribute_arclength")
    return out


def _host_ptr(name, a, shape, dtype_name):
    """numpy array or CPU torch tensor -> (pointer, keepalive)."""
    import numpy as np
    if hasattr(a, "data_ptr"):                      # torch CPU tensor (possibly pinned)
        if a.is_cuda or not a.is_contiguous():
            raise ValueError(f"{name} must be a contiguous HOST tensor")
        if tuple(a.shape) != tuple(shape) or str(a.dtype).split(".")[-1] != dtype_name:
            raise ValueError(f"{name}: expected {dtype_name}{tuple(shape)}")
        return a.data_ptr(), a
    a = np.asarray(a)
    if not a.flags["C_CONTIGUOUS"] or a.shape != tuple(shape) or a.dtype.name != dtype_name:
        raise ValueError(f"{name}: expected C-contiguous {dtype_name}{tuple(shape)}")
    return a.ctypes.data, a


def vn_farfield_host(X, F, W=None, mu: float = 1.0, out=None):
    """Whole hot path from host buffers (numpy arrays or CPU torch tensors); synchronous.
    W=None computes the arclength weights on the device from X."""
    import numpy as np
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    dtype_name = str(X.dtype).split(".")[-1]
    if dtype_name not in ("float32", "float64"):
        raise TypeError("dtype must be float32 or float64")
    prec = VN_F32 if dtype_name == "float32" else VN_F64
    pX, kX = _host_ptr("X", X, (nves, npts, 2), dtype_name)
    pF, kF = _host_ptr("F", F, (nves, npts, 2), dtype_name)
    pW, kW = (None, None) if W is None else _host_ptr("W", W, (nves, npts), dtype_name)
    if out is None:
        out = np.empty((nves, npts, 2), dtype=dtype_name)
    pU, kU = _host_ptr("out", out, (nves, npts, 2), dtype_name)
    rc = lib().vn_farfield_host(pX, pF, pW, nves, npts, float(mu), pU, prec)
    if rc != VN_OK:
        raise VesnetError(rc, "vn_farfield_host")
    return out


def vn_plan_farfield(nves: int, npts: int, precision: int = VN_F32, resident_blocks: int = 148 * 3):
    """Host-only: the work decomposition of vn_farfield as a dict (no GPU needed)."""
    buf = (ctypes.c_int32 * 5)()
    rc = lib().vn_plan_farfield(nves, npts, precision, resident_blocks, buf)
    if rc != VN_OK:
        raise VesnetError(rc, "vn_plan_farfield")
    return dict(super_tile=buf[0], tiles_per_super_tile=buf[1], n_super_tiles=buf[2], n_chunks=buf[3], tile=buf[4])


def vn_profile_enable(enable: bool) -> None:
    lib().vn_profile_enable(1 if enable else 0)


def vn_profile_read(max_entries: int = 4096):
    """Durations (ms) of the pair kernel of every vn_farfield call since the last read."""
    buf = (ctypes.c_double * max_entries)()
    n = lib().vn_profile_read(buf, max_entries)
    if n < 0:
        raise VesnetError(VN_ERR_CUDA, "vn_profile_read")
    return [buf[i] for i in range(n)]


def vn_selfcheck(X, F, W, mu: float = 1.0, out=None, stream=None):
    """vn_farfield through the verification build of the pair kernels (ring reads compared with global memory, scratch
    poisoned).  Returns (U, mismatches); synchronous."""
    import torch
    nves, npts, two = X.shape
    if two != 2:
        raise ValueError("X must be [nves, npts, 2]")
    _check_dev("X", X)
    _check_dev("F", F, X.shape, X.dtype)
    _check_dev("W", W, (nves, npts), X.dtype)
    if out is None:
        out = torch.empty_like(X)
    _check_dev("out", out, X.shape, X.dtype)
    n = ctypes.c_int64(-1)
    with _on(X.device):
        rc = lib().vn_selfcheck(X.data_ptr(), F.data_ptr(), W.data_ptr(), nves, npts, float(mu), out.data_ptr(),
                                _prec(X), _stream_ptr(stream), ctypes.byref(n))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_selfcheck")
    return out, int(n.value)


def vn_pipe_peaks(stream=None):
    """Measured pipe rates in lane-operations per second: dict(ffma2, ffma, mufu, dfma, sms).  Synchronous."""
    buf = (ctypes.c_double * 8)()
    rc = lib().vn_pipe_peaks(buf, _stream_ptr(stream))
    if rc != VN_OK:
        raise VesnetError(rc, "vn_pipe_peaks")
    return dict(ffma2=buf[0], ffma=buf[1], mufu=buf[2], dfma=buf[3], sms=int(buf[4]), ffma2_noreuse=buf[5],
                dfma_noreuse=buf[6])


def vn_launch_count() -> int:
    return int(lib().vn_launch_count())


def vn_version() -> int:
    return int(lib().vn_version())
