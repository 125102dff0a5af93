"""ctypes binding of include/lipfit.h -- argument marshalling only.

Every step of the path runs in the CUDA kernels of liblipfit.so; nothing here computes a distance,
a bound, a neighbour or a penalty.  torch is used for device memory and streams only.  There is no
CPU fallback: if the library cannot be built/loaded, or no CUDA device is visible, the calls raise.
Nothing under oracle/ is imported from here.
"""
from __future__ import annotations

import ctypes as C
from typing import Optional, Sequence

import numpy as np

from . import build as _build

LIPFIT_L1, LIPFIT_L2, LIPFIT_LINF = 1, 2, 3
LIPFIT_MAX_DIM, LIPFIT_MAX_K = 32, 128

EXPORTS = [
    "lipfit_bounds", "lipfit_bounds_host", "lipfit_knn", "lipfit_knn_host",
    "lipfit_smooth_objective", "lipfit_smooth", "lipfit_smooth_host", "lipfit_lbfgs",
    "lipfit_status_string", "lipfit_version", "lipfit_launch_count", "lipfit_bounds_variant",
    "lipfit_set_timing", "lipfit_get_timing", "lipfit_knn_ex", "lipfit_release_workspace",
    "lipfit_lipschitz_constant", "lipfit_lipschitz_constant_host", "lipfit_knn_variant",
    "lipfit_distance_quantiles", "lipfit_local_lipschitz", "lipfit_values_local", "lipfit_bounds_topk",
    "lipfit_bounds_pruned", "lipfit_smooth_objective_pruned",
    "lipfit_bounds_ex", "lipfit_bounds_host_ex", "lipfit_bounds_region", "lipfit_pipe_throughput", "lipfit_pipe_name",
    "lipfit_bounds_noalloc",
]
LIPFIT_NOALLOC_MAX_RECORD_FLOATS, LIPFIT_NOALLOC_MAX_Q = 1 << 20, 1 << 19
LIPFIT_BOUNDS_AUTO, LIPFIT_BOUNDS_BRUTE, LIPFIT_BOUNDS_PRUNED = 0, 1, 2
LIPFIT_MAX_TOPK = 8
LIPFIT_LOCAL_KNOTS = 16
LIPFIT_KNN_NO_TENSOR_CORES = 1


__all__ = [n for n in EXPORTS if n not in ("lipfit_status_string", "lipfit_version", "lipfit_launch_count",
                                           "lipfit_bounds_variant", "lipfit_set_timing", "lipfit_get_timing",
                                           "lipfit_knn_variant", "lipfit_release_workspace", "lipfit_pipe_name",
                                           "lipfit_pipe_throughput")] + [
    "LIPFIT_L1", "LIPFIT_L2", "LIPFIT_LINF", "LIPFIT_MAX_DIM", "LIPFIT_MAX_K", "LIPFIT_MAX_TOPK",
    "LIPFIT_LOCAL_KNOTS", "LIPFIT_KNN_NO_TENSOR_CORES", "LIPFIT_BOUNDS_AUTO", "LIPFIT_BOUNDS_BRUTE",
    "LIPFIT_BOUNDS_PRUNED", "LIPFIT_NOALLOC_MAX_RECORD_FLOATS", "LIPFIT_NOALLOC_MAX_Q"]


class LipfitError(RuntimeError):
    def __init__(self, code: int, where: str):
        self.code = code
        super().__init__(f"{where}: {status_string(code)} ({code})")


class SmoothInfo(C.Structure):
    _fields_ = [("iters", C.c_int32), ("evals", C.c_int32), ("status", C.c_int32),
                ("reserved", C.c_int32), ("F0", C.c_double), ("F", C.c_double),
                ("gnorm_inf", C.c_double), ("max_violation0", C.c_double),
                ("max_violation", C.c_double)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_ if k != "reserved"}


class KnnInfo(C.Structure):
    _fields_ = [("fallbacks", C.c_int64), ("key_error_ratio", C.c_double), ("tensor_cores", C.c_int32),
                ("reserved", C.c_int32)]

    def as_dict(self):
        return {"fallbacks": int(self.fallbacks), "key_error_ratio": float(self.key_error_ratio),
                "tensor_cores": bool(self.tensor_cores)}


EVAL_FN = C.CFUNCTYPE(C.c_int, C.c_void_p, C.POINTER(C.c_double), C.POINTER(C.c_double),
                      C.POINTER(C.c_double))

_lib = None


def load():
    """Builds (if stale) and loads liblipfit.so; raises if that is impossible."""
    global _lib
    if _lib is not None:
        return _lib
    lib = C.CDLL(_build.build())
    P, i64, i32, f32, f64 = C.c_void_p, C.c_int64, C.c_int32, C.c_float, C.c_double
    lib.lipfit_bounds.argtypes = [P, P, i64, i32, P, i64, f32, P, i32, P, P, P, P, P]
    lib.lipfit_bounds_host.argtypes = lib.lipfit_bounds.argtypes
    lib.lipfit_bounds_ex.argtypes = [P, P, i64, i32, P, i64, f32, P, i32, P, P, P, P, i32, P, P]
    lib.lipfit_bounds_host_ex.argtypes = lib.lipfit_bounds_ex.argtypes
    lib.lipfit_bounds_noalloc.argtypes = lib.lipfit_bounds.argtypes
    lib.lipfit_bounds_region.argtypes = [P, P, i64, i32, P, i64, f32, P, P, P, i32, P, P, P, P, P]
    lib.lipfit_knn.argtypes = [P, i64, i32, P, i64, P, i32, i32, P, i32, P, P, P]
    lib.lipfit_knn_host.argtypes = lib.lipfit_knn.argtypes
    lib.lipfit_knn_ex.argtypes = [P, i64, i32, P, i64, P, i32, i32, P, i32, P, P, i32, P, P]
    lib.lipfit_smooth_objective_pruned.argtypes = [P, P, i64, i32, f32, P, i32, P, f32, P, P, P, P, P]
    lib.lipfit_smooth_objective.argtypes = [P, P, i64, i32, f32, P, i32, P, f32, P, P, P, P]
    lib.lipfit_smooth.argtypes = [P, P, i64, i32, f32, P, i32, P, f32, i32, f64, P, P, P]
    lib.lipfit_smooth_host.argtypes = lib.lipfit_smooth.argtypes
    lib.lipfit_lbfgs.argtypes = [i64, P, EVAL_FN, P, i32, f64, i32, P]
    lib.lipfit_bounds_pruned.argtypes = [P, P, i64, i32, P, i64, f32, P, i32, P, P, P, P, P, P]
    lib.lipfit_bounds_topk.argtypes = [P, P, i64, i32, P, i64, f32, P, i32, P, i32, P, P, P, P, P]
    lib.lipfit_distance_quantiles.argtypes = [P, i64, i32, i32, P, P, P, i64, i32, P, P]
    lib.lipfit_local_lipschitz.argtypes = [P, P, i64, i32, i32, P, P, i32, P, P]
    lib.lipfit_values_local.argtypes = [P, P, i64, i32, P, i64, i32, P, P, i32, P, P, P, P, P]
    lib.lipfit_lipschitz_constant.argtypes = [P, P, i64, i32, P, i32, P, P, P]
    lib.lipfit_lipschitz_constant_host.argtypes = lib.lipfit_lipschitz_constant.argtypes
    lib.lipfit_bounds_variant.argtypes = [i32, P, i32, C.c_char_p, i32]
    for name in EXPORTS:
        getattr(lib, name).restype = C.c_int
    lib.lipfit_status_string.restype = C.c_char_p
    lib.lipfit_status_string.argtypes = [C.c_int]
    lib.lipfit_version.restype = C.c_char_p
    lib.lipfit_launch_count.restype = C.c_int64
    lib.lipfit_set_timing.restype = None
    lib.lipfit_knn_variant.argtypes = [i32, i32, i32, i32, C.c_char_p, i32]
    lib.lipfit_release_workspace.argtypes = []
    lib.lipfit_pipe_throughput.argtypes = [i32, P, P, P]
    lib.lipfit_pipe_name.argtypes = [i32]
    lib.lipfit_pipe_name.restype = C.c_char_p
    lib.lipfit_set_timing.argtypes = [i32]
    lib.lipfit_get_timing.argtypes = [i32, P, P]
    _lib = lib
    return lib


def status_string(code: int) -> str:
    return load().lipfit_status_string(int(code)).decode()


def version() -> str:
    return load().lipfit_version().decode()


def launch_count() -> int:
    return int(load().lipfit_launch_count())


def pipe_throughput(which: int):
    """(name, lane-results / clk / SM, warp instructions / clk / SM) of instruction class `which` (diagnostic)."""
    a, b = C.c_double(0.0), C.c_double(0.0)
    _check(load().lipfit_pipe_throughput(int(which), C.cast(C.byref(a), C.c_void_p), C.cast(C.byref(b), C.c_void_p),
                                         _stream(None)), "lipfit_pipe_throughput")
    return load().lipfit_pipe_name(int(which)).decode(), float(a.value), float(b.value)


def release_workspace() -> None:
    """Hands the cached workspaces of the library's private memory pool back to the driver."""
    _check(load().lipfit_release_workspace(), "lipfit_release_workspace")


def knn_variant(d: int, side: int = 0, norm: int = LIPFIT_L2, tensor_cores: bool = True) -> str:
    buf = C.create_string_buffer(96)
    _check(load().lipfit_knn_variant(d, side, norm, 0 if tensor_cores else LIPFIT_KNN_NO_TENSOR_CORES, buf, 96),
           "lipfit_knn_variant")
    return buf.value.decode()


def set_timing(on: bool) -> None:
    load().lipfit_set_timing(1 if on else 0)


def get_timing(which: int):
    """(total device ms, launches) of dominant kernel `which` (0 bounds, 1 kNN select, 2 smooth)."""
    ms, n = C.c_double(0.0), C.c_int64(0)
    _check(load().lipfit_get_timing(int(which), C.cast(C.byref(ms), C.c_void_p),
                                    C.cast(C.byref(n), C.c_void_p)), "lipfit_get_timing")
    return float(ms.value), int(n.value)


def _check(rc: int, where: str):
    if rc != 0:
        raise LipfitError(rc, where)


def _host_params(d: int, mono_mask, weights):
    m = None if mono_mask is None else np.ascontiguousarray(mono_mask, dtype=np.int32).reshape(d)
    w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32).reshape(d)
    return m, w


def _np_ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def bounds_variant(d: int, mono_mask=None, norm: int = LIPFIT_L2) -> str:
    m, _ = _host_params(d, mono_mask, None)
    buf = C.create_string_buffer(96)
    _check(load().lipfit_bounds_variant(d, _np_ptr(m), norm, buf, 96), "lipfit_bounds_variant")
    return buf.value.decode()


# ---------------------------------------------------------------------------------------------
# Device-pointer entry points (torch CUDA tensors in, torch CUDA tensors out)
# ---------------------------------------------------------------------------------------------
def _torch():
    import torch
    if not torch.cuda.is_available():
        raise RuntimeError("paper_2606_04670_b200 needs a CUDA device (no CPU fallback)")
    return torch


def _dev_f32(t, ndim, name):
    torch = _torch()
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float32
            and t.dim() == ndim and t.is_contiguous()):
        raise TypeError(f"{name}: need a contiguous float32 CUDA tensor with {ndim} dims")
    return t


def _stream(stream):
    torch = _torch()
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


def lipfit_bounds_ex(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                     policy: int = LIPFIT_BOUNDS_AUTO, count_pairs: bool = False, stream=None):
    """(upper, lower, g[, pairs_evaluated list of 3]) through lipfit_bounds_ex with an explicit evaluation
    policy (LIPFIT_BOUNDS_AUTO / BRUTE / PRUNED); count_pairs=True synchronises."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    if Xq.shape[1] != d or y.shape[0] != N:
        raise ValueError("shape mismatch")
    m, w = _host_params(d, mono_mask, weights)
    outs = [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    n = (C.c_int64 * 3)()
    rc = load().lipfit_bounds_ex(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M), _np_ptr(m),
                                 int(norm), _np_ptr(w), outs[0].data_ptr(), outs[1].data_ptr(),
                                 outs[2].data_ptr(), int(policy), n if count_pairs else None, _stream(stream))
    _check(rc, "lipfit_bounds_ex")
    return (*outs, [int(v) for v in n]) if count_pairs else tuple(outs)


def lipfit_bounds_noalloc(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None, out=None,
                          stream=None):
    """(upper, lower, g) through lipfit_bounds_noalloc: no device allocation inside the library (fixed 8 MiB
    scratch; LipfitError -7 beyond N (DP + 4) <= 2^20 floats or Q <= 2^19).  `out`: three preallocated float32
    CUDA tensors of length Q (so that this binding allocates nothing either)."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    if Xq.shape[1] != d or y.shape[0] != N:
        raise ValueError("shape mismatch")
    m, w = _host_params(d, mono_mask, weights)
    outs = list(out) if out is not None else [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    for o in outs:
        if _dev_f32(o, 1, "out").shape[0] != Q:
            raise ValueError("shape mismatch")
    rc = load().lipfit_bounds_noalloc(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M), _np_ptr(m),
                                      int(norm), _np_ptr(w), outs[0].data_ptr(), outs[1].data_ptr(),
                                      outs[2].data_ptr(), _stream(stream))
    _check(rc, "lipfit_bounds_noalloc")
    return tuple(outs)


def lipfit_bounds_region(X, y, Xq, M: float, mon, a, b, norm: int = LIPFIT_L2, weights=None, stream=None):
    """(upper, lower, g) under monotonicity on parts of the domain: mon in {0..4}^d
    (0 unrestricted, 1..4 = case I..IV), thresholds a <= b per coordinate (host arrays)."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    if Xq.shape[1] != d or y.shape[0] != N:
        raise ValueError("shape mismatch")
    mon_h, w = _host_params(d, mon, weights)
    a_h = None if a is None else np.ascontiguousarray(a, dtype=np.float32).reshape(d)
    b_h = None if b is None else np.ascontiguousarray(b, dtype=np.float32).reshape(d)
    outs = [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    rc = load().lipfit_bounds_region(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M), _np_ptr(mon_h),
                                     _np_ptr(a_h), _np_ptr(b_h), int(norm), _np_ptr(w), outs[0].data_ptr(),
                                     outs[1].data_ptr(), outs[2].data_ptr(), _stream(stream))
    _check(rc, "lipfit_bounds_region")
    return tuple(outs)


def lipfit_bounds(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                  want: Sequence[str] = ("upper", "lower", "g"), stream=None):
    """(upper, lower, g) float32 CUDA tensors of length Q (None for those not in `want`)."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    if Xq.shape[1] != d or y.shape[0] != N:
        raise ValueError("shape mismatch")
    m, w = _host_params(d, mono_mask, weights)
    outs = {k: (torch.empty(Q, dtype=torch.float32, device=X.device) if k in want else None)
            for k in ("upper", "lower", "g")}
    ptr = {k: (None if v is None else C.c_void_p(v.data_ptr())) for k, v in outs.items()}
    rc = load().lipfit_bounds(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M),
                              _np_ptr(m), int(norm), _np_ptr(w), ptr["upper"], ptr["lower"],
                              ptr["g"], _stream(stream))
    _check(rc, "lipfit_bounds")
    return outs["upper"], outs["lower"], outs["g"]


def lipfit_bounds_pruned(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                         count_pairs: bool = False, stream=None):
    """(upper, lower, g[, pairs_evaluated]) as lipfit_bounds, evaluated with exact spatial pruning."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    if Xq.shape[1] != d or y.shape[0] != N:
        raise ValueError("shape mismatch")
    m, w = _host_params(d, mono_mask, weights)
    outs = [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    n = (C.c_int64 * 3)()
    rc = load().lipfit_bounds_pruned(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M), _np_ptr(m),
                                     int(norm), _np_ptr(w), outs[0].data_ptr(), outs[1].data_ptr(),
                                     outs[2].data_ptr(), n if count_pairs else None, _stream(stream))
    _check(rc, "lipfit_bounds_pruned")
    if count_pairs == "all":
        return (*outs, [int(v) for v in n])
    return (*outs, int(n[0])) if count_pairs else tuple(outs)


def lipfit_bounds_topk(X, y, Xq, M: float, wk, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                       stream=None):
    """(upper, lower, g): weighted sums of the k = len(wk) best bound values."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _host_params(d, mono_mask, weights)
    wk = np.ascontiguousarray(wk, dtype=np.float32)
    outs = [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    rc = load().lipfit_bounds_topk(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, float(M), _np_ptr(m),
                                   int(norm), _np_ptr(w), len(wk), _np_ptr(wk), outs[0].data_ptr(),
                                   outs[1].data_ptr(), outs[2].data_ptr(), _stream(stream))
    _check(rc, "lipfit_bounds_topk")
    return tuple(outs)


def lipfit_knn_ex(X, Xq, k: int, mono_mask=None, side: int = 0, norm: int = LIPFIT_L2, weights=None,
                  tensor_cores: bool = True, want_info: bool = True, stream=None):
    """(idx, dist, info dict or None) through lipfit_knn_ex: per-call kernel choice and diagnostics
    (want_info=True synchronises the stream)."""
    torch = _torch()
    X, Xq = _dev_f32(X, 2, "X"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _host_params(d, mono_mask, weights)
    idx = torch.empty((Q, k), dtype=torch.int32, device=X.device)
    dist = torch.empty((Q, k), dtype=torch.float32, device=X.device)
    info = KnnInfo()
    rc = load().lipfit_knn_ex(X.data_ptr(), N, d, Xq.data_ptr(), Q, _np_ptr(m), int(side), int(norm),
                              _np_ptr(w), int(k), idx.data_ptr(), dist.data_ptr(),
                              0 if tensor_cores else LIPFIT_KNN_NO_TENSOR_CORES,
                              C.cast(C.byref(info), C.c_void_p) if want_info else None, _stream(stream))
    _check(rc, "lipfit_knn_ex")
    return idx, dist, (info.as_dict() if want_info else None)


def lipfit_knn(X, Xq, k: int, mono_mask=None, side: int = 0, norm: int = LIPFIT_L2, weights=None,
               stream=None):
    """(idx int32 [Q,k], dist float32 [Q,k]) CUDA tensors, ascending distance."""
    torch = _torch()
    X, Xq = _dev_f32(X, 2, "X"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _host_params(d, mono_mask, weights)
    idx = torch.empty((Q, k), dtype=torch.int32, device=X.device)
    dist = torch.empty((Q, k), dtype=torch.float32, device=X.device)
    rc = load().lipfit_knn(X.data_ptr(), N, d, Xq.data_ptr(), Q, _np_ptr(m), int(side), int(norm),
                           _np_ptr(w), int(k), idx.data_ptr(), dist.data_ptr(), _stream(stream))
    _check(rc, "lipfit_knn")
    return idx, dist


def lipfit_smooth_objective(X, y, M: float, eps=None, mono_mask=None, norm: int = LIPFIT_L2,
                            weights=None, p: float = 1.0, want_grad: bool = True, stream=None):
    """(F python float, grad float32 CUDA tensor or None)."""
    torch = _torch()
    X, y = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y")
    N, d = X.shape
    m, w = _host_params(d, mono_mask, weights)
    if eps is not None:
        eps = _dev_f32(eps, 1, "eps")
    grad = torch.empty(N, dtype=torch.float32, device=X.device) if want_grad else None
    F = C.c_double(0.0)
    rc = load().lipfit_smooth_objective(
        X.data_ptr(), y.data_ptr(), N, d, float(M), _np_ptr(m), int(norm), _np_ptr(w), float(p),
        None if eps is None else C.c_void_p(eps.data_ptr()), C.cast(C.byref(F), C.c_void_p),
        None if grad is None else C.c_void_p(grad.data_ptr()), _stream(stream))
    _check(rc, "lipfit_smooth_objective")
    return float(F.value), grad


def lipfit_smooth_objective_pruned(X, y, M: float, eps=None, mono_mask=None, norm: int = LIPFIT_L2,
                                   weights=None, p: float = 1.0, want_grad: bool = True, count_pairs: bool = False,
                                   stream=None):
    """(F, grad[, pairs_evaluated]) as lipfit_smooth_objective, evaluated with exact spatial pruning."""
    torch = _torch()
    X, y = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y")
    N, d = X.shape
    m, w = _host_params(d, mono_mask, weights)
    if eps is not None:
        eps = _dev_f32(eps, 1, "eps")
    grad = torch.empty(N, dtype=torch.float32, device=X.device) if want_grad else None
    F = C.c_double(0.0)
    n = C.c_int64(0)
    rc = load().lipfit_smooth_objective_pruned(
        X.data_ptr(), y.data_ptr(), N, d, float(M), _np_ptr(m), int(norm), _np_ptr(w), float(p),
        None if eps is None else C.c_void_p(eps.data_ptr()), C.cast(C.byref(F), C.c_void_p),
        None if grad is None else C.c_void_p(grad.data_ptr()),
        C.cast(C.byref(n), C.c_void_p) if count_pairs else None, _stream(stream))
    _check(rc, "lipfit_smooth_objective_pruned")
    return (float(F.value), grad, int(n.value)) if count_pairs else (float(F.value), grad)


def lipfit_lipschitz_constant(X, y, mono_mask=None, norm: int = LIPFIT_L2, weights=None, stream=None):
    """Smallest Lipschitz constant consistent with the data as a 1-element
    float32 CUDA tensor (asynchronous on the stream)."""
    torch = _torch()
    X, y = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y")
    N, d = X.shape
    if y.shape[0] != N:
        raise ValueError("shape mismatch")
    m, w = _host_params(d, mono_mask, weights)
    out = torch.empty(1, dtype=torch.float32, device=X.device)
    rc = load().lipfit_lipschitz_constant(X.data_ptr(), y.data_ptr(), N, d, _np_ptr(m), int(norm),
                                          _np_ptr(w), out.data_ptr(), _stream(stream))
    _check(rc, "lipfit_lipschitz_constant")
    return out


def lipfit_lipschitz_constant_host(X, y, mono_mask=None, norm: int = LIPFIT_L2, weights=None) -> float:
    X, y = _host_f32(X, 2), _host_f32(y, 1)
    N, d = X.shape
    m, w = _host_params(d, mono_mask, weights)
    out = np.zeros(1, dtype=np.float32)
    rc = load().lipfit_lipschitz_constant_host(_np_ptr(X), _np_ptr(y), N, d, _np_ptr(m), int(norm),
                                               _np_ptr(w), _np_ptr(out), None)
    _check(rc, "lipfit_lipschitz_constant_host")
    return float(out[0])


def lipfit_distance_quantiles(X, pair_i, pair_k, J: int = LIPFIT_LOCAL_KNOTS, norm: int = LIPFIT_L2,
                              weights=None, stream=None):
    """Knots (numpy float32 [J]) = nearest-rank quantiles of the sampled inter-point distances."""
    torch = _torch()
    X = _dev_f32(X, 2, "X")
    N, d = X.shape
    _, w = _host_params(d, None, weights)
    pi = pair_i.to(device=X.device, dtype=torch.int32).contiguous()
    pk = pair_k.to(device=X.device, dtype=torch.int32).contiguous()
    knots = np.zeros(J, dtype=np.float32)
    rc = load().lipfit_distance_quantiles(X.data_ptr(), N, d, int(norm), _np_ptr(w), pi.data_ptr(),
                                          pk.data_ptr(), pi.numel(), int(J), _np_ptr(knots), _stream(stream))
    _check(rc, "lipfit_distance_quantiles")
    return knots


def lipfit_local_lipschitz(X, y, knots, norm: int = LIPFIT_L2, weights=None, stream=None):
    """Step tables M_k as a float32 CUDA tensor [N, J]."""
    torch = _torch()
    X, y = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y")
    N, d = X.shape
    _, w = _host_params(d, None, weights)
    kn = np.ascontiguousarray(knots, dtype=np.float32)
    table = torch.empty((N, len(kn)), dtype=torch.float32, device=X.device)
    rc = load().lipfit_local_lipschitz(X.data_ptr(), y.data_ptr(), N, d, int(norm), _np_ptr(w), _np_ptr(kn),
                                       len(kn), table.data_ptr(), _stream(stream))
    _check(rc, "lipfit_local_lipschitz")
    return table


def lipfit_values_local(X, y, Xq, knots, table, norm: int = LIPFIT_L2, weights=None, stream=None):
    """(upper, lower, g) with M replaced by M_k(D(x, x^k))."""
    torch = _torch()
    X, y, Xq = _dev_f32(X, 2, "X"), _dev_f32(y, 1, "y"), _dev_f32(Xq, 2, "Xq")
    N, d = X.shape
    Q = Xq.shape[0]
    _, w = _host_params(d, None, weights)
    kn = np.ascontiguousarray(knots, dtype=np.float32)
    table = _dev_f32(table, 2, "table")
    outs = [torch.empty(Q, dtype=torch.float32, device=X.device) for _ in range(3)]
    rc = load().lipfit_values_local(X.data_ptr(), y.data_ptr(), N, d, Xq.data_ptr(), Q, int(norm), _np_ptr(w),
                                    _np_ptr(kn), len(kn), table.data_ptr(), outs[0].data_ptr(),
                                    outs[1].data_ptr(), outs[2].data_ptr(), _stream(stream))
    _check(rc, "lipfit_values_local")
    return tuple(outs)


def lipfit_smooth(X, y_inout, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                  p: float = 1.0, max_iter: int = 200, tol_grad: float = 1e-7, stream=None):
    """Smooths y in place (y <- y + eps); returns (eps CUDA tensor, info dict)."""
    torch = _torch()
    X, y_inout = _dev_f32(X, 2, "X"), _dev_f32(y_inout, 1, "y_inout")
    N, d = X.shape
    m, w = _host_params(d, mono_mask, weights)
    eps = torch.empty(N, dtype=torch.float32, device=X.device)
    info = SmoothInfo()
    rc = load().lipfit_smooth(X.data_ptr(), y_inout.data_ptr(), N, d, float(M), _np_ptr(m),
                              int(norm), _np_ptr(w), float(p), int(max_iter), float(tol_grad),
                              eps.data_ptr(), C.cast(C.byref(info), C.c_void_p), _stream(stream))
    _check(rc, "lipfit_smooth")
    return eps, info.as_dict()


# ---------------------------------------------------------------------------------------------
# Host-pointer entry points (numpy in, numpy out; copies happen inside the library)
# ---------------------------------------------------------------------------------------------
def _host_f32(a, ndim):
    a = np.ascontiguousarray(a, dtype=np.float32)
    if a.ndim != ndim:
        raise ValueError("bad rank")
    return a


def lipfit_bounds_host(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                       out=None, stream_ptr: Optional[int] = None):
    """numpy in / numpy out through lipfit_bounds_host.  `out` may be a preallocated (e.g. pinned)
    tuple of three float32 arrays of length Q."""
    return lipfit_bounds_host_ex(X, y, Xq, M, mono_mask, norm, weights, out, stream_ptr, None)


def lipfit_bounds_host_ex(X, y, Xq, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                          out=None, stream_ptr: Optional[int] = None, policy: Optional[int] = LIPFIT_BOUNDS_AUTO):
    """As lipfit_bounds_host with an explicit evaluation policy (policy=None: the plain entry point)."""
    X, y, Xq = _host_f32(X, 2), _host_f32(y, 1), _host_f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _host_params(d, mono_mask, weights)
    up, lo, g = out if out is not None else (np.empty(Q, np.float32) for _ in range(3))
    if policy is None:
        rc = load().lipfit_bounds_host(_np_ptr(X), _np_ptr(y), N, d, _np_ptr(Xq), Q, float(M), _np_ptr(m),
                                       int(norm), _np_ptr(w), _np_ptr(up), _np_ptr(lo), _np_ptr(g),
                                       C.c_void_p(stream_ptr or 0))
    else:
        rc = load().lipfit_bounds_host_ex(_np_ptr(X), _np_ptr(y), N, d, _np_ptr(Xq), Q, float(M), _np_ptr(m),
                                          int(norm), _np_ptr(w), _np_ptr(up), _np_ptr(lo), _np_ptr(g),
                                          int(policy), None, C.c_void_p(stream_ptr or 0))
    _check(rc, "lipfit_bounds_host")
    return up, lo, g


def lipfit_knn_host(X, Xq, k: int, mono_mask=None, side: int = 0, norm: int = LIPFIT_L2,
                    weights=None, stream_ptr: Optional[int] = None):
    X, Xq = _host_f32(X, 2), _host_f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _host_params(d, mono_mask, weights)
    idx = np.empty((Q, k), np.int32)
    dist = np.empty((Q, k), np.float32)
    rc = load().lipfit_knn_host(_np_ptr(X), N, d, _np_ptr(Xq), Q, _np_ptr(m), int(side), int(norm),
                                _np_ptr(w), int(k), _np_ptr(idx), _np_ptr(dist),
                                C.c_void_p(stream_ptr or 0))
    _check(rc, "lipfit_knn_host")
    return idx, dist


def lipfit_smooth_host(X, y, M: float, mono_mask=None, norm: int = LIPFIT_L2, weights=None,
                       p: float = 1.0, max_iter: int = 200, tol_grad: float = 1e-7,
                       stream_ptr: Optional[int] = None):
    """Returns (y_smoothed, eps, info dict); the input y is not modified."""
    X = _host_f32(X, 2)
    y = np.array(y, dtype=np.float32, copy=True)
    N, d = X.shape
    m, w = _host_params(d, mono_mask, weights)
    eps = np.empty(N, np.float32)
    info = SmoothInfo()
    rc = load().lipfit_smooth_host(_np_ptr(X), _np_ptr(y), N, d, float(M), _np_ptr(m), int(norm),
                                   _np_ptr(w), float(p), int(max_iter), float(tol_grad), _np_ptr(eps),
                                   C.cast(C.byref(info), C.c_void_p), C.c_void_p(stream_ptr or 0))
    _check(rc, "lipfit_smooth_host")
    return y, eps, info.as_dict()


def lipfit_lbfgs(fun, x0, max_iter: int = 200, tol_grad: float = 1e-8, history: int = 20):
    """Host LBFGS of the library on a Python callable fun(x) -> (f, grad).  No GPU involved."""
    x = np.array(x0, dtype=np.float64, copy=True)
    n = x.size

    def _cb(_user, xp, fp, gp):
        xv = np.ctypeslib.as_array(xp, shape=(n,))
        f, g = fun(xv.copy())
        fp[0] = float(f)
        np.ctypeslib.as_array(gp, shape=(n,))[:] = g
        return 0

    cb = EVAL_FN(_cb)
    info = SmoothInfo()
    rc = load().lipfit_lbfgs(n, _np_ptr(x), cb, None, int(max_iter), float(tol_grad), int(history),
                             C.cast(C.byref(info), C.c_void_p))
    _check(rc, "lipfit_lbfgs")
    return x, info.as_dict()
