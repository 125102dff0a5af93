"""CPU oracle for the LipFit hot path -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Thin ctypes shim over oracle/lipfit_oracle.c (plain C, fp64) plus the
smoothing minimiser (scipy L-BFGS-B around the C objective: a library routine
used as a step; Eq.(7)'s minimiser is unique, so the optimiser is immaterial).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It imports nothing from
paper_2606_04670_b200/ and vice versa.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = None


def load():
    global _lib
    if _lib is None:
        lib = C.CDLL(_build.build())
        i64, i32, f64 = C.c_int64, C.c_int32, C.c_double
        P = C.c_void_p
        lib.oracle_bounds.argtypes = [P, P, i64, i32, P, i64, f64, P, i32, P, P, P, P]
        lib.oracle_knn.argtypes = [P, i64, i32, P, i64, P, i32, i32, P, i32, P, P]
        lib.oracle_smooth_objective.argtypes = [P, P, i64, i32, f64, P, i32, P, f64, P, P, P]
        lib.oracle_max_violation.argtypes = [P, P, i64, i32, f64, P, i32, P, P, P]
        lib.oracle_smooth_rows.argtypes = [P, P, i64, i32, f64, P, i32, P, f64, P, P, i64, P, P]
        lib.oracle_lipschitz_constant.argtypes = [P, P, i64, i32, P, i32, P, P]
        lib.oracle_distance_quantiles.argtypes = [P, i64, i32, i32, P, P, P, i64, i32, P]
        lib.oracle_local_lipschitz.argtypes = [P, P, i64, i32, i32, P, P, i32, P]
        lib.oracle_values_local.argtypes = [P, P, i64, i32, P, i64, i32, P, P, i32, P, P, P, P]
        lib.oracle_bounds_topk.argtypes = [P, P, i64, i32, P, i64, f64, P, i32, P, i32, P, P, P, P]
        lib.oracle_bounds_topk.restype = C.c_int
        lib.oracle_local_lipschitz_rows.argtypes = [P, P, i64, i32, i32, P, P, i32, P, i64, P]
        lib.oracle_local_lipschitz_rows.restype = C.c_int
        lib.oracle_bounds_region.argtypes = [P, P, i64, i32, P, i64, f64, P, P, P, i32, P, P, P, P]
        lib.oracle_bounds_region.restype = C.c_int
        for fn in (lib.oracle_distance_quantiles, lib.oracle_local_lipschitz, lib.oracle_values_local):
            fn.restype = C.c_int
        for fn in (lib.oracle_bounds, lib.oracle_knn, lib.oracle_smooth_objective,
                   lib.oracle_max_violation, lib.oracle_num_threads, lib.oracle_smooth_rows,
                   lib.oracle_lipschitz_constant):
            fn.restype = C.c_int
        _lib = lib
    return _lib


def _f32(a, ndim):
    a = np.ascontiguousarray(a, dtype=np.float32)
    assert a.ndim == ndim
    return a


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


def _params(d, mask, weights):
    m = None if mask is None else np.ascontiguousarray(mask, dtype=np.int32).reshape(d)
    w = None if weights is None else np.ascontiguousarray(weights, dtype=np.float32).reshape(d)
    return m, w


def num_threads() -> int:
    return int(load().oracle_num_threads())


def bounds(X, y, Xq, M, mask=None, norm=2, weights=None):
    """(upper, lower, g) as float64 arrays of length Q.  Eq.(2),(3),(4)."""
    X, y, Xq = _f32(X, 2), _f32(y, 1), _f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _params(d, mask, weights)
    up, lo, g = (np.empty(Q, dtype=np.float64) for _ in range(3))
    rc = load().oracle_bounds(_ptr(X), _ptr(y), N, d, _ptr(Xq), Q, float(np.float32(M)),
                              _ptr(m), int(norm), _ptr(w), _ptr(up), _ptr(lo), _ptr(g))
    if rc:
        raise ValueError(f"oracle_bounds rc={rc}")
    return up, lo, g


def bounds_topk(X, y, Xq, M, wk, mask=None, norm=2, weights=None):
    """(upper, lower, g): weighted sums of the k = len(wk) best bound values."""
    X, y, Xq = _f32(X, 2), _f32(y, 1), _f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _params(d, mask, weights)
    wk = np.ascontiguousarray(wk, dtype=np.float32)
    U, L, G = (np.empty(Q, dtype=np.float64) for _ in range(3))
    rc = load().oracle_bounds_topk(_ptr(X), _ptr(y), N, d, _ptr(Xq), Q, float(np.float32(M)), _ptr(m),
                                   int(norm), _ptr(w), len(wk), _ptr(wk), _ptr(U), _ptr(L), _ptr(G))
    if rc:
        raise ValueError(f"oracle_bounds_topk rc={rc}")
    return U, L, G


def knn(X, Xq, k, mask=None, side=0, norm=2, weights=None):
    """(idx int32 [Q,k], dist float64 [Q,k]) ascending; ties by lower index."""
    X, Xq = _f32(X, 2), _f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    m, w = _params(d, mask, weights)
    idx = np.empty((Q, k), dtype=np.int32)
    dist = np.empty((Q, k), dtype=np.float64)
    rc = load().oracle_knn(_ptr(X), N, d, _ptr(Xq), Q, _ptr(m), int(side), int(norm), _ptr(w),
                           int(k), _ptr(idx), _ptr(dist))
    if rc:
        raise ValueError(f"oracle_knn rc={rc}")
    return idx, dist


def smooth_objective(X, y, M, eps, mask=None, norm=2, weights=None, p=1.0, want_grad=True):
    """F(eps) of Eq.(7) and its gradient (float64)."""
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    m, w = _params(d, mask, weights)
    eps = np.ascontiguousarray(eps, dtype=np.float64).reshape(N)
    F = C.c_double(0.0)
    grad = np.empty(N, dtype=np.float64) if want_grad else None
    rc = load().oracle_smooth_objective(_ptr(X), _ptr(y), N, d, float(np.float32(M)), _ptr(m),
                                        int(norm), _ptr(w), float(p), _ptr(eps), C.byref(F),
                                        _ptr(grad))
    if rc:
        raise ValueError(f"oracle_smooth_objective rc={rc}")
    return float(F.value), grad


def max_violation(X, y, M, eps=None, mask=None, norm=2, weights=None):
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    m, w = _params(d, mask, weights)
    e = None if eps is None else np.ascontiguousarray(eps, dtype=np.float64).reshape(N)
    out = C.c_double(0.0)
    rc = load().oracle_max_violation(_ptr(X), _ptr(y), N, d, float(np.float32(M)), _ptr(m),
                                     int(norm), _ptr(w), _ptr(e), C.byref(out))
    if rc:
        raise ValueError(f"oracle_max_violation rc={rc}")
    return float(out.value)


def smooth_rows(X, y, M, eps, rows, mask=None, norm=2, weights=None, p=1.0):
    """dF/deps_i and the row share of F for the listed rows i (Eq.(7)); returns (grad_rows, f_rows)."""
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    m, w = _params(d, mask, weights)
    eps = np.ascontiguousarray(eps, dtype=np.float64).reshape(N)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    g = np.empty(len(rows), dtype=np.float64)
    f = np.empty(len(rows), dtype=np.float64)
    rc = load().oracle_smooth_rows(_ptr(X), _ptr(y), N, d, float(np.float32(M)), _ptr(m), int(norm),
                                   _ptr(w), float(p), _ptr(eps), _ptr(rows), len(rows), _ptr(g), _ptr(f))
    if rc:
        raise ValueError(f"oracle_smooth_rows rc={rc}")
    return g, f


def lipschitz_constant(X, y, mask=None, norm=2, weights=None) -> float:
    """Smallest M consistent with the data."""
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    m, w = _params(d, mask, weights)
    out = C.c_double(0.0)
    rc = load().oracle_lipschitz_constant(_ptr(X), _ptr(y), N, d, _ptr(m), int(norm), _ptr(w),
                                          C.byref(out))
    if rc:
        raise ValueError(f"oracle_lipschitz_constant rc={rc}")
    return float(out.value)


def distance_quantiles(X, pair_i, pair_k, J, norm=2, weights=None):
    """J spline knots (float64): nearest-rank quantiles of the sampled inter-point distances."""
    X = _f32(X, 2)
    N, d = X.shape
    _, w = _params(d, None, weights)
    pi = np.ascontiguousarray(pair_i, dtype=np.int32)
    pk = np.ascontiguousarray(pair_k, dtype=np.int32)
    knots = np.empty(J, dtype=np.float64)
    rc = load().oracle_distance_quantiles(_ptr(X), N, d, int(norm), _ptr(w), _ptr(pi), _ptr(pk), len(pi),
                                          int(J), _ptr(knots))
    if rc:
        raise ValueError(f"oracle_distance_quantiles rc={rc}")
    return knots


def local_lipschitz(X, y, knots, norm=2, weights=None):
    """table [N, J] (float64) of the per-datum step functions M_k."""
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    _, w = _params(d, None, weights)
    knots = np.ascontiguousarray(knots, dtype=np.float64)
    table = np.empty((N, len(knots)), dtype=np.float64)
    rc = load().oracle_local_lipschitz(_ptr(X), _ptr(y), N, d, int(norm), _ptr(w), _ptr(knots), len(knots),
                                       _ptr(table))
    if rc:
        raise ValueError(f"oracle_local_lipschitz rc={rc}")
    return table


def local_lipschitz_rows(X, y, knots, rows, norm=2, weights=None):
    """table rows [len(rows), J] (float64) of the step functions M_k of the listed data only."""
    X, y = _f32(X, 2), _f32(y, 1)
    N, d = X.shape
    _, w = _params(d, None, weights)
    knots = np.ascontiguousarray(knots, dtype=np.float64)
    rows = np.ascontiguousarray(rows, dtype=np.int64)
    out = np.empty((len(rows), len(knots)), dtype=np.float64)
    rc = load().oracle_local_lipschitz_rows(_ptr(X), _ptr(y), N, d, int(norm), _ptr(w), _ptr(knots), len(knots),
                                            _ptr(rows), len(rows), _ptr(out))
    if rc:
        raise ValueError(f"oracle_local_lipschitz_rows rc={rc}")
    return out


def bounds_region(X, y, Xq, M, mon, a, b, norm=2, weights=None):
    """(upper, lower, g) under monotonicity on parts of the domain (reading R26)."""
    X, y, Xq = _f32(X, 2), _f32(y, 1), _f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    _, w = _params(d, None, weights)
    mon = None if mon is None else np.ascontiguousarray(mon, dtype=np.int32).reshape(d)
    a = None if a is None else np.ascontiguousarray(a, dtype=np.float32).reshape(d)
    b = None if b is None else np.ascontiguousarray(b, dtype=np.float32).reshape(d)
    U, L, G = (np.empty(Q, dtype=np.float64) for _ in range(3))
    rc = load().oracle_bounds_region(_ptr(X), _ptr(y), N, d, _ptr(Xq), Q, float(np.float32(M)), _ptr(mon), _ptr(a), _ptr(b),
                                     int(norm), _ptr(w), _ptr(U), _ptr(L), _ptr(G))
    if rc:
        raise ValueError(f"oracle_bounds_region rc={rc}")
    return U, L, G


def values_local(X, y, Xq, knots, table, norm=2, weights=None):
    """(upper, lower, g) with M replaced by M_k(D(x, x^k))."""
    X, y, Xq = _f32(X, 2), _f32(y, 1), _f32(Xq, 2)
    N, d = X.shape
    Q = Xq.shape[0]
    _, w = _params(d, None, weights)
    knots = np.ascontiguousarray(knots, dtype=np.float64)
    table = np.ascontiguousarray(table, dtype=np.float64).reshape(N, len(knots))
    U, L, G = (np.empty(Q, dtype=np.float64) for _ in range(3))
    rc = load().oracle_values_local(_ptr(X), _ptr(y), N, d, _ptr(Xq), Q, int(norm), _ptr(w), _ptr(knots),
                                    len(knots), _ptr(table), _ptr(U), _ptr(L), _ptr(G))
    if rc:
        raise ValueError(f"oracle_values_local rc={rc}")
    return U, L, G


def smooth(X, y, M, mask=None, norm=2, weights=None, p=1.0, max_iter=10000, gtol=1e-12):
    """Minimiser eps* of Eq.(7) from eps=0 ("an unconstrained
    minimisation method like LBFGS").  F is strongly convex (Hessian >= 2/p I),
    so eps* is unique and any convergent optimiser gives it; this uses
    scipy.optimize.minimize(L-BFGS-B, jac=True) on the C objective above.
    Returns (eps*, info dict)."""
    from scipy.optimize import minimize

    N = np.asarray(X).shape[0]

    def fun(e):
        return smooth_objective(X, y, M, e, mask, norm, weights, p)

    res = minimize(fun, np.zeros(N), jac=True, method="L-BFGS-B",
                   options=dict(maxiter=max_iter, maxfun=50 * max_iter, gtol=gtol, ftol=0.0,
                                maxcor=30, maxls=60))
    F, grad = fun(res.x)
    return res.x, dict(F=F, gnorm_inf=float(np.abs(grad).max()), iters=int(res.nit),
                       evals=int(res.nfev), message=str(res.message))
