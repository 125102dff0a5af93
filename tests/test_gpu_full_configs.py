"""GPU parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times.

The oracle cannot afford the full configs, so each test compares sampled outputs it can compute one
by one (the deterministic subset of inputs.oracle_subset), and adds properties that hold at any size.
Config 1 is small enough to be checked in full (tests/test_gpu_bounds.py::test_config1_full).
"""
import numpy as np
import pytest

import oracle
from inputs import make_workload, oracle_subset

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).to("cuda:0")


def _bounds_full(wl, y=None, n_sample=200):
    import torch
    import paper_2606_04670_b200 as L
    yv = wl.y if y is None else y
    up, lo, g = L.lipfit_bounds(_dev(wl.X), _dev(yv), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
    torch.cuda.synchronize()
    up, lo, g = up.cpu().numpy(), lo.cpu().numpy(), g.cpu().numpy()
    sel = oracle_subset(wl.Q, n_sample)
    U, Lo, G = oracle.bounds(wl.X, yv, wl.Xq[sel], wl.M, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range                                   # the north_star bar (R18: range of the INPUT y)
    assert np.abs(up[sel] - U).max() <= tol
    assert np.abs(lo[sel] - Lo).max() <= tol
    assert np.abs(g[sel] - G).max() <= tol
    # any size: g is the midpoint; every bound is finite; upper >= min y, lower <= max y
    assert np.all(np.isfinite(up)) and np.all(np.isfinite(lo))
    assert np.abs(g - 0.5 * (up.astype(np.float64) + lo)).max() <= 1e-6 * max(1.0, np.abs(g).max())
    assert up.min() >= yv.min() and lo.max() <= yv.max()
    return up, lo, g


def test_config2_full():
    wl = make_workload(2)
    _bounds_full(wl, n_sample=300)


def test_config3_full():
    wl = make_workload(3)
    _bounds_full(wl, n_sample=96)


def test_config4_full():
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(4)
    idx, dist, info = L.lipfit_knn_ex(_dev(wl.X), _dev(wl.Xq), wl.k, None, 0, wl.norm)
    assert info["fallbacks"] <= wl.Q // 1000                  # the certificate holds almost everywhere
    assert info["key_error_ratio"] <= 1.0 and info["tensor_cores"]
    idx, dist = idx.cpu().numpy(), dist.cpu().numpy()
    sel = oracle_subset(wl.Q, 48)
    oi, od = oracle.knn(wl.X, wl.Xq[sel], wl.k, None, 0, wl.norm)
    np.testing.assert_array_equal(idx[sel], oi)               # no ties in general position: exact index parity
    np.testing.assert_array_equal(dist[sel], od.astype(np.float32))
    # P12 at full size: ascending, in range, distinct; the k-th distance bounds a random non-member
    assert np.all(np.diff(dist, axis=1) >= 0)
    assert idx.min() >= 0 and idx.max() < wl.N
    rows = oracle_subset(wl.Q, 4000)
    srt = np.sort(idx[rows], axis=1)
    assert np.all(np.diff(srt, axis=1) > 0)
    rng = np.random.default_rng(0)
    other = rng.integers(0, wl.N, len(rows))
    d_other = np.sqrt(((wl.Xq[rows].astype(np.float64) - wl.X[other].astype(np.float64)) ** 2).sum(axis=1))
    member = (idx[rows] == other[:, None]).any(axis=1)
    assert np.all(member | (d_other >= dist[rows, -1].astype(np.float64) * (1 - 1e-6)))


def test_config5_objective_full():
    import paper_2606_04670_b200 as L
    wl = make_workload(5, Q=1)
    N = wl.N
    rng = np.random.default_rng(7)
    rows = oracle_subset(N, 48)
    X, y = _dev(wl.X), _dev(wl.y)
    for eps in (None, (0.05 * rng.standard_normal(N)).astype(np.float32)):
        e64 = np.zeros(N) if eps is None else eps.astype(np.float64)
        F, grad = L.lipfit_smooth_objective(X, y, wl.M, None if eps is None else _dev(eps), wl.mask, wl.norm,
                                            None, wl.p)
        grad = grad.cpu().numpy().astype(np.float64)
        g_ref, _ = oracle.smooth_rows(wl.X, wl.y, wl.M, e64, rows, wl.mask, wl.norm, None, wl.p)
        # gradient rows against the oracle; scale = the largest sampled component (the full-N max is unaffordable)
        assert np.abs(grad[rows] - g_ref).max() <= 1e-5 * np.abs(g_ref).max()
        # P14: the pair terms cancel in the sum of the gradient: sum_i dF/deps_i = (2/p) sum_i eps_i
        assert abs(grad.sum() - 2.0 * e64.sum() / wl.p) <= 1e-6 * np.abs(grad).sum()
        # F against its own (oracle-checked) gradient: central difference along a random direction; F is
        # piecewise quadratic, so this is exact up to the kinks crossed and the fp32 resolution of F
        v = rng.choice([-1.0, 1.0], N)
        h = 2e-3
        base = np.zeros(N, np.float32) if eps is None else eps
        Fp, _ = L.lipfit_smooth_objective(X, y, wl.M, _dev((base + h * v).astype(np.float32)), wl.mask,
                                          wl.norm, None, wl.p, want_grad=False)
        Fm, _ = L.lipfit_smooth_objective(X, y, wl.M, _dev((base - h * v).astype(np.float32)), wl.mask,
                                          wl.norm, None, wl.p, want_grad=False)
        dd = (Fp - Fm) / (2 * h)
        assert abs(dd - grad @ v) <= 2e-3 * max(abs(dd), np.abs(grad).sum() / np.sqrt(N)), (dd, grad @ v)
        assert F > 0


def test_config5_smooth_then_bounds_full():
    """S(3) of SURVEY.md §8(c): the LBFGS trajectory is unpinned by design (R14); at full N the checks
    are: F decreases, the worst violation drops, sum(eps) ~ 0 (P14), and the bounds evaluated on the
    GPU's own smoothed z match the oracle's bounds ON THE SAME z."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(5)
    yd = _dev(wl.y.copy())
    eps, info = L.lipfit_smooth(_dev(wl.X), yd, wl.M, wl.mask, wl.norm, None, wl.p, wl.max_iter, 1e-6)
    torch.cuda.synchronize()
    info = info if isinstance(info, dict) else info.as_dict()
    assert info["F"] < 0.05 * info["F0"]
    assert info["max_violation"] < 0.5 * info["max_violation0"]
    e = eps.cpu().numpy().astype(np.float64)
    assert abs(e.sum()) <= 1e-3 * np.abs(e).sum()
    z = yd.cpu().numpy()
    np.testing.assert_allclose(z, wl.y + eps.cpu().numpy(), rtol=0, atol=1e-6)   # y <- y + eps
    _bounds_full(wl, y=z, n_sample=200)
