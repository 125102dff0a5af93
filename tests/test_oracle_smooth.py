"""Pins for oracle.smooth_objective / oracle.smooth (Eq.(5)-(7); R11-R14)."""
import numpy as np
import pytest
from scipy.optimize import minimize

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

import _brute

NORMS = [L1, L2, LINF]


@pytest.mark.parametrize("p", [0.25, 1.0, 10.0, 1e6])
def test_p13_two_point_closed_form(p):
    # N=2, symmetric, Delta = y1 - y2 - M d > 0: minimiser eps = (-t, +t), t = 2 p Delta / (4p + 1).
    X = np.array([[0.0, 0.0], [0.6, 0.8]], np.float32)           # d = 1 in L2
    y = np.array([3.0, 0.5], np.float32)
    M = 1.5
    Delta = 3.0 - 0.5 - 1.5 * np.sqrt(np.float64(np.float32(0.6)) ** 2 + np.float64(np.float32(0.8)) ** 2)
    t = 2 * p * Delta / (4 * p + 1)
    eps, info = oracle.smooth(X, y, M, None, L2, None, p)
    np.testing.assert_allclose(eps, [-t, t], atol=1e-9)
    F, grad = oracle.smooth_objective(X, y, M, [-t, t], None, L2, None, p)
    np.testing.assert_allclose(grad, 0.0, atol=1e-9)
    # F at the minimiser: 2 t^2 / p + 2 (Delta - 2t)^2  (both sums of Eq.(7) carry the violated pair once)
    np.testing.assert_allclose(F, 2 * t * t / p + 2 * (Delta - 2 * t) ** 2, rtol=1e-12)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("mask", [None, [1, 0, -1], [1, 1, 1]])
def test_p14_identity_and_finite_differences(norm, mask):
    X, y, _ = random_problem(5, 40, 1, 3, spread=0.5)
    w = np.array([1.0, 2.0, 0.5], np.float32)
    rng = np.random.default_rng(1)
    M, p = 0.8, 0.7
    for eps in (np.zeros(40), 0.3 * rng.standard_normal(40)):
        F, grad = oracle.smooth_objective(X, y, M, eps, mask, norm, w, p)
        Fb, gb = _brute.smooth_F_identity(X, y, np.float64(np.float32(M)), eps, mask, norm, w, p)
        np.testing.assert_allclose(F, Fb, rtol=1e-12)            # literal Eq.(7) == ||eps||^2/p + 2 sum V^2
        np.testing.assert_allclose(grad, gb, rtol=1e-11, atol=1e-11)
        h = 1e-6
        for i in (0, 7, 39):
            e1, e2 = eps.copy(), eps.copy()
            e1[i] += h
            e2[i] -= h
            fd = (oracle.smooth_objective(X, y, M, e1, mask, norm, w, p, False)[0]
                  - oracle.smooth_objective(X, y, M, e2, mask, norm, w, p, False)[0]) / (2 * h)
            np.testing.assert_allclose(grad[i], fd, rtol=2e-5, atol=1e-6)
        # the pair terms cancel in the sum of the gradient: sum_i dF/deps_i = 2 sum eps / p
        np.testing.assert_allclose(grad.sum(), 2 * eps.sum() / p, atol=1e-9)


def test_p14_consistent_data_need_no_smoothing():
    wl = make_workload(1, N=300)
    F, grad = oracle.smooth_objective(wl.X, wl.y, wl.M, np.zeros(300), wl.mask, wl.norm)
    assert F == 0.0 and np.all(grad == 0.0)
    eps, info = oracle.smooth(wl.X, wl.y, wl.M, wl.mask, wl.norm)
    assert np.all(eps == 0.0)


@pytest.mark.parametrize("norm,mask", [(L2, None), (L1, [1, 0]), (LINF, [1, -1]), (L2, [1, 1])])
def test_minimiser_against_independent_optimiser(norm, mask):
    """Strong convexity => unique minimiser: BFGS on the independent NumPy objective must land on
    the same point as oracle.smooth (R14), and sum eps = 0 there (P14)."""
    X, y, _ = random_problem(17, 25, 1, 2, spread=0.4)
    M, p = 0.5, 2.0
    eps, info = oracle.smooth(X, y, M, mask, norm, None, p)
    res = minimize(lambda e: _brute.smooth_F_identity(X, y, np.float64(np.float32(M)), e, mask, norm, None, p),
                   np.zeros(25), jac=True, method="BFGS", options=dict(gtol=1e-11, maxiter=5000))
    np.testing.assert_allclose(eps, res.x, atol=2e-7)
    assert abs(eps.sum()) < 1e-8
    assert info["gnorm_inf"] < 1e-6
    # smoothing reduces the worst violation of (5),(6)
    assert oracle.max_violation(X, y, M, eps, mask, norm) < oracle.max_violation(X, y, M, None, mask, norm)


def test_large_p_is_projection_onto_consistent_set():
    """p -> inf: eps* -> Euclidean projection of y on {z: z_i - z_k <= M D_ik}; check feasibility and the
    KKT sign structure on a 3-point example solved by hand:
    collinear points 0, 1, 2 with y = (0, 3, 0), M = 1, symmetric.  Constraints |z_i - z_k| <= |x_i - x_k|.
    Projection: by symmetry z = (a, b, a), b - a <= 1 active; minimise 2a^2 + (b-3)^2 s.t. b = a + 1
    -> a = 2/3, b = 5/3."""
    X = np.array([[0.0], [1.0], [2.0]], np.float32)
    y = np.array([0.0, 3.0, 0.0], np.float32)
    eps, info = oracle.smooth(X, y, 1.0, None, L2, None, 1e9)
    np.testing.assert_allclose(y + eps, [2 / 3, 5 / 3, 2 / 3], atol=1e-6)


def test_validation():
    X, y, _ = random_problem(1, 5, 1, 2)
    with pytest.raises(ValueError):
        oracle.smooth_objective(X, y, 1.0, np.zeros(5), None, L2, None, 0.0)
