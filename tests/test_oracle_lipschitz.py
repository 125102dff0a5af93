"""Pins for oracle.lipschitz_constant and oracle.smooth_rows (Eq.(7), row form)."""
import numpy as np
import pytest
from scipy.spatial.distance import cdist

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

import _brute

NORMS = [L1, L2, LINF]
METRIC = {L1: "cityblock", L2: "euclidean", LINF: "chebyshev"}


@pytest.mark.parametrize("norm", NORMS)
def test_symmetric_case_is_max_ratio_over_scipy_cdist(norm):
    # no monotonicity: max |y_i - y_k| / ||w (x^i - x^k)||_p  (library distance, P8)
    X, y, _ = random_problem(3, 120, 1, 4)
    w = np.array([1.0, 0.5, 2.0, 1.5])
    D = cdist(X.astype(np.float64) * w, X.astype(np.float64) * w, METRIC[norm])
    dy = np.abs(y.astype(np.float64)[:, None] - y.astype(np.float64)[None, :])
    np.fill_diagonal(D, np.inf)
    np.testing.assert_allclose(oracle.lipschitz_constant(X, y, None, norm, w.astype(np.float32)),
                               (dy / D).max(), rtol=1e-12)


def test_one_dimension_is_the_steepest_adjacent_slope():
    # textbook: in 1-D the largest ratio over all pairs is attained by two adjacent points
    rng = np.random.default_rng(0)
    x = np.sort(rng.random(200)).astype(np.float32)
    y = rng.standard_normal(200).astype(np.float32)
    slopes = np.abs(np.diff(y.astype(np.float64)) / np.diff(x.astype(np.float64)))
    np.testing.assert_allclose(oracle.lipschitz_constant(x[:, None], y, None, L2), slopes.max(), rtol=1e-12)
    # increasing-monotone distance: only DEcreases of y along x are constrained by (x^i - x^k)_+ = 0 ...
    # d_s(x^k, x^i) = (x^i - x^k)_+ : pairs with x^i <= x^k and y_i > y_k are inconsistent for every M
    assert oracle.lipschitz_constant(x[:, None], y, [1], L2) == np.inf
    ys = np.sort(y)                                           # increasing data: steepest rise
    rise = np.diff(ys.astype(np.float64)) / np.diff(x.astype(np.float64))
    np.testing.assert_allclose(oracle.lipschitz_constant(x[:, None], ys, [1], L2), rise.max(), rtol=1e-12)


def test_linear_function_attains_the_dual_norm_on_aligned_pairs():
    # f(x) = a.x: |f(u) - f(v)| / ||u - v||_p <= ||a||_q with equality for u - v along the dual direction
    a = np.array([3.0, -4.0])
    X = np.array([[0, 0], [3, -4], [1, 1], [1, -1], [1, 0], [0, -1]], np.float32)
    y = (X.astype(np.float64) @ a).astype(np.float32)
    assert oracle.lipschitz_constant(X, y, None, L2) == pytest.approx(5.0, rel=1e-12)      # ||a||_2
    assert oracle.lipschitz_constant(X, y, None, L1) == pytest.approx(4.0, rel=1e-12)      # ||a||_inf
    assert oracle.lipschitz_constant(X, y, None, LINF) == pytest.approx(7.0, rel=1e-12)    # ||a||_1


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("mask", [None, [1, 0, -1], [1, 1, 1]])
def test_it_is_the_threshold_of_consistency(norm, mask):
    # L is the least M with zero violation of constraint (5): brute force (P7) + definition
    X, _, _ = random_problem(11, 60, 1, 3)
    s = np.zeros(3) if mask is None else np.asarray(mask, np.float64)
    y = (X.astype(np.float64) @ np.where(s == 0, 0.3, s)).astype(np.float32)   # monotone where masked
    L = oracle.lipschitz_constant(X, y, mask, norm)
    Du, _ = _brute.distances(X, X, mask, norm, None)
    dy = y.astype(np.float64)[:, None] - y.astype(np.float64)[None, :]
    with np.errstate(divide="ignore", invalid="ignore"):
        ratio = np.where((dy > 0) & (Du > 0), dy / Du, 0.0)
    assert np.isfinite(L) and L == pytest.approx(ratio.max(), rel=1e-12)
    assert oracle.max_violation(X, y, L * (1 + 1e-6), None, mask, norm) == 0.0
    assert oracle.max_violation(X, y, L * (1 - 1e-3), None, mask, norm) > 0.0


def test_degenerate_cases():
    X = np.zeros((1, 2), np.float32)
    assert oracle.lipschitz_constant(X, np.ones(1, np.float32)) == 0.0
    X = np.array([[0, 0], [0, 0], [1, 0]], np.float32)
    assert oracle.lipschitz_constant(X, np.array([1, 1, 1], np.float32)) == 0.0          # constant data
    assert oracle.lipschitz_constant(X, np.array([1, 2, 1], np.float32)) == np.inf       # duplicate x, different y
    wl = make_workload(1, N=300)
    assert oracle.lipschitz_constant(wl.X, wl.y, None, L2) <= np.sqrt(13.0)              # Lip(f) of config 1


@pytest.mark.parametrize("norm,mask", [(L2, [1, 1, 1, 1, 1]), (L1, [1, 0, -1, 0, 0]), (LINF, None)])
def test_smooth_rows_is_the_row_form_of_eq7(norm, mask):
    wl = make_workload(5, N=90)
    rng = np.random.default_rng(4)
    eps = 0.05 * rng.standard_normal(90)
    rows = np.array([0, 7, 33, 89, 7])
    g, f = oracle.smooth_rows(wl.X, wl.y, 1.7, eps, rows, mask, norm, None, 0.6)
    Fb, gb = _brute.smooth_F_identity(wl.X, wl.y, np.float64(np.float32(1.7)), eps, mask, norm, None, 0.6)
    np.testing.assert_allclose(g, gb[rows], rtol=1e-10, atol=1e-12)                      # independent NumPy
    _, f_all = oracle.smooth_rows(wl.X, wl.y, 1.7, eps, np.arange(90), mask, norm, None, 0.6)
    np.testing.assert_allclose(f_all.sum(), Fb, rtol=1e-12)                              # shares add up to F
