"""Pins for oracle.bounds_topk (reading R24)."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, random_problem

import _brute

NORMS = [L1, L2, LINF]


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("mask", [None, [1, 0, -1]])
def test_k1_is_eq2(norm, mask):
    X, y, Xq = random_problem(1, 90, 40, 3)
    U, L, G = oracle.bounds_topk(X, y, Xq, 1.5, [1.0], mask, norm)
    Ub, Lb, Gb = oracle.bounds(X, y, Xq, 1.5, mask, norm)
    np.testing.assert_array_equal(U, Ub)
    np.testing.assert_array_equal(L, Lb)
    np.testing.assert_array_equal(G, Gb)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("mask", [None, [1, 0, -1], [1, 1, 1]])
def test_brute_force_with_library_sort(norm, mask):
    X, y, Xq = random_problem(2, 60, 25, 3)
    w = np.array([1.0, 2.0, 0.5], np.float32)
    wk = np.array([0.8, 0.1, 0.1], np.float32)            # the paper's example
    M = np.float64(np.float32(0.9))
    Du, Dl = _brute.distances(X, Xq, mask, norm, w)        # independent NumPy distances (P7)
    hi = np.sort(y.astype(np.float64)[None, :] + M * Du, axis=1)[:, :3]
    lo = -np.sort(-(y.astype(np.float64)[None, :] - M * Dl), axis=1)[:, :3]
    U, L, G = oracle.bounds_topk(X, y, Xq, 0.9, wk, mask, norm, w)
    np.testing.assert_allclose(U, hi @ wk.astype(np.float64), rtol=1e-13)
    np.testing.assert_allclose(L, lo @ wk.astype(np.float64), rtol=1e-13)
    np.testing.assert_allclose(G, 0.5 * (U + L), rtol=0, atol=1e-15)


def test_unit_weights_pick_order_statistics_and_convex_weights_loosen_the_bounds():
    X, y, Xq = random_problem(3, 50, 30, 2)
    e = np.eye(4, dtype=np.float32)
    stats_u = np.stack([oracle.bounds_topk(X, y, Xq, 2.0, e[j])[0] for j in range(4)])
    stats_l = np.stack([oracle.bounds_topk(X, y, Xq, 2.0, e[j])[1] for j in range(4)])
    assert np.all(np.diff(stats_u, axis=0) >= 0) and np.all(np.diff(stats_l, axis=0) <= 0)
    U1, L1_, _ = oracle.bounds(X, y, Xq, 2.0)
    np.testing.assert_array_equal(stats_u[0], U1)
    wk = np.array([0.4, 0.3, 0.2, 0.1], np.float32)
    U, L, _ = oracle.bounds_topk(X, y, Xq, 2.0, wk)
    assert np.all(U >= U1 - 1e-12) and np.all(L <= L1_ + 1e-12)     # "The data set will not be interpolated"
    np.testing.assert_allclose(U, wk.astype(np.float64) @ stats_u, rtol=1e-13)
    with pytest.raises(ValueError):
        oracle.bounds_topk(X[:2], y[:2], Xq, 1.0, [0.5, 0.25, 0.25])    # k > N
