"""Pins for oracle.knn (neighbours by distance; readings R5-R7).  CPU only."""
import numpy as np
import pytest
from hypothesis import given, settings, strategies as st
from scipy.spatial import cKDTree

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

import _brute

NORMS = [L1, L2, LINF]


@pytest.mark.parametrize("norm,p", [(L1, 1), (L2, 2), (LINF, np.inf)])
def test_p8_ckdtree(norm, p):
    X, _, Xq = random_problem(7, 3000, 200, 4)
    w = np.array([1.0, 0.5, 2.0, 1.5], np.float32)
    k = 9
    idx, dist = oracle.knn(X, Xq, k, None, 0, norm, w)
    dd, ii = cKDTree(X.astype(np.float64) * w).query(Xq.astype(np.float64) * w, k=k, p=p)
    np.testing.assert_allclose(dist, dd, rtol=1e-13, atol=1e-13)
    np.testing.assert_array_equal(idx, ii)          # continuous random data: no ties


@settings(max_examples=60, deadline=None)
@given(seed=st.integers(0, 10_000), d=st.integers(1, 5), norm=st.sampled_from(NORMS),
       N=st.integers(1, 20), Q=st.integers(1, 6), side=st.sampled_from([-1, 0, 1]), data=st.data())
def test_p7_brute_force_tiny_with_ties(seed, d, norm, N, Q, side, data):
    mask = data.draw(st.lists(st.sampled_from([-1, 0, 1]), min_size=d, max_size=d))
    k = data.draw(st.integers(1, N))
    rng = np.random.default_rng(seed)
    # integer grid coordinates => many exact ties, including zeros from positive parts
    X = rng.integers(-2, 3, (N, d)).astype(np.float32)
    Xq = rng.integers(-2, 3, (Q, d)).astype(np.float32)
    w = rng.choice([0.5, 1.0, 2.0], d).astype(np.float32)
    idx, dist = oracle.knn(X, Xq, k, mask, side, norm, w)
    ib, db = _brute.knn(X, Xq, k, mask, side, norm, w)
    np.testing.assert_array_equal(idx, ib)          # ties by lower index (R7)
    np.testing.assert_allclose(dist, db, rtol=0, atol=1e-13)


@pytest.mark.parametrize("norm", NORMS)
def test_p12_structure(norm):
    X, _, Xq = random_problem(9, 2000, 50, 3)
    Xq[:10] = X[100:110]                            # queries equal to data
    k = 16
    idx, dist = oracle.knn(X, Xq, k, None, 0, norm)
    assert np.all(np.diff(dist, axis=1) >= 0)
    assert idx.min() >= 0 and idx.max() < 2000
    assert all(len(set(r)) == k for r in idx)
    np.testing.assert_array_equal(idx[:10, 0], np.arange(100, 110))
    assert np.all(dist[:10, 0] == 0.0)
    Du, _ = _brute.distances(X, Xq, None, norm, None)
    for q in range(50):
        rest = np.delete(Du[q], idx[q])
        assert rest.min() >= dist[q, -1]
    i1, d1 = oracle.knn(X, Xq, 1, None, 0, norm)
    np.testing.assert_array_equal(i1[:, 0], Du.argmin(axis=1))


def test_one_sided_distance_selects_the_right_side():
    # d=1, increasing mask: D^u = (x - x^k)_+ is 0 for data to the right of the query.
    X = np.array([[0.0], [1.0], [2.0], [3.0]], np.float32)
    Xq = np.array([[1.5]], np.float32)
    idx, dist = oracle.knn(X, Xq, 4, [1], +1, L2)
    np.testing.assert_array_equal(idx[0], [2, 3, 1, 0])
    np.testing.assert_allclose(dist[0], [0, 0, 0.5, 1.5])
    idx, dist = oracle.knn(X, Xq, 4, [1], -1, L2)
    np.testing.assert_array_equal(idx[0], [0, 1, 2, 3])
    np.testing.assert_allclose(dist[0], [0, 0, 0.5, 1.5])
    idx, dist = oracle.knn(X, Xq, 4, [1], 0, L2)      # side 0 ignores the mask (R6)
    np.testing.assert_array_equal(idx[0], [1, 2, 0, 3])


def test_validation():
    X, _, Xq = random_problem(1, 10, 2, 2)
    with pytest.raises(ValueError):
        oracle.knn(X, Xq, 11)
    with pytest.raises(ValueError):
        oracle.knn(X, Xq, 0)


def test_config4_shape_small():
    wl = make_workload(4, N=5000, Q=40)
    idx, dist = oracle.knn(wl.X, wl.Xq, wl.k, None, 0, wl.norm)
    dd, ii = cKDTree(wl.X.astype(np.float64)).query(wl.Xq.astype(np.float64), k=wl.k, p=2)
    np.testing.assert_array_equal(idx, ii)
    np.testing.assert_allclose(dist, dd, rtol=1e-13)
