"""Pins for the local Lipschitz oracle (readings R20-R23): knots, step tables M_k, values_local."""
import numpy as np
import pytest
from scipy.spatial.distance import cdist

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem, sample_pairs

NORMS = [L1, L2, LINF]
METRIC = {L1: "cityblock", L2: "euclidean", LINF: "chebyshev"}


def _problem(seed, N, Q, d):
    X, _, Xq = random_problem(seed, N, Q, d)
    y = (np.sin(2 * X[:, 0].astype(np.float64)) + 0.3 * X.astype(np.float64).sum(axis=1) ** 2).astype(np.float32)
    return X, y, Xq


def _brute_table(X, y, knots, norm, w):
    """Independent NumPy statement of PAPER.md:179 (whole-matrix form)."""
    Xw = X.astype(np.float64) * (np.ones(X.shape[1]) if w is None else np.asarray(w, np.float64))
    D = cdist(Xw, Xw, METRIC[norm])
    dy = np.abs(y.astype(np.float64)[:, None] - y.astype(np.float64)[None, :])
    np.fill_diagonal(D, np.nan)
    with np.errstate(divide="ignore", invalid="ignore"):
        R = dy / D
    N, J = len(y), len(knots)
    T = np.zeros((N, J))
    for k in range(N):
        dk, rk = D[k], R[k]
        ok = ~np.isnan(dk)
        dmin = dk[ok].min()
        rnn = rk[ok & (dk == dmin)].max()
        for j in range(J):
            sel = ok if j == J - 1 else ok & (dk <= knots[j])
            T[k, j] = max(rnn, rk[sel].max() if sel.any() else 0.0)
    return T


@pytest.mark.parametrize("norm", NORMS)
def test_knots_are_nearest_rank_quantiles_of_the_sampled_distances(norm):
    X, y, _ = _problem(1, 300, 1, 3)
    w = np.array([1.0, 0.5, 2.0], np.float32)
    pi, pk = sample_pairs(5, 300, 4000)
    assert np.all(pi != pk)
    Xw = X.astype(np.float64) * w
    ds = np.array([cdist(Xw[i:i + 1], Xw[k:k + 1], METRIC[norm])[0, 0] for i, k in zip(pi, pk)])
    J = 16
    ref = np.quantile(ds, np.arange(1, J + 1) / J, method="inverted_cdf")       # library routine (P8)
    np.testing.assert_allclose(oracle.distance_quantiles(X, pi, pk, J, norm, w), ref, rtol=1e-13)


@pytest.mark.parametrize("norm", NORMS)
def test_table_matches_brute_force_and_its_invariants(norm):
    X, y, _ = _problem(2, 120, 1, 3)
    w = np.array([1.0, 2.0, 0.5], np.float32)
    pi, pk = sample_pairs(6, 120, 2000)
    knots = oracle.distance_quantiles(X, pi, pk, 8, norm, w)
    knots[0] *= 1e-3                       # a first knot below every nearest-neighbour distance
    T = oracle.local_lipschitz(X, y, knots, norm, w)
    np.testing.assert_allclose(T, _brute_table(X, y, knots, norm, w), rtol=1e-12)
    assert np.all(np.diff(T, axis=1) >= 0)                     # M_k is a non-decreasing step function
    # the first segment has the value |y_k - y_(1)| / d_(1)
    Xw = X.astype(np.float64) * w
    D = cdist(Xw, Xw, METRIC[norm])
    np.fill_diagonal(D, np.inf)
    nn = D.argmin(axis=1)
    first = np.abs(y.astype(np.float64) - y[nn].astype(np.float64)) / D[np.arange(120), nn]
    np.testing.assert_allclose(T[:, 0], first, rtol=1e-12)
    # the last column is the maximum over all data; its maximum over k is the global Lipschitz constant
    assert T[:, -1].max() == pytest.approx(oracle.lipschitz_constant(X, y, None, norm, w), rel=1e-12)


@pytest.mark.parametrize("norm", NORMS)
def test_values_local_interpolates_and_tightens_the_global_bounds(norm):
    X, y, Xq = _problem(3, 150, 200, 2)
    pi, pk = sample_pairs(7, 150, 3000)
    knots = oracle.distance_quantiles(X, pi, pk, 6, norm)
    T = oracle.local_lipschitz(X, y, knots, norm)
    # "The resulting approximation interpolates the data"
    U, L, G = oracle.values_local(X, y, X, knots, T, norm)
    scale = np.abs(y).max()
    np.testing.assert_allclose(U, y, atol=1e-12 * scale)
    np.testing.assert_allclose(L, y, atol=1e-12 * scale)
    # M_k(D) <= global constant => local bounds lie inside the global ones
    Lc = oracle.lipschitz_constant(X, y, None, norm)
    U, L, G = oracle.values_local(X, y, Xq, knots, T, norm)
    Ug, Lg, _ = oracle.bounds(X, y, Xq, Lc * (1 + 1e-6), None, norm)   # tiny slack: M is rounded to fp32 there
    assert np.all(U <= Ug + 1e-9) and np.all(L >= Lg - 1e-9)
    np.testing.assert_allclose(G, 0.5 * (U + L), rtol=0, atol=1e-15)


@pytest.mark.parametrize("norm", NORMS)
def test_constant_table_reduces_to_eq2(norm):
    X, y, Xq = _problem(4, 80, 60, 3)
    w = np.array([0.5, 1.0, 2.0], np.float32)
    knots = np.array([0.1, 0.5, 1.0, 2.0])
    T = np.full((80, 4), 1.75)
    U, L, G = oracle.values_local(X, y, Xq, knots, T, norm, w)
    Ub, Lb, Gb = oracle.bounds(X, y, Xq, 1.75, None, norm, w)
    np.testing.assert_allclose(U, Ub, rtol=1e-14)
    np.testing.assert_allclose(L, Lb, rtol=1e-14)


def test_step_function_lookup_by_brute_force():
    # one datum, hand-made table: M(D) = table[first j with D <= t_j], last knot = +inf
    X = np.zeros((1, 1), np.float32)
    y = np.array([2.0], np.float32)
    knots = np.array([1.0, 2.0, 3.0])
    T = np.array([[10.0, 20.0, 30.0]])
    Xq = np.array([[0.0], [0.5], [1.0], [1.5], [2.0], [2.5], [3.0], [7.0]], np.float32)
    U, L, G = oracle.values_local(X, y, Xq, knots, T, L2)
    Ms = np.array([10, 10, 10, 20, 20, 30, 30, 30.0])
    D = np.abs(Xq[:, 0].astype(np.float64))
    np.testing.assert_allclose(U, 2.0 + Ms * D)
    np.testing.assert_allclose(L, 2.0 - Ms * D)


def test_duplicates_and_degenerate_inputs():
    X = np.array([[0, 0], [0, 0], [1, 0], [0, 0]], np.float32)
    y = np.array([1, 1, 3, 2], np.float32)          # 0,1 duplicates; 3 = same point, different value
    T = oracle.local_lipschitz(X, y, np.array([0.5, 2.0]), L2)
    assert np.all(np.isinf(T[0])) and np.all(np.isinf(T[3]))      # a different value at zero distance
    assert np.all(np.isinf(T[2]) == False) and T[2, 1] == pytest.approx(2.0)
    U, L, G = oracle.values_local(X, y, X[2:3], np.array([0.5, 2.0]), T, L2)
    assert U[0] == 3.0 and L[0] == 3.0                              # inf * 0 := 0 at the datum itself


def test_rows_variant_equals_the_full_table():
    """oracle.local_lipschitz_rows (full-size parity samples) is the same loop over a list of data: its rows
    equal the rows of the whole table bit for bit, which the brute-force pin above fixes."""
    X, y, _ = _problem(91, 700, 1, 4)
    w = np.array([1.0, 0.5, 2.0, 1.0], np.float32)
    pi, pk = sample_pairs(5, 700, 5000)
    for norm in NORMS:
        knots = oracle.distance_quantiles(X, pi, pk, 16, norm, w)
        full = oracle.local_lipschitz(X, y, knots, norm, w)
        rows = np.array([0, 699, 13, 13, 350], np.int64)
        np.testing.assert_array_equal(oracle.local_lipschitz_rows(X, y, knots, rows, norm, w), full[rows])
    with pytest.raises(ValueError):
        oracle.local_lipschitz_rows(X, y, knots, [700], L2, w)
