"""Pins for oracle.bounds (Eq.(2),(3),(4)).  CPU only.

Each test names the pin of SURVEY.md §8(c) it implements; together they are
chosen so that a dropped term, a swapped side (D^u <-> D^l), a wrong sign of
the mask, a missing weight or a wrong norm fails at least one of them.
"""
import os

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st
from scipy.spatial.distance import cdist

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

import _brute

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "p0_worked_example.txt")
NORMS = [L1, L2, LINF]


def _golden_rows():
    rows = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            parts = [p.split() for p in line.split("|")]
            rows.append(dict(mask=[int(v) for v in parts[0]], w=[float(v) for v in parts[1]],
                             norm=int(parts[2][0]), M=float(parts[3][0]),
                             q=[float(v) for v in parts[4]], out=[float(v) for v in parts[5]]))
    return rows


@pytest.mark.parametrize("row", _golden_rows(), ids=lambda r: f"m{r['mask']}n{r['norm']}")
def test_p0_worked_example(row):
    X = np.array([[0, 0], [1, 0], [0, 1]], np.float32)
    y = np.array([0, 1, 2], np.float32)
    U, L, g = oracle.bounds(X, y, np.array([row["q"]], np.float32), row["M"], row["mask"],
                            row["norm"], row["w"])
    np.testing.assert_allclose([U[0], L[0], g[0]], row["out"], rtol=0, atol=1e-15 * 8)


def _consistent(norm, mask, N=400, Q=300, seed=3):
    """Noise-free data from a smooth generator that is monotone where masked,
    with M above its Lipschitz constant in the chosen norm."""
    rng = np.random.default_rng(seed)
    d = len(mask)
    X = rng.random((N, d)).astype(np.float32)
    Xq = rng.random((Q, d)).astype(np.float32)
    s = np.asarray(mask, np.float64)
    coef = np.where(s == 0, np.linspace(-1.0, 1.0, d), s * np.linspace(0.5, 1.5, d))

    def f(x):
        x = np.asarray(x, np.float64)
        return (coef * x).sum(axis=1) + 0.1 * np.sin(3.0 * x[:, 0] * (s[0] == 0))

    grad_bound = np.abs(coef) + np.array([0.3 if s[0] == 0 else 0.0] + [0.0] * (d - 1))
    # Lipschitz constant w.r.t. ||.||_p is the dual norm of the gradient bound.
    lip = {L1: grad_bound.max(), L2: np.sqrt((grad_bound ** 2).sum()), LINF: grad_bound.sum()}[norm]
    y64 = f(X)
    # y must be EXACTLY representable so that the data stay consistent after rounding:
    # round y to fp32 and widen M by a margin that dominates the rounding (2^-24 * |y| / min dist).
    return X, y64.astype(np.float32), Xq, f, 1.25 * lip + 0.05


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("mask", [[0, 0, 0], [1, 0, -1], [1, 1, 1], [-1, -1, 0]])
def test_p1_p2_p3_consistent_data(norm, mask):
    X, y, Xq, f, M = _consistent(norm, mask)
    # P1 interpolation: g(x^k) = y^k exactly.
    U, L, g = oracle.bounds(X, y, X, M, mask, norm)
    assert oracle.max_violation(X, y, M, None, mask, norm) == 0.0
    np.testing.assert_array_equal(U, y.astype(np.float64))
    np.testing.assert_array_equal(L, y.astype(np.float64))
    np.testing.assert_array_equal(g, y.astype(np.float64))
    # P2 sandwich and P3 enclosure of the generator + error bound.
    U, L, g = oracle.bounds(X, y, Xq, M, mask, norm)
    assert np.all(L <= g) and np.all(g <= U)
    fq = f(Xq)
    tol = 1e-6  # y was rounded to fp32
    assert np.all(L <= fq + tol) and np.all(fq <= U + tol)
    Du, Dl = _brute.distances(X, Xq, None, norm, None)      # symmetric distance
    assert np.all(np.abs(fq - g) <= 0.5 * (U - L) + tol)
    assert np.all(0.5 * (U - L) <= M * Du.min(axis=1) + tol)


def test_p2_converse_inconsistent_point_breaks_sandwich():
    X, y, Xq, f, M = _consistent(L2, [0, 0, 0])
    y = y.copy()
    y[7] += 5.0            # R8: still returns min / max / midpoint, no error
    U, L, g = oracle.bounds(X, y, X[6:9], M, None, L2)
    assert np.any(L > U)
    np.testing.assert_allclose(g, 0.5 * (U + L))


@pytest.mark.parametrize("norm", NORMS)
def test_p4_lipschitz_any_data(norm):
    X, y, Xq = random_problem(11, 200, 150, 3)
    w = np.array([0.5, 2.0, 1.0], np.float32)
    M = 1.7
    for mask in ([0, 0, 0], [1, -1, 0]):
        U, L, g = oracle.bounds(X, y, Xq, M, mask, norm, w)
        diff = (Xq[:, None, :].astype(np.float64) - Xq[None, :, :].astype(np.float64)) * w
        D = _brute.pnorm(np.abs(diff), norm)
        for H in (U, L, g):
            assert np.all(np.abs(H[:, None] - H[None, :]) <= np.float64(np.float32(M)) * D + 1e-12)


@pytest.mark.parametrize("norm", NORMS)
def test_p5_monotone_any_data(norm):
    X, y, _ = random_problem(12, 300, 1, 3)
    rng = np.random.default_rng(5)
    base = rng.standard_normal((100, 3)).astype(np.float32)
    step = np.abs(rng.standard_normal((100, 3))).astype(np.float32)
    mask = [1, -1, 0]
    # move along +x1 (increasing) and -x2 (x2 is decreasing-constrained): all three must not decrease
    hi = base.copy()
    hi[:, 0] += step[:, 0]
    hi[:, 1] -= step[:, 1]
    a = oracle.bounds(X, y, base, 2.0, mask, norm)
    b = oracle.bounds(X, y, hi, 2.0, mask, norm)
    for Ha, Hb in zip(a, b):
        assert np.all(Hb >= Ha)
    # and moving along the free coordinate can go either way (sanity that the mask matters)
    fr = base.copy()
    fr[:, 2] += step[:, 2]
    c = oracle.bounds(X, y, fr, 2.0, mask, norm)
    assert np.any(c[2] < a[2]) and np.any(c[2] > a[2])


@pytest.mark.parametrize("norm", NORMS)
def test_p6_one_dimensional_closed_forms(norm):
    rng = np.random.default_rng(21)
    xs = np.sort(rng.random(40)).astype(np.float32)
    ys = np.cumsum(rng.random(40) * 0.02).astype(np.float32)          # increasing, slope < M
    M = 50.0
    X = xs[:, None]
    assert oracle.max_violation(X, ys, M, None, [1], norm) == 0.0
    xq = (xs[0] + (xs[-1] - xs[0]) * rng.random(500)).astype(np.float32)
    j = np.clip(np.searchsorted(xs, xq, side="right") - 1, 0, len(xs) - 2)
    x0, x1 = xs[j].astype(np.float64), xs[j + 1].astype(np.float64)
    y0, y1 = ys[j].astype(np.float64), ys[j + 1].astype(np.float64)
    x = xq.astype(np.float64)
    U, L, g = oracle.bounds(X, ys, xq[:, None], M, [0], norm)
    np.testing.assert_allclose(U, np.minimum(y0 + M * (x - x0), y1 + M * (x1 - x)), atol=1e-13)
    np.testing.assert_allclose(L, np.maximum(y0 - M * (x - x0), y1 - M * (x1 - x)), atol=1e-13)
    U, L, g = oracle.bounds(X, ys, xq[:, None], M, [1], norm)
    np.testing.assert_allclose(U, np.minimum(y1, y0 + M * (x - x0)), atol=1e-13)
    np.testing.assert_allclose(L, np.maximum(y0, y1 - M * (x1 - x)), atol=1e-13)
    # decreasing data under mask -1 mirror the increasing case
    U2, L2_, _ = oracle.bounds(-X, ys, -xq[:, None], M, [-1], norm)
    np.testing.assert_allclose(U2, U, atol=1e-13)
    np.testing.assert_allclose(L2_, L, atol=1e-13)
    # N = 1
    U, L, g = oracle.bounds(X[:1], ys[:1], xq[:, None], M, [1], norm)
    np.testing.assert_allclose(U, ys[0] + M * np.maximum(x - xs[0], 0), atol=1e-13)
    np.testing.assert_allclose(L, ys[0] - M * np.maximum(xs[0] - x, 0), atol=1e-13)


@settings(max_examples=60, deadline=None)
@given(seed=st.integers(0, 10_000), d=st.integers(1, 6), norm=st.sampled_from(NORMS),
       N=st.integers(1, 12), Q=st.integers(0, 7), data=st.data())
def test_p7_brute_force_tiny(seed, d, norm, N, Q, data):
    mask = data.draw(st.lists(st.sampled_from([-1, 0, 1]), min_size=d, max_size=d))
    w = np.array(data.draw(st.lists(st.sampled_from([0.0, 0.25, 1.0, 1.5, 3.0]), min_size=d,
                                    max_size=d)), np.float32)
    M = data.draw(st.sampled_from([0.0, 0.5, 1.0, 7.0]))
    X, y, Xq = random_problem(seed, N, Q, d)
    U, L, g = oracle.bounds(X, y, Xq, M, mask, norm, w)
    if Q == 0:
        assert U.size == 0
        return
    Ub, Lb, gb = _brute.bounds(X, y, Xq, M, mask, norm, w)
    np.testing.assert_allclose(U, Ub, rtol=0, atol=1e-12)
    np.testing.assert_allclose(L, Lb, rtol=0, atol=1e-12)
    np.testing.assert_allclose(g, gb, rtol=0, atol=1e-12)


@pytest.mark.parametrize("norm,metric", [(L1, "cityblock"), (L2, "euclidean"), (LINF, "chebyshev")])
def test_p8_scipy_cdist_special_case(norm, metric):
    X, y, Xq = random_problem(31, 500, 200, 5)
    w = np.array([1.0, 0.5, 2.0, 1.0, 3.0], np.float32)
    M = 1.3
    # scipy's weighted metrics use sum w|d| (L1), sqrt(sum w d^2) (L2), max over w>0 of |d|?  -> avoid the
    # ambiguity: scale the coordinates by w instead and use the unweighted metric.
    D = cdist(Xq.astype(np.float64) * w, X.astype(np.float64) * w, metric=metric)
    Mf = np.float64(np.float32(M))
    U, L, g = oracle.bounds(X, y, Xq, M, None, norm, w)
    np.testing.assert_allclose(U, (y[None, :] + Mf * D).min(axis=1), atol=1e-12)
    np.testing.assert_allclose(L, (y[None, :] - Mf * D).max(axis=1), atol=1e-12)


@pytest.mark.parametrize("norm", NORMS)
def test_p9_metamorphic(norm):
    X, y, Xq = random_problem(41, 300, 100, 4)
    mask = np.array([1, -1, 0, 1])
    w = np.array([1.0, 2.0, 0.5, 1.0], np.float32)
    M = 2.0
    U, L, g = oracle.bounds(X, y, Xq, M, mask, norm, w)
    # (y, mask) -> (-y, -mask): H^u' = -H^l, H^l' = -H^u
    U2, L2_, _ = oracle.bounds(X, -y, Xq, M, -mask, norm, w)
    np.testing.assert_allclose(U2, -L, atol=1e-13)
    np.testing.assert_allclose(L2_, -U, atol=1e-13)
    # negating coordinate i together with s_i changes nothing (R2)
    Xn, Xqn, mn = X.copy(), Xq.copy(), mask.copy()
    Xn[:, 1] *= -1
    Xqn[:, 1] *= -1
    mn[1] *= -1
    np.testing.assert_allclose(oracle.bounds(Xn, y, Xqn, M, mn, norm, w)[2], g, atol=1e-13)
    # permuting the data changes nothing
    perm = np.random.default_rng(0).permutation(len(y))
    np.testing.assert_array_equal(oracle.bounds(X[perm], y[perm], Xq, M, mask, norm, w)[0], U)
    # y + c shifts, (2y, 2M) scales (powers of two keep fp32 inputs exact)
    np.testing.assert_allclose(oracle.bounds(X, y + np.float32(0), Xq, M, mask, norm, w)[2], g)
    U3, L3, g3 = oracle.bounds(X, 2 * y, Xq, 2 * M, mask, norm, w)
    np.testing.assert_allclose(g3, 2 * g, atol=1e-13)
    # (2X, 2Xq, M/2) and (w -> 4w, M -> M/4) leave the outputs unchanged
    np.testing.assert_allclose(oracle.bounds(2 * X, y, 2 * Xq, M / 2, mask, norm, w)[2], g, atol=1e-13)
    np.testing.assert_allclose(oracle.bounds(X, y, Xq, M / 4, mask, norm, 4 * w)[2], g, atol=1e-13)
    # permuting coordinates together with mask and weights changes nothing
    cp = [2, 0, 3, 1]
    np.testing.assert_allclose(
        oracle.bounds(X[:, cp], y, Xq[:, cp], M, mask[cp], norm, w[cp])[2], g, atol=1e-13)


def test_p10_cross_norm_order_and_p11_range():
    X, y, Xq = random_problem(51, 300, 200, 4)
    mask = [1, 0, -1, 0]
    r = {n: oracle.bounds(X, y, Xq, 1.5, mask, n) for n in NORMS}
    assert np.all(r[L1][0] >= r[L2][0]) and np.all(r[L2][0] >= r[LINF][0])
    assert np.all(r[L1][1] <= r[L2][1]) and np.all(r[L2][1] <= r[LINF][1])
    for n in NORMS:     # P11: symmetric distance keeps g inside the data range
        U, L, g = oracle.bounds(X, y, Xq, 1.5, None, n)
        assert np.all(g >= y.min()) and np.all(g <= y.max())


def test_m_zero_and_validation():
    X, y, Xq = random_problem(61, 50, 20, 2)
    U, L, g = oracle.bounds(X, y, Xq, 0.0, None, L2)
    assert np.all(U == y.min()) and np.all(L == y.max())
    with pytest.raises(ValueError):
        oracle.bounds(X, y, Xq, -1.0, None, L2)
    with pytest.raises(ValueError):
        oracle.bounds(X, y, Xq, 1.0, [2, 0], L2)
    with pytest.raises(ValueError):
        oracle.bounds(X, y, Xq, 1.0, None, 7)


def test_config1_is_consistent_and_interpolates():
    """BASELINE.json config 1: |grad f|_2 <= sqrt(13) < M = 4 => consistent."""
    wl = make_workload(1)
    assert oracle.max_violation(wl.X, wl.y, wl.M, None, wl.mask, wl.norm) == 0.0
    U, L, g = oracle.bounds(wl.X, wl.y, wl.X, wl.M, wl.mask, wl.norm)
    np.testing.assert_array_equal(g, wl.y.astype(np.float64))
    U, L, g = oracle.bounds(wl.X, wl.y, wl.Xq[:2000], wl.M, wl.mask, wl.norm)
    fq = wl.f(wl.Xq[:2000].astype(np.float64))
    assert np.all(L <= fq + 1e-6) and np.all(fq <= U + 1e-6)
