"""Pins for oracle.bounds_region (monotonicity on parts of the domain, cases I-IV;
reading R26 of DESIGN.md derives the formula the paper withholds).  CPU only.

What fixes it, other than itself: the hand-computed table tests/golden/p1_region_example.txt; the limits
a = b (simple monotonicity, Eq.(4)) and a = -inf, b = +inf (no constraint), where it must equal
oracle.bounds; an independent numerical integration of the "f may grow here" indicator along the way; the
closed form via the two non-decreasing transforms psi_up / psi_down retyped in NumPy; enclosure of admissible
functions (the paper's own f(x) = x^2 on [-1, 1], is case III); and attainment: for a single
datum H^upper itself is admissible, so no smaller upper bound is valid.
"""
import os

import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF

GOLDEN = os.path.join(os.path.dirname(__file__), "golden", "p1_region_example.txt")
NORMS = [L1, L2, LINF]
INC_A = {1: True, 2: False, 3: False, 4: True}     # f increasing on A  (cases I, IV)
INC_B = {1: True, 2: False, 3: True, 4: False}     # f increasing on B  (cases I, III)


def _rows():
    out = []
    with open(GOLDEN) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            p = [c.split() for c in line.split("|")]
            out.append(dict(mon=int(p[0][0]), w=float(p[1][0]), M=float(p[2][0]), xk=float(p[3][0]),
                            yk=float(p[3][1]), q=float(p[4][0]), U=float(p[5][0]), L=float(p[5][1])))
    return out


@pytest.mark.parametrize("r", _rows(), ids=lambda r: f"case{r['mon']}_{r['xk']}to{r['q']}")
def test_p1_worked_example(r):
    U, L, g = oracle.bounds_region(np.array([[r["xk"]]], np.float32), np.array([r["yk"]], np.float32),
                                   np.array([[r["q"]]], np.float32), r["M"], [r["mon"]], [1.0], [2.0], L2,
                                   [r["w"]])
    assert U[0] == pytest.approx(r["U"], abs=1e-14) and L[0] == pytest.approx(r["L"], abs=1e-14)
    assert g[0] == pytest.approx(0.5 * (r["U"] + r["L"]), abs=1e-14)


def _problem(seed, N, Q, d):
    rng = np.random.default_rng(seed)
    X = rng.uniform(-2, 2, (N, d)).astype(np.float32)
    Xq = rng.uniform(-2.5, 2.5, (Q, d)).astype(np.float32)
    y = rng.standard_normal(N).astype(np.float32)
    return X, y, Xq


@pytest.mark.parametrize("norm", NORMS)
def test_limit_a_equals_b_is_simple_monotonicity(norm):
    """a = b: AB is a point, so case I is 'increasing everywhere' (mask +1) and case II 'decreasing
    everywhere' (mask -1): Eq.(4) PAPER.md:142 -- wherever the common threshold sits."""
    X, y, Xq = _problem(1, 60, 50, 4)
    w = np.array([1.0, 0.5, 2.0, 1.5], np.float32)
    mon = [1, 2, 0, 1]
    c = np.array([0.3, -0.7, 9.0, 5.0], np.float32)        # the last threshold lies outside the data
    got = oracle.bounds_region(X, y, Xq, 1.3, mon, c, c, norm, w)
    ref = oracle.bounds(X, y, Xq, 1.3, [1, -1, 0, 1], norm, w)
    for u, v in zip(got, ref):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-12)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("case", [1, 2, 3, 4])
def test_limit_infinite_ab_is_unconstrained(norm, case):
    X, y, Xq = _problem(2, 50, 40, 3)
    inf = np.float32(np.inf)
    got = oracle.bounds_region(X, y, Xq, 0.8, [case] * 3, [-inf] * 3, [inf] * 3, norm)
    ref = oracle.bounds(X, y, Xq, 0.8, None, norm)
    for u, v in zip(got, ref):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-12)
    # mon = 0 ignores a, b altogether (they may be NULL)
    got0 = oracle.bounds_region(X, y, Xq, 0.8, [0] * 3, None, None, norm)
    for u, v in zip(got0, ref):
        np.testing.assert_array_equal(u, v)
    # the data lie inside AB = [-10, 10]: the constraint never bites
    got1 = oracle.bounds_region(X, y, Xq, 0.8, [case] * 3, [-10.0] * 3, [10.0] * 3, norm)
    for u, v in zip(got1, ref):
        np.testing.assert_allclose(u, v, rtol=0, atol=1e-12)


@pytest.mark.parametrize("case", [1, 2, 3, 4])
def test_half_infinite_regions(case):
    """a = -inf: A is empty, only B constrains; b = +inf: only A constrains.  1-D, one datum."""
    inf = np.float32(np.inf)
    xk, yk, M = 0.0, 0.5, 2.0
    q = np.linspace(-3, 3, 25).astype(np.float32)[:, None]
    # only B = [1, inf) constrains
    U, L, _ = oracle.bounds_region([[xk]], [yk], q, M, [case], [-inf], [1.0])
    t = q[:, 0].astype(np.float64)
    in_b = np.maximum(t, 1.0) - 1.0                       # length of the way [0, t] inside B (t > 1)
    below = np.minimum(t, 1.0)                            # signed length of the rest (t < 0: travelling down)
    if INC_B[case]:
        u = np.abs(below) + in_b
        l = np.abs(below)
    else:
        u = np.abs(below)
        l = np.abs(below) + in_b
    np.testing.assert_allclose(U, yk + M * u, atol=1e-12)
    np.testing.assert_allclose(L, yk - M * l, atol=1e-12)
    # only A = (-inf, -1] constrains
    U, L, _ = oracle.bounds_region([[xk]], [yk], q, M, [case], [-1.0], [inf])
    in_a = -1.0 - np.minimum(t, -1.0)                     # length of the way inside A (t < -1, travelling down)
    rest = np.abs(np.maximum(t, -1.0))
    if INC_A[case]:                                       # travelling down through an increasing region: f falls
        u, l = rest, rest + in_a
    else:
        u, l = rest + in_a, rest
    np.testing.assert_allclose(U, yk + M * u, atol=1e-12)
    np.testing.assert_allclose(L, yk - M * l, atol=1e-12)


def _indicator_integral(frm, to, case, a, b, want_grow, n=200001):
    """Length of the part of the way frm -> to on which f may grow (want_grow) / may fall in the direction of
    travel, by brute-force midpoint integration of the indicator: independent of the oracle's interval
    arithmetic."""
    if frm == to:
        return 0.0
    t = frm + (to - frm) * (np.arange(n) + 0.5) / n
    up = to > frm
    inc = np.where(t < a, INC_A[case], np.where(t > b, INC_B[case], np.nan))     # nan = unrestricted
    free = np.isnan(inc)
    grows = free | ((inc == 1.0) == up)           # travelling up an increasing / down a decreasing region
    falls = free | ((inc == 1.0) != up)
    return float(np.mean(grows if want_grow else falls)) * abs(to - frm)


@pytest.mark.parametrize("case", [1, 2, 3, 4])
def test_against_numerical_integration_of_the_indicator(case):
    rng = np.random.default_rng(10 + case)
    a, b, M = -0.4, 0.9, 1.75
    for _ in range(12):
        xk, x = rng.uniform(-2, 2, 2).astype(np.float32)
        U, L, _ = oracle.bounds_region([[xk]], [0.25], [[x]], M, [case], [a], [b])
        a32, b32 = float(np.float32(a)), float(np.float32(b))
        u = _indicator_integral(float(xk), float(x), case, a32, b32, True)
        l = _indicator_integral(float(xk), float(x), case, a32, b32, False)
        assert U[0] == pytest.approx(0.25 + M * u, abs=1e-4) and L[0] == pytest.approx(0.25 - M * l, abs=1e-4)


def _psi_components(X, Xq, mon, a, b, w):
    """Closed form through two non-decreasing transforms per coordinate (R26):
    u = max(psi_up(x) - psi_up(xk), psi_dn(xk) - psi_dn(x)), l = max(psi_up(xk) - psi_up(x), psi_dn(x) - psi_dn(xk))
    with psi = clamp(t, a, b) + [flag A] min(t - a, 0) + [flag B] max(t - b, 0)."""
    X, Xq = X.astype(np.float64), Xq.astype(np.float64)
    d = X.shape[1]
    u = np.zeros((Xq.shape[0], X.shape[0], d))
    l = np.zeros_like(u)
    for i in range(d):
        if mon[i] == 0:
            dl = np.abs(Xq[:, None, i] - X[None, :, i])
            u[:, :, i] = l[:, :, i] = w[i] * dl
            continue
        ai, bi = float(a[i]), float(b[i])

        def psi(t, fa, fb):
            return np.clip(t, ai, bi) + fa * np.minimum(t - ai, 0.0) + fb * np.maximum(t - bi, 0.0)
        ia, ib = INC_A[mon[i]], INC_B[mon[i]]
        pu_q, pu_x = psi(Xq[:, i], ia, ib), psi(X[:, i], ia, ib)
        pd_q, pd_x = psi(Xq[:, i], not ia, not ib), psi(X[:, i], not ia, not ib)
        u[:, :, i] = w[i] * np.maximum(pu_q[:, None] - pu_x[None, :], pd_x[None, :] - pd_q[:, None])
        l[:, :, i] = w[i] * np.maximum(pu_x[None, :] - pu_q[:, None], pd_q[:, None] - pd_x[None, :])
    return u, l


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("seed", range(4))
def test_against_the_transform_closed_form(norm, seed):
    rng = np.random.default_rng(100 + seed)
    d = 5
    X, y, Xq = _problem(20 + seed, 70, 60, d)
    mon = rng.integers(0, 5, d)
    a = rng.uniform(-1.5, 0.5, d).astype(np.float32)
    b = (a + rng.uniform(0, 1.5, d)).astype(np.float32)
    w = rng.uniform(0.2, 2.0, d).astype(np.float32)
    M = 1.125                                                  # exactly representable in fp32 (the oracle's input type)
    u, l = _psi_components(X, Xq, mon, a, b, w.astype(np.float64))
    if norm == L1:
        Du, Dl = u.sum(-1), l.sum(-1)
    elif norm == L2:
        Du, Dl = np.sqrt((u ** 2).sum(-1)), np.sqrt((l ** 2).sum(-1))
    else:
        Du, Dl = u.max(-1), l.max(-1)
    y64 = y.astype(np.float64)
    U, L, g = oracle.bounds_region(X, y, Xq, M, mon, a, b, norm, w)
    np.testing.assert_allclose(U, (y64[None, :] + M * Du).min(1), atol=1e-12)
    np.testing.assert_allclose(L, (y64[None, :] - M * Dl).max(1), atol=1e-12)
    np.testing.assert_allclose(g, 0.5 * (U + L), atol=1e-15)


def test_paper_example_x_squared_is_case_iii():
    """f(x) = x^2 on [-1, 1] is not monotone, but decreasing on x <= 0 and increasing on x >= 0:
    case III with a = b = 0.  Lip(f) = 2.  The bounds enclose f, interpolate the data, and are at least as
    tight as the unconstrained ones -- strictly tighter somewhere."""
    xs = np.linspace(-1, 1, 21).astype(np.float32)[:, None]
    f = lambda t: t.astype(np.float64)[:, 0] ** 2
    y = f(xs).astype(np.float32)
    q = np.random.default_rng(0).uniform(-1, 1, (400, 1)).astype(np.float32)
    U, L, g = oracle.bounds_region(xs, y, q, 2.0, [3], [0.0], [0.0])
    U0, L0, _ = oracle.bounds(xs, y, q, 2.0, None)
    fq = f(q)
    assert np.all(L <= fq + 1e-7) and np.all(fq <= U + 1e-7)
    assert np.all(U <= U0 + 1e-12) and np.all(L >= L0 - 1e-12)
    assert (U0 - U).max() > 0.05 and (L - L0).max() > 0.05
    Ud, Ld, gd = oracle.bounds_region(xs, y, xs, 2.0, [3], [0.0], [0.0])
    np.testing.assert_allclose(gd, y.astype(np.float64), atol=1e-7)
    # declaring the wrong case (IV: increasing on A, decreasing on B) is inconsistent with these data:
    Uw, Lw, _ = oracle.bounds_region(xs, y, q, 2.0, [4], [0.0], [0.0])
    assert np.any(Lw > Uw + 1e-6)


@pytest.mark.parametrize("case", [1, 2, 3, 4])
def test_enclosure_of_admissible_functions_in_3d(case):
    """f = sum_i h_i(x_i), h piecewise linear with slopes allowed by the case (any sign in AB): admissible with
    Lipschitz constant max|slope| in the L1-dual sense, so M = max|slope| works for L-infinity of the gradient,
    i.e. the L1 norm of the displacement; H^lower <= f <= H^upper must hold."""
    rng = np.random.default_rng(40 + case)
    d, a, b = 3, -0.5, 0.7
    sA = (1.0 if INC_A[case] else -1.0) * rng.uniform(0.2, 1.0, d)
    sB = (1.0 if INC_B[case] else -1.0) * rng.uniform(0.2, 1.0, d)
    sM = rng.uniform(-1.0, 1.0, d)

    def f(P):
        P = P.astype(np.float64)
        return (sA * np.minimum(P - a, 0) + sM * (np.clip(P, a, b) - a) + sB * np.maximum(P - b, 0)).sum(1)
    X = rng.uniform(-2, 2, (300, d)).astype(np.float32)
    Xq = rng.uniform(-2, 2, (500, d)).astype(np.float32)
    y = f(X).astype(np.float32)
    M = 1.0                                                    # >= every |slope|: Lipschitz in the L1 norm
    U, L, _ = oracle.bounds_region(X, y, Xq, M, [case] * d, [a] * d, [b] * d, L1)
    fq = f(Xq)
    assert np.all(L <= fq + 1e-6) and np.all(fq <= U + 1e-6)
    U0, L0, _ = oracle.bounds(X, y, Xq, M, None, L1)
    assert np.all(U <= U0 + 1e-12) and np.all(L >= L0 - 1e-12) and (U0 - U).max() > 0.1


@pytest.mark.parametrize("case", [1, 2, 3, 4])
def test_single_datum_bound_is_itself_admissible(case):
    """Attainment (why the bound cannot be lowered): with one datum, t -> H^upper(t) is M-Lipschitz, passes
    through the datum, and is monotone in the prescribed sense on A and on B; same for H^lower."""
    a, b, M, xk, yk = -0.3, 0.8, 1.5, 0.1, 2.0
    for xk in (-1.2, 0.1, 1.7):                                # datum in A, in AB, in B
        t = np.linspace(-3, 3, 2401).astype(np.float32)[:, None]
        U, L, _ = oracle.bounds_region([[xk]], [yk], t, M, [case], [a], [b])
        for H in (U, L):
            dH = np.diff(H)
            dt = np.diff(t[:, 0].astype(np.float64))
            assert np.all(np.abs(dH) <= M * dt + 1e-9)         # Lipschitz
            ta = t[:-1, 0] < a - 1e-3
            tb = t[:-1, 0] > b + 1e-3
            sa = 1.0 if INC_A[case] else -1.0
            sb = 1.0 if INC_B[case] else -1.0
            assert np.all(sa * dH[ta] >= -1e-12) and np.all(sb * dH[tb] >= -1e-12)
        k = int(np.argmin(np.abs(t[:, 0] - np.float32(xk))))
        assert U[k] == pytest.approx(yk, abs=M * 3e-3) and L[k] == pytest.approx(yk, abs=M * 3e-3)


def test_argument_checks():
    X, y, Xq = _problem(3, 5, 4, 2)
    with pytest.raises(ValueError):
        oracle.bounds_region(X, y, Xq, 1.0, [5, 0], [0, 0], [1, 1])
    with pytest.raises(ValueError):
        oracle.bounds_region(X, y, Xq, 1.0, [1, 0], [1.0, 0], [0.5, 1])       # a > b
    with pytest.raises(ValueError):
        oracle.bounds_region(X, y, Xq, 1.0, [1, 0], None, None)
    with pytest.raises(ValueError):
        oracle.bounds_region(X, y, Xq, -1.0, [0, 0], None, None)
