"""GPU parity for local Lipschitz interpolation: knots, step tables M_k, values_local.

Where fp32 vs fp64 rounding of a distance decides on which side of a knot it falls, several results
are correct: the checks compare what is unique exactly (within fp32 tolerance) and sandwich the rest
between two oracle evaluations with the knots moved by -eps / +eps (M_k[j] is non-decreasing in knot j,
M_k(D) non-increasing in the knots)."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem, sample_pairs

pytestmark = pytest.mark.gpu
NORMS = [L1, L2, LINF]
J = 16
EPS = 4e-6          # relative width of the knot band in which fp32 and fp64 may disagree on D <= t_j


def _dev(a, dtype=np.float32):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=dtype)).to("cuda:0")


def _problem(seed, N, Q, d):
    X, _, Xq = random_problem(seed, N, Q, d)
    y = (np.sin(2 * X[:, 0].astype(np.float64)) + 0.3 * X.astype(np.float64).sum(axis=1) ** 2).astype(np.float32)
    return X, y, Xq


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d", [2, 5, 11, 20])
def test_knots(norm, d):
    import paper_2606_04670_b200 as L
    X, y, _ = _problem(50 + d, 5000, 1, d)
    w = (2.0 ** (np.arange(d) % 3 - 1)).astype(np.float32)      # powers of two: exact weighting
    pi, pk = sample_pairs(9, 5000, 100003)
    ref = oracle.distance_quantiles(X, pi, pk, J, norm, w)
    got = L.lipfit_distance_quantiles(_dev(X), _dev(pi, np.int32), _dev(pk, np.int32), J, norm, w)
    np.testing.assert_allclose(got, ref, rtol=2e-6)              # same order statistic, fp32 distance
    assert np.all(np.diff(got) >= 0)
    with pytest.raises(L.LipfitError):                           # an index outside [0, N)
        L.lipfit_distance_quantiles(_dev(X), _dev(pi + 5000, np.int32), _dev(pk, np.int32), J, norm, w)


def _check_table(X, y, knots, norm, w, tol=2e-5, min_same=0.995):
    import torch
    import paper_2606_04670_b200 as L
    got = L.lipfit_local_lipschitz(_dev(X), _dev(y), knots, norm, w)
    torch.cuda.synchronize()
    got = got.cpu().numpy().astype(np.float64)
    k64 = knots.astype(np.float64)
    lo = oracle.local_lipschitz(X, y, k64 * (1 - EPS), norm, w)
    hi = oracle.local_lipschitz(X, y, k64 * (1 + EPS), norm, w)
    assert np.all(got >= lo * (1 - tol)) and np.all(got <= hi * (1 + tol))
    same = lo == hi
    assert same.mean() > min_same                                # the band matters for a handful of entries only
    ref = oracle.local_lipschitz(X, y, k64, norm, w)
    np.testing.assert_allclose(got[same], ref[same], rtol=tol)
    assert np.all(got[:, 1:] >= got[:, :-1])                     # non-decreasing step function (inf rows included)
    return got, ref


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,N", [(1, 700), (3, 3001), (8, 2500), (16, 1500), (25, 900)])
def test_step_tables(norm, d, N):
    import paper_2606_04670_b200 as L
    X, y, _ = _problem(60 + d, N, 1, d)
    w = (2.0 ** (np.arange(d) % 3 - 1)).astype(np.float32)
    pi, pk = sample_pairs(10, N, 20000)
    knots = L.lipfit_distance_quantiles(_dev(X), _dev(pi, np.int32), _dev(pk, np.int32), J, norm, w)
    knots[0] *= 0.05                                             # exercise the first-segment rule
    got, ref = _check_table(X, y, knots, norm, w)
    # max_k of the last column is the global Lipschitz constant (PAPER.md:179 with t = +inf)
    Lc = oracle.lipschitz_constant(X, y, None, norm, w)
    assert got[:, -1].max() == pytest.approx(Lc, rel=2e-5)


def test_step_tables_config_scaled_and_duplicates():
    wl = make_workload(5, N=20011)
    pi, pk = sample_pairs(11, wl.N, 50000)
    knots = oracle.distance_quantiles(wl.X, pi, pk, J, L2).astype(np.float32)
    _check_table(wl.X, wl.y, knots, L2, None)
    # duplicates: equal values are ignored, different values at zero distance give +inf
    X = np.array([[0, 0], [0, 0], [1, 0], [0, 0]] + [[2 + i, 1] for i in range(40)], np.float32)
    y = np.array([1, 1, 3, 2] + [0.1 * i for i in range(40)], np.float32)
    knots = np.linspace(0.5, 8.0, J).astype(np.float32)          # several distances sit exactly ON a knot
    got, ref = _check_table(X, y, knots, L2, None, min_same=0.9)
    assert np.all(np.isinf(got[0])) and np.all(np.isinf(got[3])) and np.all(np.isfinite(got[2]))


def _check_values(X, y, Xq, knots, table, norm, w):
    import torch
    import paper_2606_04670_b200 as L
    up, lo, g = L.lipfit_values_local(_dev(X), _dev(y), _dev(Xq), knots, _dev(table), norm, w)
    torch.cuda.synchronize()
    up, lo, g = (t.cpu().numpy().astype(np.float64) for t in (up, lo, g))
    k64 = knots.astype(np.float64)
    t64 = table.astype(np.float64)
    rng = max(float(y.max() - y.min()), 1e-30)
    mag = max(np.abs(up[np.isfinite(up)]).max(initial=0), np.abs(lo[np.isfinite(lo)]).max(initial=0))
    tol = 1e-5 * rng + (X.shape[1] + 6) * 2.0 ** -24 * mag       # as in tests/test_gpu_bounds.py
    Ua, La, _ = oracle.values_local(X, y, Xq, k64 * (1 - EPS), t64, norm, w)     # knots down: M_k(D) up
    Ub, Lb, _ = oracle.values_local(X, y, Xq, k64 * (1 + EPS), t64, norm, w)
    assert np.all(up <= np.maximum(Ua, Ub) + tol) and np.all(up >= np.minimum(Ua, Ub) - tol)
    assert np.all(lo <= np.maximum(La, Lb) + tol) and np.all(lo >= np.minimum(La, Lb) - tol)
    U, Lo, G = oracle.values_local(X, y, Xq, k64, t64, norm, w)
    same = (Ua == Ub) & (La == Lb)
    assert same.mean() > 0.99
    assert np.abs(up[same] - U[same]).max() <= tol and np.abs(lo[same] - Lo[same]).max() <= tol
    assert np.abs(g - 0.5 * (up + lo)).max() <= 1e-6 * max(1.0, mag)
    return up, lo, g


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,N,Q", [(1, 600, 999), (3, 3001, 2050), (8, 2500, 1300), (16, 1200, 700), (25, 700, 300)])
def test_values_local(norm, d, N, Q):
    X, y, Xq = _problem(70 + d, N, Q, d)
    w = (2.0 ** (np.arange(d) % 3 - 1)).astype(np.float32)
    pi, pk = sample_pairs(12, N, 20000)
    knots = oracle.distance_quantiles(X, pi, pk, J, norm, w).astype(np.float32)
    table = oracle.local_lipschitz(X, y, knots.astype(np.float64), norm, w).astype(np.float32)
    _check_values(X, y, Xq, knots, table, norm, w)


def test_local_pipeline_interpolates_the_data():
    """knots -> tables -> evaluation, all on the GPU: "The resulting approximation interpolates the data"
    (PAPER.md:183), and lies inside the global bounds."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(1, N=3000, Q=2000)
    pi, pk = sample_pairs(13, wl.N, 30000)
    Xd, yd = _dev(wl.X), _dev(wl.y)
    knots = L.lipfit_distance_quantiles(Xd, _dev(pi, np.int32), _dev(pk, np.int32), J, wl.norm)
    table = L.lipfit_local_lipschitz(Xd, yd, knots, wl.norm)
    up, lo, g = L.lipfit_values_local(Xd, yd, Xd, knots, table, wl.norm)
    torch.cuda.synchronize()
    tol = 1e-5 * wl.y_range
    assert np.abs(g.cpu().numpy() - wl.y).max() <= tol
    assert np.abs(up.cpu().numpy() - wl.y).max() <= tol and np.abs(lo.cpu().numpy() - wl.y).max() <= tol
    Lc = float(L.lipfit_lipschitz_constant(Xd, yd, None, wl.norm).cpu()[0])
    up, lo, g = L.lipfit_values_local(Xd, yd, _dev(wl.Xq), knots, table, wl.norm)
    Ug, Lg, _ = L.lipfit_bounds(Xd, yd, _dev(wl.Xq), Lc * (1 + 1e-5), None, wl.norm)
    assert bool((up <= Ug + tol).all()) and bool((lo >= Lg - tol).all())
    with pytest.raises(L.LipfitError):
        L.lipfit_local_lipschitz(Xd, yd, knots[:8], wl.norm)                     # J must be LIPFIT_LOCAL_KNOTS
    with pytest.raises(L.LipfitError):
        L.lipfit_local_lipschitz(Xd, yd, knots[::-1].copy(), wl.norm)            # knots must be non-decreasing


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("case", ["quantiles", "wide", "repeated", "zero_first", "one_ulp_apart"])
def test_knot_lookup_paths(norm, case):
    """The kernels look a distance up among the knots either through a cell table on the float bits (when no
    cell of the 1024-cell table holds two knots) or by a two-level search (local.cu: local_lut_params).  Knot
    sets that take the table (quantiles; 12 octaves wide, coarse cells) and sets that cannot (a repeated knot,
    a zero knot, two knots one ulp apart) against the oracle, tables and evaluation."""
    d, N, Q = 5, 2500, 1500
    X, y, Xq = _problem(90, N, Q, d)
    pi, pk = sample_pairs(14, N, 20000)
    knots = oracle.distance_quantiles(X, pi, pk, J, norm, None).astype(np.float32)
    if case == "wide":
        knots = (knots[7] * 2.0 ** np.linspace(-6, 6, J)).astype(np.float32)
    elif case == "repeated":
        knots[5] = knots[4]
    elif case == "zero_first":
        knots[0] = 0.0
    elif case == "one_ulp_apart":
        knots[9] = np.nextafter(knots[8], np.float32(np.inf))
    assert np.all(np.diff(knots) >= 0)
    got, _ = _check_table(X, y, knots, norm, None, min_same=0.99)
    table = oracle.local_lipschitz(X, y, knots.astype(np.float64), norm, None).astype(np.float32)
    _check_values(X, y, Xq, knots, table, norm, None)
