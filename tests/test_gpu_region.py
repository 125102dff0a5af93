"""GPU parity: lipfit_bounds_region (monotonicity on parts of the domain, cases I-IV;
reading R26) vs the fp64 oracle, element by element.  The oracle measures the way from the datum to the query
interval by interval; the kernel subtracts two non-decreasing transforms per coordinate -- two formulations
of the same derivation."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

pytestmark = pytest.mark.gpu
NORMS = [L1, L2, LINF]
INF = np.float32(np.inf)


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _check(X, y, Xq, M, mon, a, b, norm, w=None, stated=False):
    import torch
    import paper_2606_04670_b200 as L
    up, lo, g = L.lipfit_bounds_region(_dev(X), _dev(y), _dev(Xq), M, mon, a, b, norm, w)
    torch.cuda.synchronize()
    up, lo, g = up.cpu().numpy(), lo.cpu().numpy(), g.cpu().numpy()
    U, Lo, G = oracle.bounds_region(X, y, Xq, M, mon, a, b, norm, w)
    rng = max(float(y.max() - y.min()), 1e-30) if len(y) > 1 else 1.0
    tol = 1e-5 * rng                                            # north_star's bar
    if not stated:                                              # unstructured inputs: + rounding of the candidate
        mag = max(np.abs(U).max(), np.abs(Lo).max())            # (2 transformed values per coordinate)
        tol += (2 * X.shape[1] + 4) * 2.0 ** -24 * mag
    assert np.abs(up - U).max(initial=0) <= tol, (np.abs(up - U).max(), tol)
    assert np.abs(lo - Lo).max(initial=0) <= tol, (np.abs(lo - Lo).max(), tol)
    assert np.abs(g - G).max(initial=0) <= tol
    return up, lo, g


def _thresholds(seed, d):
    rng = np.random.default_rng(seed)
    mon = rng.integers(0, 5, d).astype(np.int32)
    a = rng.uniform(-1.0, 0.2, d).astype(np.float32)
    b = (a + rng.uniform(0.0, 1.2, d)).astype(np.float32)
    return mon, a, b


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d", [1, 2, 3, 4, 5, 8, 11, 16, 23, 32])
def test_shapes(norm, d):
    X, y, Xq = random_problem(500 + d, 1500 + d, 777 + d, d)    # ragged tiles, ragged last block
    mon, a, b = _thresholds(d, d)
    w = (0.25 + np.arange(d) % 3).astype(np.float32)
    _check(X, y, Xq, 1.25, mon, a, b, norm, w)
    _check(X, y, Xq, 0.5, mon, a, b, norm, None)


@pytest.mark.parametrize("case", [1, 2, 3, 4])
@pytest.mark.parametrize("cfg,N,Q", [(2, 3000, 5003), (3, 2500, 4099), (5, 3001, 4097), (2, 40000, 700),
                                     (1, 1000, 10000)])
def test_configs_scaled_every_case(case, cfg, N, Q):
    """Config-shaped data (stated bar only), thresholds inside the data range, the same case on every coordinate
    that the config constrains and on the first coordinate otherwise."""
    wl = make_workload(cfg, N=N, Q=Q)
    mon = np.where(wl.mask != 0, case, 0).astype(np.int32)
    mon[0] = case
    lo_, hi_ = (0.3, 0.6) if cfg != 3 else (-0.5, 0.8)
    a = np.full(wl.d, lo_, np.float32)
    b = np.full(wl.d, hi_, np.float32)
    _check(wl.X, wl.y, wl.Xq, wl.M, mon, a, b, wl.norm, wl.weights, stated=True)


@pytest.mark.parametrize("norm", NORMS)
def test_limits_reduce_to_lipfit_bounds(norm):
    """a = b: simple monotonicity (Eq.(4)); a = -inf, b = +inf or mon = 0: no constraint -- compared with the
    GPU's own lipfit_bounds as well as with the oracle."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(2, N=5000, Q=3000)
    c = np.array([0.4, 0.7, 0.0, 0.0], np.float32)
    up, lo, g = _check(wl.X, wl.y, wl.Xq, wl.M, [1, 2, 0, 0], c, c, norm, None, stated=True)
    ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, [1, -1, 0, 0], norm)
    tol = 1e-5 * wl.y_range
    assert np.abs(up - ub.cpu().numpy()).max() <= tol and np.abs(lo - lb.cpu().numpy()).max() <= tol
    up, lo, g = _check(wl.X, wl.y, wl.Xq, wl.M, [3, 4, 1, 2], [-INF] * 4, [INF] * 4, norm, None, stated=True)
    ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, None, norm)
    assert np.abs(up - ub.cpu().numpy()).max() <= tol and np.abs(lo - lb.cpu().numpy()).max() <= tol
    _check(wl.X, wl.y, wl.Xq, wl.M, None, None, None, norm, None, stated=True)
    # half-infinite: only B (a = -inf) / only A (b = +inf) constrains
    _check(wl.X, wl.y, wl.Xq, wl.M, [1, 2, 3, 4], [-INF, -INF, 0.2, 0.3], [0.5, 0.5, INF, INF], norm, None,
           stated=True)


def test_paper_example_x_squared_case_iii():
    """f(x) = x^2 on [-1, 1] is case III with a = b = 0; the GPU bounds enclose f and interpolate."""
    import torch
    import paper_2606_04670_b200 as L
    xs = np.linspace(-1, 1, 41).astype(np.float32)[:, None]
    y = (xs[:, 0].astype(np.float64) ** 2).astype(np.float32)
    q = np.random.default_rng(0).uniform(-1, 1, (5000, 1)).astype(np.float32)
    up, lo, g = _check(xs, y, q, 2.0, [3], [0.0], [0.0], L2, None, stated=True)
    fq = q[:, 0].astype(np.float64) ** 2
    assert np.all(lo <= fq + 1e-5) and np.all(fq <= up + 1e-5)
    ug, lg, gg = L.lipfit_bounds_region(_dev(xs), _dev(y), _dev(xs), 2.0, [3], [0.0], [0.0], L2)
    assert np.abs(gg.cpu().numpy() - y).max() <= 1e-5


@pytest.mark.parametrize("N,Q", [(1, 5), (2, 1), (511, 300), (513, 129), (70000, 64), (300, 70000)])
def test_ragged_and_chunked(N, Q):
    X, y, Xq = random_problem(8, N, Q, 3)
    _check(X, y, Xq, 2.0, [3, 0, 1], [-0.3, 0.0, 0.1], [0.4, 0.0, 0.1], L2)


def test_degenerate_and_errors():
    import torch
    import paper_2606_04670_b200 as L
    X, y, Xq = random_problem(9, 100, 50, 3)
    up, lo, g = L.lipfit_bounds_region(_dev(X), _dev(y), _dev(Xq), 0.0, [1, 2, 3], [0, 0, 0], [1, 1, 1], L2)
    assert bool((up == float(y.min())).all()) and bool((lo == float(y.max())).all())          # M = 0 (R9)
    X2, y2 = np.concatenate([X, X[:10]]), np.concatenate([y, y[:10] + 1])                     # duplicates, zero weight
    _check(X2, y2, Xq, 1.0, [4, 0, 2], [-0.5, 0, -INF], [0.5, 0, 0.3], LINF, np.array([0.0, 1.0, 2.0], np.float32))
    up, lo, g = L.lipfit_bounds_region(_dev(X), _dev(y), _dev(Xq[:0]), 1.0, [1, 0, 0], [0, 0, 0], [1, 1, 1])
    assert up.numel() == 0
    for bad in (dict(mon=[5, 0, 0]), dict(a=[2.0, 0, 0]), dict(a=[float("nan"), 0, 0]), dict(M=-1.0),
                dict(a=None), dict(a=[float("inf"), 0, 0], b=[float("inf"), 1, 1])):
        kw = dict(M=1.0, mon=[1, 0, 0], a=[0.0, 0, 0], b=[1.0, 1, 1])
        kw.update(bad)
        with pytest.raises(L.LipfitError):
            L.lipfit_bounds_region(_dev(X), _dev(y), _dev(Xq), kw["M"], kw["mon"], kw["a"], kw["b"])
