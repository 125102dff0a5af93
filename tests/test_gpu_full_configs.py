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
    """Both evaluation policies bench.py times: the all-pairs kernels (LIPFIT_BOUNDS_BRUTE) and what the plain
    entry point lipfit_bounds does at these sizes (LIPFIT_BOUNDS_AUTO -> exact pruning)."""
    import torch
    import paper_2606_04670_b200 as L
    yv = wl.y if y is None else y
    sel = oracle_subset(wl.Q, n_sample)
    U, Lo, G = oracle.bounds(wl.X, yv, wl.Xq[sel], wl.M, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range                                   # the north_star bar (R18: range of the INPUT y)
    res = {}
    for policy in (L.LIPFIT_BOUNDS_BRUTE, L.LIPFIT_BOUNDS_AUTO):
        if policy == L.LIPFIT_BOUNDS_AUTO:
            up, lo, g = L.lipfit_bounds(_dev(wl.X), _dev(yv), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
        else:
            up, lo, g = L.lipfit_bounds_ex(_dev(wl.X), _dev(yv), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights,
                                           policy=policy)
        torch.cuda.synchronize()
        up, lo, g = up.cpu().numpy(), lo.cpu().numpy(), g.cpu().numpy()
        assert np.abs(up[sel] - U).max() <= tol
        assert np.abs(lo[sel] - Lo).max() <= tol
        assert np.abs(g[sel] - G).max() <= tol
        # any size: g is the midpoint; every bound is finite; upper >= min y, lower <= max y
        assert np.all(np.isfinite(up)) and np.all(np.isfinite(lo))
        assert np.abs(g - 0.5 * (up.astype(np.float64) + lo)).max() <= 1e-6 * max(1.0, np.abs(g).max())
        assert up.min() >= yv.min() and lo.max() <= yv.max()
        res[policy] = (up, lo, g)
    # the two passes take the minimum / maximum over the same N data: they agree everywhere within the bar
    for u, v in zip(res[L.LIPFIT_BOUNDS_BRUTE], res[L.LIPFIT_BOUNDS_AUTO]):
        assert np.abs(u - v).max() <= tol
    return res[L.LIPFIT_BOUNDS_AUTO]


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


def test_local_lipschitz_full():
    """NEXT-1 at full size (config 5's data, N = 2e5, J = 16 knots from 1e6 sampled pairs): 64 rows of the step
    tables against oracle.local_lipschitz_rows, and 400 queries of the evaluation against oracle.values_local
    on a SYNTHETIC seeded table (non-decreasing rows; the oracle never sees a GPU result).  Knot-band
    sandwich as in tests/test_gpu_local.py (R22)."""
    import torch
    import paper_2606_04670_b200 as L
    from inputs import sample_pairs
    EPS, TOL = 4e-6, 2e-5
    wl = make_workload(5)
    J = L.LIPFIT_LOCAL_KNOTS
    pi, pk = sample_pairs(3, wl.N, 1_000_000)
    Xd, yd = _dev(wl.X), _dev(wl.y)
    knots = L.lipfit_distance_quantiles(Xd, _dev(pi), _dev(pk), J, wl.norm)
    np.testing.assert_allclose(knots, oracle.distance_quantiles(wl.X, pi, pk, J, wl.norm), rtol=2e-6)
    table = L.lipfit_local_lipschitz(Xd, yd, knots, wl.norm)
    torch.cuda.synchronize()
    rows = oracle_subset(wl.N, 64)
    got = table.cpu().numpy()[rows].astype(np.float64)
    k64 = knots.astype(np.float64)
    lo = oracle.local_lipschitz_rows(wl.X, wl.y, k64 * (1 - EPS), rows, wl.norm)
    hi = oracle.local_lipschitz_rows(wl.X, wl.y, k64 * (1 + EPS), rows, wl.norm)
    assert np.all(got >= lo * (1 - TOL)) and np.all(got <= hi * (1 + TOL))
    same = lo == hi
    assert same.mean() > 0.98
    ref = oracle.local_lipschitz_rows(wl.X, wl.y, k64, rows, wl.norm)
    np.testing.assert_allclose(got[same], ref[same], rtol=TOL)
    # evaluation on a synthetic table: running maxima of positive draws around the config's slope scale
    rng = np.random.default_rng(5)
    syn = np.maximum.accumulate(rng.uniform(0.2, 6.0, (wl.N, J)), axis=1).astype(np.float32)
    sel = oracle_subset(wl.Q, 400)
    up, lo_, g = L.lipfit_values_local(Xd, yd, _dev(wl.Xq), knots, _dev(syn), wl.norm)
    torch.cuda.synchronize()
    up, lo_ = up.cpu().numpy()[sel].astype(np.float64), lo_.cpu().numpy()[sel].astype(np.float64)
    t64 = syn.astype(np.float64)
    Ua, La, _ = oracle.values_local(wl.X, wl.y, wl.Xq[sel], k64 * (1 - EPS), t64, wl.norm)
    Ub, Lb, _ = oracle.values_local(wl.X, wl.y, wl.Xq[sel], k64 * (1 + EPS), t64, wl.norm)
    tol = 1e-5 * wl.y_range
    assert np.all(up <= np.maximum(Ua, Ub) + tol) and np.all(up >= np.minimum(Ua, Ub) - tol)
    assert np.all(lo_ <= np.maximum(La, Lb) + tol) and np.all(lo_ >= np.minimum(La, Lb) - tol)
    U, Lo, _ = oracle.values_local(wl.X, wl.y, wl.Xq[sel], k64, t64, wl.norm)
    same = (Ua == Ub) & (La == Lb)
    assert same.mean() > 0.95
    assert np.abs(up[same] - U[same]).max() <= tol and np.abs(lo_[same] - Lo[same]).max() <= tol


def test_bounds_topk_full():
    """NEXT-2 at full size (config 2, k = 4 best bound values): 300 sampled queries against the oracle."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(2)
    wk = np.array([0.4, 0.3, 0.2, 0.1], np.float32)
    up, lo, g = L.lipfit_bounds_topk(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wk, wl.mask, wl.norm, wl.weights)
    torch.cuda.synchronize()
    sel = oracle_subset(wl.Q, 300)
    U, Lo, G = oracle.bounds_topk(wl.X, wl.y, wl.Xq[sel], wl.M, wk, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range
    assert np.abs(up.cpu().numpy()[sel] - U).max() <= tol
    assert np.abs(lo.cpu().numpy()[sel] - Lo).max() <= tol
    assert np.abs(g.cpu().numpy()[sel] - G).max() <= tol


def test_bounds_region_full():
    """NEXT-4(iii) at full size (config 2's data and queries, case III on x1, case I on x2, thresholds inside
    the data): 300 sampled queries against the oracle."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(2)
    mon, a, b = [3, 1, 0, 0], [0.3, 0.4, 0, 0], [0.6, 0.4, 0, 0]
    up, lo, g = L.lipfit_bounds_region(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, mon, a, b, wl.norm, wl.weights)
    torch.cuda.synchronize()
    sel = oracle_subset(wl.Q, 300)
    U, Lo, G = oracle.bounds_region(wl.X, wl.y, wl.Xq[sel], wl.M, mon, a, b, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range
    assert np.abs(up.cpu().numpy()[sel] - U).max() <= tol
    assert np.abs(lo.cpu().numpy()[sel] - Lo).max() <= tol
    assert np.abs(g.cpu().numpy()[sel] - G).max() <= tol


def test_concurrent_calls_on_two_streams_from_two_threads():
    """include/lipfit.h, "Thread safety": compute calls keep no state outside their arguments.  lipfit_bounds
    and lipfit_knn_ex run at the same time from two host threads on two non-default streams, repeatedly, and
    must reproduce the serial results bit for bit."""
    import threading
    import torch
    import paper_2606_04670_b200 as L
    wb = make_workload(2, N=20000, Q=150000)
    wk = make_workload(4, N=50000, Q=20000)
    Xb, yb, Qb = _dev(wb.X), _dev(wb.y), _dev(wb.Xq)
    Xk, Qk = _dev(wk.X), _dev(wk.Xq)
    ref_b = [t.clone() for t in L.lipfit_bounds(Xb, yb, Qb, wb.M, wb.mask, wb.norm, wb.weights)]
    ri, rd, _ = L.lipfit_knn_ex(Xk, Qk, wk.k)
    torch.cuda.synchronize()
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    out, err = {}, []

    def run_bounds():
        try:
            with torch.cuda.stream(s1):
                for _ in range(6):
                    out["b"] = L.lipfit_bounds(Xb, yb, Qb, wb.M, wb.mask, wb.norm, wb.weights, stream=s1)
            s1.synchronize()
        except Exception as e:  # surfaced below
            err.append(e)

    def run_knn():
        try:
            with torch.cuda.stream(s2):
                for _ in range(3):
                    out["k"] = L.lipfit_knn_ex(Xk, Qk, wk.k, stream=s2)
            s2.synchronize()
        except Exception as e:
            err.append(e)

    ts = [threading.Thread(target=run_bounds), threading.Thread(target=run_knn)]
    for t in ts:
        t.start()
    for t in ts:
        t.join()
    assert not err, err
    torch.cuda.synchronize()
    for u, v in zip(out["b"], ref_b):
        assert torch.equal(u, v)
    assert torch.equal(out["k"][0], ri) and torch.equal(out["k"][1], rd)
    assert out["k"][2]["fallbacks"] == 0 and out["k"][2]["key_error_ratio"] <= 1.0
