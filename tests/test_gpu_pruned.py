"""GPU parity: lipfit_bounds_pruned (NEXT-4(ii), exact spatial pruning of Eq.(2),(3) PAPER.md:103-116)
vs the fp64 oracle, and vs the unpruned lipfit_bounds (pruning must not change which datum wins)."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, oracle_subset, random_problem

pytestmark = pytest.mark.gpu
NORMS = [L1, L2, LINF]


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _check(X, y, Xq, M, mask, norm, w=None, stated=False):
    """stated=True (config-shaped inputs): north_star's 1e-5 * range only; otherwise the rounding term of
    tests/test_gpu_bounds.py::_check is added."""
    import torch
    import paper_2606_04670_b200 as L
    up, lo, g, pairs = L.lipfit_bounds_pruned(_dev(X), _dev(y), _dev(Xq), M, mask, norm, w, count_pairs=True)
    torch.cuda.synchronize()
    U, Lo, G = oracle.bounds(X, y, Xq, M, mask, norm, w)
    rng = max(float(y.max() - y.min()), 1e-30)
    mag = max(np.abs(U).max(), np.abs(Lo).max())
    tol = 1e-5 * rng + (0.0 if stated else (X.shape[1] + 4) * 2.0 ** -24 * mag)
    assert np.abs(up.cpu().numpy() - U).max() <= tol
    assert np.abs(lo.cpu().numpy() - Lo).max() <= tol
    assert np.abs(g.cpu().numpy() - G).max() <= tol
    assert pairs >= 1024 and pairs % 1024 == 0                           # whole 32 x 32 tiles, at least the seed
    return up, lo, g, pairs


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,mask", [(1, [1]), (2, None), (3, [1, -1, 0]), (4, [1, 1, 0, 0]), (5, [1] * 5),
                                    (8, [1] + [0] * 7), (12, [1, 0] * 6), (21, None), (32, [0, 1, -1, 0] * 8)])
def test_shapes(norm, d, mask):
    X, y, Xq = random_problem(900 + d, 3000 + d, 1000 + d, d)            # ragged last tile, ragged last warp
    w = (0.25 + np.arange(d) % 3).astype(np.float32)
    _check(X, y, Xq, 1.25, mask, norm, w)
    _check(X, y, Xq, 40.0, mask, norm, None)                             # large M: strong pruning
    _check(X, y, Xq, 0.0, mask, norm, None)                              # M = 0: min y / max y, nothing prunable


@pytest.mark.parametrize("cfg,N,Q", [(1, 1000, 10000), (2, 30000, 5000), (3, 9000, 1200), (5, 12000, 1500)])
def test_configs_and_same_winner_as_unpruned(cfg, N, Q):
    import paper_2606_04670_b200 as L
    wl = make_workload(cfg, N=N, Q=Q)
    up, lo, g, pairs = _check(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights, stated=True)
    ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range
    assert float((up - ub).abs().max()) <= tol and float((lo - lb).abs().max()) <= tol
    assert pairs <= (N + 31) // 32 * 32 * ((Q + 31) // 32 * 32)


def test_pruning_is_effective_on_config2_shape():
    wl = make_workload(2, N=100000, Q=20000)
    *_, pairs = _check(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights, stated=True)
    assert pairs < 0.2 * wl.N * wl.Q                                     # measured: a few per cent


def test_edges():
    import paper_2606_04670_b200 as L
    X, y, Xq = random_problem(5, 40, 130, 2)
    _check(X[:1], y[:1], Xq, 1.0, None, L2)                              # N = 1
    _check(X, y, Xq[:1], 1.0, [1, 0], L1)                                # Q = 1
    _check(X, y, Xq[:33], 1.0, [-1, 1], LINF)                            # one full warp + one query
    Xd = np.repeat(X[:3], 50, axis=0)                                    # duplicated points, different values
    yd = np.arange(150, dtype=np.float32) % 7
    _check(Xd, yd, Xq, 2.0, None, L2)
    Xc = X.copy()
    Xc[:, 1] = 0.5                                                       # a coordinate with zero range
    _check(Xc, y, Xq, 1.0, None, L2)
    _check(X, y, Xq, 1.0, None, L2, np.array([1.0, 0.0], dtype=np.float32))   # a zero weight
    _check(X, y, 100.0 * Xq, 1.0, [1, 1], L2)                            # queries far outside the data range
    out = L.lipfit_bounds_pruned(_dev(X), _dev(y), _dev(Xq[:0]), 1.0, count_pairs=True)
    assert out[0].numel() == 0 and out[3] == 0
    with pytest.raises(L.LipfitError):
        L.lipfit_bounds_pruned(_dev(X), _dev(y), _dev(Xq), -1.0)


def test_config2_full_sampled():
    """BASELINE.json configs[1] at full size, in the launch configuration bench.py --configs 9 times."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(2)
    up, lo, g, pairs = L.lipfit_bounds_pruned(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm,
                                              wl.weights, count_pairs=True)
    torch.cuda.synchronize()
    up, lo, g = up.cpu().numpy(), lo.cpu().numpy(), g.cpu().numpy()
    sel = oracle_subset(wl.Q, 300)
    U, Lo, G = oracle.bounds(wl.X, wl.y, wl.Xq[sel], wl.M, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range
    assert np.abs(up[sel] - U).max() <= tol and np.abs(lo[sel] - Lo).max() <= tol and np.abs(g[sel] - G).max() <= tol
    ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
    assert np.abs(up - ub.cpu().numpy()).max() <= tol and np.abs(lo - lb.cpu().numpy()).max() <= tol
    assert pairs < 0.2 * wl.N * wl.Q


# ---- Eq.(7) objective / gradient with the same pruning (lipfit_smooth_objective_pruned) -------------------
def _check_smooth(X, y, M, eps, mask, norm, w=None, p=1.0):
    import paper_2606_04670_b200 as L
    N = X.shape[0]
    e64 = np.zeros(N) if eps is None else eps.astype(np.float64)
    F, grad, pairs = L.lipfit_smooth_objective_pruned(_dev(X), _dev(y), M, None if eps is None else _dev(eps), mask,
                                                      norm, w, p, count_pairs=True)
    Fo, go = oracle.smooth_objective(X, y, M, e64, mask, norm, w, p)
    assert abs(F - Fo) <= 1e-5 * max(Fo, 1e-30)                          # SURVEY.md §8(c) acceptance rule (S)
    assert np.abs(grad.cpu().numpy() - go).max() <= 1e-5 * max(np.abs(go).max(), 1e-30)
    assert pairs % 1024 == 0
    return F, grad, pairs


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,mask", [(1, [1]), (2, None), (3, [1, -1, 0]), (5, [1] * 5), (8, [1] + [0] * 7),
                                    (12, [1, 0] * 6), (21, None)])
def test_smooth_objective_shapes(norm, d, mask):
    X, y, _ = random_problem(300 + d, 1500 + d, 1, d)                    # ragged last tile
    rng = np.random.default_rng(d)
    w = (0.25 + np.arange(d) % 3).astype(np.float32)
    _check_smooth(X, y, 1.25, None, mask, norm, w, 1.0)
    _check_smooth(X, y, 6.0, (0.3 * rng.standard_normal(X.shape[0])).astype(np.float32), mask, norm, None, 2.5)


def test_smooth_objective_config5_and_unpruned():
    import paper_2606_04670_b200 as L
    wl = make_workload(5, N=20000, Q=1)
    rng = np.random.default_rng(3)
    for eps in (None, (0.05 * rng.standard_normal(wl.N)).astype(np.float32)):
        F, grad, pairs = _check_smooth(wl.X, wl.y, wl.M, eps, wl.mask, wl.norm, None, wl.p)
        Fu, gu = L.lipfit_smooth_objective(_dev(wl.X), _dev(wl.y), wl.M, None if eps is None else _dev(eps), wl.mask,
                                           wl.norm, None, wl.p)
        assert abs(F - Fu) <= 1e-5 * Fu and float((grad - gu).abs().max()) <= 1e-5 * float(gu.abs().max())
        assert pairs <= 625 * 625 * 1024                                 # at most every tile pair
    # without the monotone mask only near pairs can violate (noise 0.05 against M d): the pruning bites
    *_, pairs_sym = _check_smooth(wl.X, wl.y, wl.M, None, None, wl.norm, None, wl.p)
    assert pairs_sym < 0.5 * wl.N * wl.N


def test_smooth_objective_edges():
    X, y, _ = random_problem(11, 40, 1, 2)
    _check_smooth(X[:1], y[:1], 1.0, None, None, L2)                     # N = 1: F = 0
    _check_smooth(X[:2], y[:2], 0.5, None, [1, 0], L1)
    _check_smooth(X[:33], y[:33], 0.5, None, [-1, 1], LINF)              # one full tile + one datum
    _check_smooth(np.repeat(X[:3], 20, axis=0), (np.arange(60) % 7).astype(np.float32), 2.0, None, None, L2)
    _check_smooth(X, y, 0.0, None, None, L2)                             # M = 0: every ordered pair violates


def test_smooth_objective_config5_full_vs_unpruned():
    """Config 5 at full N, in the launch configuration bench.py --configs 12 times: the pruned pass against
    the (oracle-checked, tests/test_gpu_full_configs.py) unpruned pass, and sampled gradient rows against the oracle."""
    import paper_2606_04670_b200 as L
    wl = make_workload(5, Q=1)
    X, y = _dev(wl.X), _dev(wl.y)
    F, grad, pairs = L.lipfit_smooth_objective_pruned(X, y, wl.M, None, wl.mask, wl.norm, None, wl.p, count_pairs=True)
    Fu, gu = L.lipfit_smooth_objective(X, y, wl.M, None, wl.mask, wl.norm, None, wl.p)
    assert abs(F - Fu) <= 1e-5 * Fu and float((grad - gu).abs().max()) <= 1e-5 * float(gu.abs().max())
    rows = oracle_subset(wl.N, 48)
    g_ref, _ = oracle.smooth_rows(wl.X, wl.y, wl.M, np.zeros(wl.N), rows, wl.mask, wl.norm, None, wl.p)
    assert np.abs(grad.cpu().numpy()[rows] - g_ref).max() <= 1e-5 * np.abs(g_ref).max()
    assert pairs < 0.5 * wl.N * wl.N                                     # measured: 0.22 (all coordinates monotone)


def test_lipfit_smooth_uses_the_pruned_pass_without_a_mask():
    """lipfit_smooth with no constrained coordinate and N >= 8192 evaluates Eq.(7) with the pruned pass: its
    report must agree with the oracle's objective / max violation at the returned eps, the returned eps must be a
    stationary point of the (oracle-checked) all-pairs pass, and the violations must shrink."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(5, N=9000, Q=1)
    X, yd = _dev(wl.X), _dev(wl.y)
    eps, info = L.lipfit_smooth(X, yd, wl.M, None, wl.norm, None, wl.p, max_iter=200, tol_grad=1e-6)
    torch.cuda.synchronize()
    e = eps.cpu().numpy()
    np.testing.assert_allclose(e + wl.y, yd.cpu().numpy(), atol=1e-6)    # y <- y + eps
    Fo, go = oracle.smooth_objective(wl.X, wl.y, wl.M, e.astype(np.float64), None, wl.norm, None, wl.p)
    F0o, _ = oracle.smooth_objective(wl.X, wl.y, wl.M, np.zeros(wl.N), None, wl.norm, None, wl.p)
    assert abs(info["F"] - Fo) <= 1e-5 * Fo and abs(info["F0"] - F0o) <= 1e-5 * F0o
    assert info["F"] < info["F0"] and info["max_violation"] < info["max_violation0"]
    assert abs(info["max_violation0"] - oracle.max_violation(wl.X, wl.y, wl.M, None, None, wl.norm)) <= 1e-5
    assert np.abs(go).max() <= 1e-3 * max(1.0, info["gnorm_inf"] * 1e3)  # stationary for the oracle's gradient too
    Fu, gu = L.lipfit_smooth_objective(X, _dev(wl.y), wl.M, eps, None, wl.norm, None, wl.p)
    assert abs(Fu - info["F"]) <= 1e-5 * Fu                              # SURVEY.md §8(c) rule (S), both passes


def test_auto_policy_guard_declines_when_pruning_cannot_help():
    """Under LIPFIT_BOUNDS_AUTO the pruned kernel watches the fraction of pairs its finished query groups
    evaluated and, above 40 %, stops handing out groups; the call then runs the all-pairs kernels
    (include/lipfit.h).  Adversarial case: the data lie on a cone y = -M |x - x0| and the queries sit around x0,
    so for every query all N candidates y_k + M D tie up to rounding and no box can be excluded; control: a
    config 2 shaped workload, where AUTO keeps the pruned pass.  Either way the outputs are the exact minimum /
    maximum (oracle on a query sample)."""
    import torch
    import paper_2606_04670_b200 as L
    N, Q, d, M = 16384, 1000000, 4, 2.0                                  # Q >= 4608 x SMs: the guard is on
    rng = np.random.default_rng(77)
    X = rng.random((N, d), dtype=np.float32)
    x0 = np.full(d, 0.5, np.float32)
    y = (-M * np.sqrt(((X.astype(np.float64) - x0) ** 2).sum(axis=1))).astype(np.float32)
    Xq = (x0 + 1e-3 * rng.standard_normal((Q, d))).astype(np.float32)
    Xd, yd, Qd = _dev(X), _dev(y), _dev(Xq)
    up, lo, g, pairs = L.lipfit_bounds_ex(Xd, yd, Qd, M, None, L2, None, policy=L.LIPFIT_BOUNDS_AUTO, count_pairs=True)
    assert pairs[0] == N * Q and pairs[1] == 0                           # declined: every pair, all-pairs kernels
    upp, lop, gp, pp = L.lipfit_bounds_ex(Xd, yd, Qd, M, None, L2, None, policy=L.LIPFIT_BOUNDS_PRUNED,
                                          count_pairs=True)
    assert pp[0] > 0.4 * N * Q                                           # the forced pruned pass: no pruning here
    torch.cuda.synchronize()
    rows = oracle_subset(Q, 300)
    U, Lo, _ = oracle.bounds(X, y, Xq[rows], M, None, L2, None)
    tol = 1e-5 * float(y.max() - y.min()) + (d + 4) * 2.0 ** -24 * max(np.abs(U).max(), np.abs(Lo).max())
    for a, b in ((up, upp), (lo, lop)):
        assert float((a - b).abs().max()) <= tol
    assert np.abs(up.cpu().numpy()[rows] - U).max() <= tol and np.abs(lo.cpu().numpy()[rows] - Lo).max() <= tol
    # control: config 2's shape at N Q = 2^32 keeps the pruned pass
    wl = make_workload(2, N=16384, Q=1000000)
    *_, pc = L.lipfit_bounds_ex(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights,
                                policy=L.LIPFIT_BOUNDS_AUTO, count_pairs=True)
    assert 0 < pc[0] < 0.4 * wl.N * wl.Q
