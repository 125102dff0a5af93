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


def _check(X, y, Xq, M, mask, norm, w=None):
    import torch
    import paper_2606_04670_b200 as L
    up, lo, g, pairs = L.lipfit_bounds_pruned(_dev(X), _dev(y), _dev(Xq), M, mask, norm, w, count_pairs=True)
    torch.cuda.synchronize()
    U, Lo, G = oracle.bounds(X, y, Xq, M, mask, norm, w)
    rng = max(float(y.max() - y.min()), 1e-30)
    mag = max(np.abs(U).max(), np.abs(Lo).max())
    tol = 1e-5 * rng + (X.shape[1] + 4) * 2.0 ** -24 * mag               # as tests/test_gpu_bounds.py
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
    up, lo, g, pairs = _check(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights)
    ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
    tol = 1e-5 * wl.y_range
    assert float((up - ub).abs().max()) <= tol and float((lo - lb).abs().max()) <= tol
    assert pairs <= (N + 31) // 32 * 32 * ((Q + 31) // 32 * 32)


def test_pruning_is_effective_on_config2_shape():
    wl = make_workload(2, N=100000, Q=20000)
    *_, pairs = _check(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights)
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
