"""GPU parity: lipfit_bounds_topk (k > 1 approximation) vs the fp64 oracle."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

pytestmark = pytest.mark.gpu
NORMS = [L1, L2, LINF]


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _check(X, y, Xq, M, wk, mask, norm, w=None, stated=False):
    """stated=True (config-shaped inputs): north_star's 1e-5 * range only; otherwise the rounding term of
    tests/test_gpu_bounds.py::_check (plus the k-term weighted sum) is added."""
    import torch
    import paper_2606_04670_b200 as L
    up, lo, g = L.lipfit_bounds_topk(_dev(X), _dev(y), _dev(Xq), M, wk, mask, norm, w)
    torch.cuda.synchronize()
    U, Lo, G = oracle.bounds_topk(X, y, Xq, M, wk, mask, norm, w)
    rng = max(float(y.max() - y.min()), 1e-30)
    mag = max(np.abs(U).max(), np.abs(Lo).max())
    tol = 1e-5 * rng + (0.0 if stated else (X.shape[1] + 4 + len(wk)) * 2.0 ** -24 * mag)
    assert np.abs(up.cpu().numpy() - U).max() <= tol
    assert np.abs(lo.cpu().numpy() - Lo).max() <= tol
    assert np.abs(g.cpu().numpy() - G).max() <= tol
    return up, lo, g


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,mask", [(1, [1]), (3, [1, -1, 0]), (4, [1, 1, 0, 0]), (5, [1] * 5), (8, None),
                                    (12, [1, 0] * 6), (21, None), (32, [0, 1, -1, 0] * 8)])
def test_shapes(norm, d, mask):
    X, y, Xq = random_problem(400 + d, 2000, 700, d)
    w = (0.25 + np.arange(d) % 3).astype(np.float32)
    _check(X, y, Xq, 1.25, [0.8, 0.1, 0.1], mask, norm, w)                # the paper's example weights
    _check(X, y, Xq, 0.5, [0.3, 0.2, 0.1, 0.1, 0.1, 0.1, 0.05, 0.05], mask, norm, None)


def test_k1_equals_lipfit_bounds_and_configs():
    import torch
    import paper_2606_04670_b200 as L
    for cfg, N, Q in ((2, 30000, 2500), (3, 9000, 1200), (5, 12000, 1500)):
        wl = make_workload(cfg, N=N, Q=Q)
        up, lo, g = _check(wl.X, wl.y, wl.Xq, wl.M, [1.0], wl.mask, wl.norm, wl.weights, stated=True)
        ub, lb, gb = L.lipfit_bounds(_dev(wl.X), _dev(wl.y), _dev(wl.Xq), wl.M, wl.mask, wl.norm, wl.weights)
        tol = 1e-5 * wl.y_range
        assert float((up - ub).abs().max()) <= tol and float((lo - lb).abs().max()) <= tol
        _check(wl.X, wl.y, wl.Xq, wl.M, [0.5, 0.3, 0.2], wl.mask, wl.norm, wl.weights, stated=True)


@pytest.mark.parametrize("cfg", [2, 3, 5])
@pytest.mark.parametrize("k", [3, 8])
def test_packed_throughput_flavour_and_chunked_small_q(cfg, k):
    """Q >= 303104 runs the packed-f32x2 top-k kernel of the config's variant (duplicated records); a small Q
    against many data runs the one-query-per-thread kernel over data chunks + the merge kernel."""
    wk = np.full(k, 1.0 / k, np.float32)
    wl = make_workload(cfg, N=700, Q=310000)
    _check(wl.X, wl.y, wl.Xq, wl.M, wk, wl.mask, wl.norm, wl.weights, stated=True)
    wl = make_workload(cfg, N=60000, Q=257)
    _check(wl.X, wl.y, wl.Xq, wl.M, wk, wl.mask, wl.norm, wl.weights, stated=True)


def test_edges_and_errors():
    import torch
    import paper_2606_04670_b200 as L
    X, y, Xq = random_problem(5, 8, 130, 2)
    _check(X, y, Xq, 1.0, np.full(8, 0.125), None, L2)                    # k = N = LIPFIT_MAX_TOPK
    _check(X[:1], y[:1], Xq, 1.0, [1.0], None, L2)                        # N = 1
    with pytest.raises(L.LipfitError):
        L.lipfit_bounds_topk(_dev(X[:2]), _dev(y[:2]), _dev(Xq), 1.0, [0.5, 0.25, 0.25])       # k > N
    with pytest.raises(L.LipfitError):
        L.lipfit_bounds_topk(_dev(X), _dev(y), _dev(Xq), 1.0, np.full(9, 1 / 9))               # k > LIPFIT_MAX_TOPK
    with pytest.raises(L.LipfitError):
        L.lipfit_bounds_topk(_dev(X), _dev(y), _dev(Xq), 1.0, [1.5, -0.5])                     # negative weight
    up, lo, g = L.lipfit_bounds_topk(_dev(X), _dev(y), _dev(Xq[:0]), 1.0, [1.0])
    assert up.numel() == 0
