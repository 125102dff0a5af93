"""GPU parity sweep: seeded random (d, mask, norm, weights, M, N, Q) cases through EVERY route to Eq.(2),(3)
PAPER.md:103-116 -- lipfit_bounds (LIPFIT_BOUNDS_AUTO: single-launch small kernel / pruned pass / all-pairs kernels),
lipfit_bounds_ex BRUTE and PRUNED, lipfit_bounds_noalloc, lipfit_bounds_region with mon = 0 and with a = b
(simple monotonicity, Eq.(4)), lipfit_bounds_topk with k = 1 -- against the fp64 oracle, element by element.
The dispatch tables (tuned shapes, even-rounded padded shapes for d <= 8, chunked generic kernels for d > 8, one
kernel per number of restricted pairs in region.cu) are walked by the random masks; sizes straddle the tile,
chunk and small-kernel boundaries."""
import numpy as np
import pytest

import oracle
from inputs import random_problem

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _case(seed):
    rng = np.random.default_rng(10_000 + seed)
    d = int(rng.choice([1, 2, 3, 4, 5, 6, 7, 8, 9, 12, 16, 17, 24, 32], p=[.08, .1, .1, .1, .1, .1, .1, .1, .04, .05, .05, .03, .03, .02]))
    mask = rng.choice([-1, 0, 1], size=d, p=[.25, .5, .25]).astype(np.int32)
    norm = int(rng.integers(1, 4))
    w = None if rng.random() < 0.3 else rng.choice([0.0, 0.25, 0.5, 1.0, 1.5, 2.0], size=d).astype(np.float32)
    M = float(rng.choice([0.0, 0.3, 1.0, 2.5, 8.0]))
    N = int(rng.choice([1, 2, 31, 32, 33, 127, 500, 1024, 1537, 3000, 9000]))
    Q = int(rng.choice([1, 31, 32, 33, 129, 700, 2049, 5000]))
    return d, mask, norm, w, M, N, Q


@pytest.mark.parametrize("seed", range(120))
def test_every_route_matches_the_oracle(seed):
    import torch
    import paper_2606_04670_b200 as L
    d, mask, norm, w, M, N, Q = _case(seed)
    X, y, Xq = random_problem(20_000 + seed, N, Q, d)
    U, Lo, G = oracle.bounds(X, y, Xq, M, mask, norm, w)
    rng = max(float(y.max() - y.min()), 1e-30) if N > 1 else 1.0
    mag = max(np.abs(U).max(), np.abs(Lo).max())
    tol = 1e-5 * rng + (2 * d + 4) * 2.0 ** -24 * mag        # unstructured inputs; 2d: region kernel
    Xd, yd, Qd = _dev(X), _dev(y), _dev(Xq)
    routes = {
        "auto": L.lipfit_bounds(Xd, yd, Qd, M, mask, norm, w),
        "brute": L.lipfit_bounds_ex(Xd, yd, Qd, M, mask, norm, w, policy=L.LIPFIT_BOUNDS_BRUTE),
        "pruned": L.lipfit_bounds_ex(Xd, yd, Qd, M, mask, norm, w, policy=L.LIPFIT_BOUNDS_PRUNED),
        "topk1": L.lipfit_bounds_topk(Xd, yd, Qd, M, [1.0], mask, norm, w),
    }
    routes["noalloc"] = L.lipfit_bounds_noalloc(Xd, yd, Qd, M, mask, norm, w)     # N (DP + 4) <= 9000 * 36 floats
    # region entry point: case I / II with a = b anywhere is simple monotonicity +1 / -1; mon = 0 is unrestricted
    mon = np.where(mask > 0, 1, np.where(mask < 0, 2, 0)).astype(np.int32)
    thr = np.random.default_rng(seed).uniform(-1, 1, d).astype(np.float32)
    routes["region"] = L.lipfit_bounds_region(Xd, yd, Qd, M, mon, thr, thr, norm, w)
    torch.cuda.synchronize()
    for name, (up, lo, g) in routes.items():
        up, lo, g = up.cpu().numpy(), lo.cpu().numpy(), g.cpu().numpy()
        assert np.abs(up - U).max() <= tol, (name, d, mask.tolist(), norm, N, Q, np.abs(up - U).max(), tol)
        assert np.abs(lo - Lo).max() <= tol, (name, d, mask.tolist(), norm, N, Q, np.abs(lo - Lo).max(), tol)
        assert np.abs(g - G).max() <= tol, (name, d, mask.tolist(), norm, N, Q)


@pytest.mark.parametrize("seed", range(40))
def test_knn_routes_match_the_oracle(seed):
    """lipfit_knn_ex with and without the tensor-core selection (where it applies), random shape / norm / side /
    k: continuous random data have no ties, so index sets and order equal the oracle's exactly and the distances
    are the fp64 distances rounded to fp32."""
    import paper_2606_04670_b200 as L
    rng = np.random.default_rng(30_000 + seed)
    d = int(rng.choice([1, 2, 3, 5, 8, 13, 16, 17, 32]))
    norm = int(rng.integers(1, 4))
    side = int(rng.choice([0, 0, 1, -1]))
    mask = rng.choice([-1, 0, 1], size=d).astype(np.int32)
    if side != 0 and not mask.any():
        mask[0] = 1
    N = int(rng.choice([40, 129, 1000, 4097, 12000]))
    Q = int(rng.choice([1, 33, 257, 700]))
    k = int(min(N, rng.choice([1, 5, 32, 100])))
    w = None if rng.random() < 0.5 else rng.choice([0.5, 1.0, 2.0], size=d).astype(np.float32)
    X, _, Xq = random_problem(40_000 + seed, N, Q, d)
    oi, od = oracle.knn(X, Xq, k, mask, side, norm, w)
    for tc in (True, False):
        idx, dist, info = L.lipfit_knn_ex(_dev(X), _dev(Xq), k, mask, side, norm, w, tensor_cores=tc)
        assert info["key_error_ratio"] <= 1.0, info
        np.testing.assert_array_equal(idx.cpu().numpy(), oi, err_msg=str((d, norm, side, N, Q, k, tc)))
        np.testing.assert_array_equal(dist.cpu().numpy(), od.astype(np.float32))


@pytest.mark.parametrize("seed", range(48))
def test_lipschitz_constant_and_smoothing_objective_shapes(seed):
    """lipfit_lipschitz_constant (exact-d symmetric kernels for d <= 8, generic otherwise) and the Eq.(7)
    objective / gradient through both passes (all pairs, exactly pruned) on random shapes against the oracle."""
    import paper_2606_04670_b200 as L
    rng = np.random.default_rng(50_000 + seed)
    d = int(rng.choice([1, 2, 3, 4, 5, 6, 7, 8, 11, 16, 20]))
    norm = int(rng.integers(1, 4))
    symmetric = seed % 3 != 0
    mask = None if symmetric else rng.choice([-1, 0, 1], size=d).astype(np.int32)
    N = int(rng.choice([2, 33, 500, 1300, 2600]))
    w = None if rng.random() < 0.5 else rng.choice([0.5, 1.0, 2.0], size=d).astype(np.float32)
    X, _, _ = random_problem(60_000 + seed, N, 1, d, spread=0.5)
    # a smooth monotone-compatible signal plus noise: finite Lipschitz constant when symmetric
    s = np.zeros(d) if mask is None else mask.astype(np.float64)
    y = ((X.astype(np.float64) * (s + 0.3)).sum(axis=1) + 0.2 * rng.standard_normal(N)).astype(np.float32)
    Xd, yd = _dev(X), _dev(y)
    ref = oracle.lipschitz_constant(X, y, mask, norm, w)
    got = float(L.lipfit_lipschitz_constant(Xd, yd, mask, norm, w).cpu()[0])
    assert (np.isinf(ref) and np.isinf(got)) or got == float(np.float32(ref)), (d, norm, symmetric, N, got, ref)
    M, p = 0.6, 0.7
    eps = (0.1 * rng.standard_normal(N)).astype(np.float32)
    F, grad = oracle.smooth_objective(X, y, M, eps.astype(np.float64), mask, norm, w, p)
    gscale = max(np.abs(grad).max(), 1e-30)
    Fa, ga = L.lipfit_smooth_objective(Xd, yd, M, _dev(eps), mask, norm, w, p)
    Fp, gp = L.lipfit_smooth_objective_pruned(Xd, yd, M, _dev(eps), mask, norm, w, p)
    for name, Fg, gg in (("all pairs", Fa, ga), ("pruned", Fp, gp)):
        assert abs(Fg - F) <= 1e-5 * max(abs(F), 1e-30), (name, d, norm, N, Fg, F)
        assert np.abs(gg.cpu().numpy() - grad).max() <= 1e-5 * gscale, (name, d, norm, N)
