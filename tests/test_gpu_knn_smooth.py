"""GPU parity: lipfit_knn and the smoothing path vs the fp64 CPU oracle."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

pytestmark = pytest.mark.gpu

NORMS = [L1, L2, LINF]


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


LAST = {}   # per-call diagnostics of the most recent _gpu_knn (lipfit_knn_info)


def _gpu_knn(X, Xq, k, mask=None, side=0, norm=L2, w=None, tensor_cores=True):
    import paper_2606_04670_b200 as L
    idx, dist, info = L.lipfit_knn_ex(_dev(X), _dev(Xq), k, mask, side, norm, w, tensor_cores=tensor_cores)
    # the certificate's error bound must dominate every observed selection-key error
    assert info["key_error_ratio"] <= 1.0, info
    LAST.clear()
    LAST.update(info)
    return idx.cpu().numpy(), dist.cpu().numpy()


def check_knn(X, Xq, k, mask=None, side=0, norm=L2, w=None):
    """Acceptance rule (DESIGN.md §6 / SURVEY §8(c)): index sets equal the oracle's except among
    candidates whose fp32-rounded oracle distance is within 1 ulp of the fp32-rounded k-th distance;
    the sorted fp32 distance lists agree within 1 ulp."""
    oi, od = oracle.knn(X, Xq, k, mask, side, norm, w)
    gi, gd = _gpu_knn(X, Xq, k, mask, side, norm, w)
    od32 = od.astype(np.float32)
    assert np.all(np.diff(gd, axis=1) >= 0)
    ulp = np.spacing(np.maximum(np.abs(od32), np.float32(1e-30)))
    assert np.all(np.abs(gd - od32) <= ulp), np.abs(gd - od32).max()
    bad = 0
    for q in range(len(Xq)):
        if np.array_equal(gi[q], oi[q]):
            continue
        so, sg = set(oi[q].tolist()), set(gi[q].tolist())
        assert len(sg) == k and min(sg) >= 0 and max(sg) < len(X)
        tau = od32[q, -1]
        tie_lo = np.nextafter(tau, np.float32(-np.inf))
        tie_hi = np.nextafter(tau, np.float32(np.inf))
        # members that differ must be boundary ties (either set), identical elsewhere
        for i in so ^ sg:
            di = oracle.knn(X[i:i + 1], Xq[q:q + 1], 1, mask, side, norm, w)[1][0, 0]
            assert tie_lo <= np.float32(di) <= tie_hi, (q, i, di, tau)
        # equal sets in a different order are only allowed among equal fp32 distances
        if so == sg:
            pos = np.nonzero(gi[q] != oi[q])[0]
            assert np.all(np.abs(gd[q, pos] - od32[q, pos]) <= ulp[q, pos])
        bad += 1
    return bad


def test_config4_scaled():
    wl = make_workload(4, N=30011, Q=1500)
    check_knn(wl.X, wl.Xq, wl.k, None, 0, wl.norm)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d", [1, 3, 4, 7, 8, 16, 21, 32])
def test_symmetric_dims(norm, d):
    X, _, Xq = random_problem(200 + d, 5000, 300, d)
    w = (0.5 + np.arange(d) % 2).astype(np.float32)
    check_knn(X, Xq, 10, None, 0, norm, w)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("side", [-1, 1])
def test_one_sided(norm, side):
    X, _, Xq = random_problem(31, 4000, 200, 5)
    check_knn(X, Xq, 7, [1, -1, 0, 1, 0], side, norm)


def test_many_exact_ties_on_a_grid():
    rng = np.random.default_rng(3)
    X = rng.integers(0, 6, (3000, 3)).astype(np.float32)
    Xq = rng.integers(0, 6, (100, 3)).astype(np.float32)
    check_knn(X, Xq, 20, None, 0, L2)
    check_knn(X, Xq, 20, [1, 1, 0], 1, L1)


@pytest.mark.parametrize("N,k", [(1, 1), (5, 5), (40, 33), (200, 128), (3000, 1), (3000, 128)])
def test_k_extremes(N, k):
    X, _, Xq = random_problem(5, N, 130, 4)
    check_knn(X, Xq, k)


def test_small_q_large_n_uses_chunks():
    X, _, Xq = random_problem(6, 120000, 64, 8)
    check_knn(X, Xq, 32)


def test_certificate_and_exact_fallback():
    """The selection pool is certified per query; where the certificate fails (ties beyond the
    margin) the exact fp64 scan answers, so integer-grid data match the oracle EXACTLY, lower
    index first (R7), through both fallback branches (candidate list / k rounds)."""
    # general position: nothing needs the fallback
    wl = make_workload(4, N=20000, Q=700)
    check_knn(wl.X, wl.Xq, wl.k, None, 0, wl.norm)
    assert LAST["fallbacks"] == 0
    # integer grid, one data chunk: dozens of exact ties straddle the k-th place and the pool threshold
    rng = np.random.default_rng(11)
    X = rng.integers(0, 5, (1000, 3)).astype(np.float32)
    Xq = rng.integers(0, 5, (150, 3)).astype(np.float32)
    for norm, mask, side in ((L2, None, 0), (L1, None, 0), (LINF, [1, 0, -1], 1)):
        oi, od = oracle.knn(X, Xq, 24, mask, side, norm)
        gi, gd = _gpu_knn(X, Xq, 24, mask, side, norm)
        assert LAST["fallbacks"] > 0
        np.testing.assert_array_equal(gi, oi)
        np.testing.assert_array_equal(gd, od.astype(np.float32))
    # all data identical: more than 768 candidates tie -> the k-round branch
    X = np.ones((2000, 4), np.float32)
    Xq = rng.standard_normal((40, 4)).astype(np.float32)
    gi, gd = _gpu_knn(X, Xq, 9)
    assert LAST["fallbacks"] == 40
    np.testing.assert_array_equal(gi, np.tile(np.arange(9, dtype=np.int32), (40, 1)))
    oi, od = oracle.knn(X, Xq, 9)
    np.testing.assert_array_equal(gd, od.astype(np.float32))


@pytest.mark.parametrize("d", [1, 2, 5, 8, 13, 16])
def test_tensor_core_and_cuda_core_selection_agree(d):
    """Symmetric L2, d <= 16 selects on the tensor cores (bf16x3 cross-term GEMM); switching them off
    uses the FFMA2 kernel.  Both feed the same exact re-rank: identical outputs, both equal to the oracle."""
    import paper_2606_04670_b200 as L
    assert "tc" in L.knn_variant(d, 0, L2) and "tc" not in L.knn_variant(17, 0, L2)
    assert "tc" not in L.knn_variant(d, 1, L2) and "tc" not in L.knn_variant(d, 0, L1)
    X, _, Xq = random_problem(300 + d, 20011, 700, d, spread=3.0)
    X += 5.0                                                   # off-centre data: the centring matters
    Xq += 5.0
    w = (0.5 + np.arange(d) % 2).astype(np.float32)
    check_knn(X, Xq, 32, None, 0, L2, w)
    a = _gpu_knn(X, Xq, 32, None, 0, L2, w)
    assert LAST["tensor_cores"]
    assert "tc" not in L.knn_variant(d, 0, L2, tensor_cores=False)
    b = _gpu_knn(X, Xq, 32, None, 0, L2, w, tensor_cores=False)
    assert not LAST["tensor_cores"]
    np.testing.assert_array_equal(a[0], b[0])
    np.testing.assert_array_equal(a[1], b[1])


@pytest.mark.parametrize("k", [32, 56, 80, 100])
def test_tensor_core_threshold_seeding(k):
    """Work items that sweep >= 768 B tiles seed their thresholds from group minima of the first tiles
    (knn_tc.cu, phase A; k + margin <= 88 of the 96 minima, so k = 100 runs unseeded; items of >= 4096 tiles,
    groups of 8 tiles, are covered by the full-size config 4 test).  Full one-chunk items (seeded) and a
    chunked tail block (not seeded) in one call; a sample of the queries against the oracle, all of them
    against the CUDA-core selection."""
    N, Q, d = 100003, 148 * 256 + 100, 16
    X, _, Xq = random_problem(77 + k, N, Q, d)
    gi, gd = _gpu_knn(X, Xq, k)
    assert LAST["fallbacks"] == 0 and LAST["tensor_cores"]
    ci, cd = _gpu_knn(X, Xq, k, tensor_cores=False)
    np.testing.assert_array_equal(gi, ci)
    np.testing.assert_array_equal(gd, cd)
    rows = np.r_[0:200, Q - 200:Q, np.arange(200, Q - 200, 97)[:300]]
    oi, od = oracle.knn(X, Xq[rows], k)
    np.testing.assert_array_equal(gi[rows], oi)
    od32 = od.astype(np.float32)
    assert np.all(np.abs(gd[rows] - od32) <= np.spacing(od32))


def test_knn_host_and_errors():
    import paper_2606_04670_b200 as L
    X, _, Xq = random_problem(7, 2000, 100, 4)
    hi, hd = L.lipfit_knn_host(X, Xq, 5)
    gi, gd = _gpu_knn(X, Xq, 5)
    np.testing.assert_array_equal(hi, gi)
    np.testing.assert_array_equal(hd, gd)
    with pytest.raises(L.LipfitError):
        L.lipfit_knn_host(X, Xq, 2001)
    with pytest.raises(L.LipfitError):
        L.lipfit_knn_host(X, Xq, 129)


# --------------------------------------------------------------------------------------------
# smoothing
# --------------------------------------------------------------------------------------------
def _gpu_obj(X, y, M, eps, mask, norm, w, p):
    import torch
    import paper_2606_04670_b200 as L
    F, g = L.lipfit_smooth_objective(_dev(X), _dev(y), M, None if eps is None else _dev(eps), mask,
                                     norm, w, p)
    torch.cuda.synchronize()
    return F, g.cpu().numpy()


def check_objective(X, y, M, mask, norm, w, p, sigma=0.05, seed=0):
    rng = np.random.default_rng(seed)
    N = len(y)
    for eps in (None, (sigma * rng.standard_normal(N)).astype(np.float32),
                (sigma * rng.standard_normal(N)).astype(np.float32)):
        e64 = np.zeros(N) if eps is None else eps.astype(np.float64)
        F, grad = oracle.smooth_objective(X, y, M, e64, mask, norm, w, p)
        Fg, gg = _gpu_obj(X, y, M, eps, mask, norm, w, p)
        assert abs(Fg - F) <= 1e-5 * max(abs(F), 1e-30), (Fg, F)
        gscale = max(np.abs(grad).max(), 1e-30)
        assert np.abs(gg - grad).max() <= 1e-5 * gscale, (np.abs(gg - grad).max(), gscale)


def test_objective_config5_scaled():
    wl = make_workload(5, N=6007)
    check_objective(wl.X, wl.y, wl.M, wl.mask, wl.norm, wl.weights, wl.p)


@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,mask", [(2, None), (3, [1, 0, -1]), (5, [1] * 5), (8, [0, 1] * 4),
                                    (13, [1] * 13), (32, [0] * 32)])
def test_objective_shapes(norm, d, mask):
    X, y, _ = random_problem(300 + d, 1300, 1, d, spread=0.3)
    w = (0.5 + np.arange(d) % 2).astype(np.float32)
    check_objective(X, y, 0.7, mask, norm, w, 0.5, sigma=0.2, seed=d)


@pytest.mark.parametrize("scale", [1.0e4, 1.0e7, 1.0e-6])
@pytest.mark.parametrize("mask", [[1] * 5, None])
def test_gradient_fixed_point_scale(scale, mask):
    """The gradient sums are 64-bit fixed point with a scale chosen per evaluation from N (z_max - z_min)
    (csrc/smooth.cu): data with |y| of order 1e4 or 1e7 (row sums far beyond 2^23, where a fixed 2^-40 scale
    wrapped silently) and of order 1e-6 (where a coarse scale would lose everything) must still match the oracle.
    Both passes: the all-pairs kernel (mask) and, for N >= 8192 without a mask, what lipfit_smooth would use."""
    wl = make_workload(5, N=6007)
    y = (wl.y.astype(np.float64) * scale).astype(np.float32)
    check_objective(wl.X, y, wl.M * scale, mask, wl.norm, None, wl.p, sigma=0.05 * scale, seed=3)


def test_objective_consistent_data_is_zero():
    wl = make_workload(1, N=900)
    F, g = _gpu_obj(wl.X, wl.y, wl.M, None, wl.mask, wl.norm, None, 1.0)
    assert F == 0.0 and np.all(g == 0.0)


@pytest.mark.parametrize("N", [2, 3, 50, 2000])
def test_minimiser_parity(N):
    """Unique minimiser (strong convexity, R14): GPU LBFGS result vs the oracle's minimiser."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(5, N=N)
    if N <= 3:   # make the tiny cases inconsistent for sure
        wl.y[:] = np.array([1.0, -1.0, 0.5][:N], np.float32)
    eps_o, info_o = oracle.smooth(wl.X, wl.y, wl.M, wl.mask, wl.norm, None, wl.p)
    yd = _dev(wl.y)
    eps, info = L.lipfit_smooth(_dev(wl.X), yd, wl.M, wl.mask, wl.norm, None, wl.p, max_iter=500,
                                tol_grad=1e-7)
    torch.cuda.synchronize()
    z_gpu = yd.cpu().numpy().astype(np.float64)
    z_or = wl.y.astype(np.float64) + eps_o
    rng = max(wl.y_range, 1e-30)
    assert np.abs(z_gpu - z_or).max() <= 1e-5 * rng, (np.abs(z_gpu - z_or).max(), info, info_o)
    np.testing.assert_allclose(eps.cpu().numpy() + wl.y, z_gpu, atol=1e-6)
    assert info["F"] <= info["F0"]
    assert info["max_violation"] <= info["max_violation0"] + 1e-7
    assert abs(float(eps.sum().cpu())) <= 1e-3 * max(1.0, float(eps.abs().sum().cpu()))


def test_smooth_then_bounds_config5_scaled():
    """S(3): the GPU bounds on the GPU's smoothed z match the oracle bounds on the same z."""
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(5, N=4000, Q=3000)
    yd = _dev(wl.y)
    eps, info = L.lipfit_smooth(_dev(wl.X), yd, wl.M, wl.mask, wl.norm, None, wl.p, max_iter=200)
    z = yd.cpu().numpy()
    assert info["F"] < info["F0"] and info["max_violation"] < info["max_violation0"]
    U, Lo, g = oracle.bounds(wl.X, z, wl.Xq, wl.M, wl.mask, wl.norm)
    up, lo, gg = L.lipfit_bounds(_dev(wl.X), yd, _dev(wl.Xq), wl.M, wl.mask, wl.norm)
    torch.cuda.synchronize()
    tol = 1e-5 * wl.y_range
    assert np.abs(up.cpu().numpy() - U).max() <= tol
    assert np.abs(lo.cpu().numpy() - Lo).max() <= tol
    assert np.abs(gg.cpu().numpy() - g).max() <= tol
    ys, e2, info2 = L.lipfit_smooth_host(wl.X, wl.y, wl.M, wl.mask, wl.norm, None, wl.p, 200)
    np.testing.assert_array_equal(ys, z)          # an evaluation is bit-reproducible


# --------------------------------------------------------------------------------------------
# NEXT-3: smallest consistent Lipschitz constant
# --------------------------------------------------------------------------------------------
@pytest.mark.parametrize("norm", NORMS)
@pytest.mark.parametrize("d,mask", [(1, [1]), (2, None), (5, [1, 1, 1, 1, 1]), (5, None), (7, [0, 1, 0, -1, 0, 0, 1]),
                                    (12, None), (20, [1, 0] * 10)])
def test_lipschitz_constant_shapes(norm, d, mask):
    import paper_2606_04670_b200 as L
    X, _, _ = random_problem(40 + d, 3001, 1, d)
    s = np.zeros(d) if mask is None else np.asarray(mask, np.float64)
    rng = np.random.default_rng(d)
    y = (X.astype(np.float64) @ np.where(s == 0, 0.3, s) +
         (0.0 if mask is not None else 0.2) * rng.standard_normal(len(X))).astype(np.float32)
    w = (0.5 + np.arange(d) % 3).astype(np.float32)
    ref = oracle.lipschitz_constant(X, y, mask, norm, w)
    got = float(L.lipfit_lipschitz_constant(_dev(X), _dev(y), mask, norm, w).cpu()[0])
    assert np.isfinite(ref) and abs(got - ref) <= 1e-5 * ref, (got, ref)
    assert L.lipfit_lipschitz_constant_host(X, y, mask, norm, w) == got


def test_lipschitz_constant_config_scaled_and_degenerate():
    import paper_2606_04670_b200 as L
    for cfg, N in ((1, 1000), (2, 9001), (5, 12000)):
        wl = make_workload(cfg, N=N)
        ref = oracle.lipschitz_constant(wl.X, wl.y, wl.mask, wl.norm, wl.weights)
        got = L.lipfit_lipschitz_constant_host(wl.X, wl.y, wl.mask, wl.norm, wl.weights)
        assert (np.isinf(ref) and np.isinf(got)) or abs(got - ref) <= 1e-5 * ref, (cfg, got, ref)
    # consistency threshold: with M slightly above L the smoothing objective at eps = 0 is exactly 0
    wl = make_workload(1, N=1000)
    Lc = L.lipfit_lipschitz_constant_host(wl.X, wl.y, wl.mask, wl.norm)
    F, _ = L.lipfit_smooth_objective(_dev(wl.X), _dev(wl.y), Lc * (1 + 1e-5), None, wl.mask, wl.norm)
    assert F == 0.0
    X = np.array([[0, 0], [0, 0], [1, 0]], np.float32)
    assert L.lipfit_lipschitz_constant_host(X, np.array([1, 1, 1], np.float32)) == 0.0
    assert L.lipfit_lipschitz_constant_host(X, np.array([1, 2, 1], np.float32)) == np.inf
    assert L.lipfit_lipschitz_constant_host(X[:1], np.ones(1, np.float32)) == 0.0
