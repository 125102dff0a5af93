"""GPU test of lipfit_bounds_noalloc (include/lipfit.h): Eq.(2),(3) with the scratch in a fixed file-scope
device array, for callers that cannot allocate (CUDA graph capture, serving loops).  Collected LAST on purpose
(the file name sorts after every other test file): the suite runs with `pytest -x`.

Checked: the entry point's output against the existing all-pairs path lipfit_bounds_ex(LIPFIT_BOUNDS_BRUTE) and
against the fp64 oracle, within the tolerance of tests/test_gpu_bounds.py, on two calls IN A ROW that share the
scratch (a larger problem first, so the second call runs over stale records and keys); that a repeated call does
not change the device's free memory; and that sizes beyond the fixed scratch are rejected with LIPFIT_E_LIMIT."""
import numpy as np
import pytest

import oracle
from inputs import L1, L2, LINF, make_workload, random_problem

pytestmark = pytest.mark.gpu


def _dev(a):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a, dtype=np.float32)).to("cuda:0")


def _compare(X, y, Xq, M, mask, norm, w, stated):
    """one call of the new entry point vs the existing path and the oracle; returns the new outputs"""
    import torch
    import paper_2606_04670_b200 as L
    Xd, yd, Qd = _dev(X), _dev(y), _dev(Xq)
    outs = [torch.full((len(Xq),), float("nan"), dtype=torch.float32, device="cuda:0") for _ in range(3)]
    got = L.lipfit_bounds_noalloc(Xd, yd, Qd, M, mask, norm, w, out=outs)
    ref = L.lipfit_bounds_ex(Xd, yd, Qd, M, mask, norm, w, policy=L.LIPFIT_BOUNDS_BRUTE)
    torch.cuda.synchronize()
    U, Lo, G = oracle.bounds(X, y, Xq, M, mask, norm, w)
    rng = max(float(np.max(y) - np.min(y)), 1e-30)
    tol = 1e-5 * rng                                            # north_star's bar (config-shaped inputs)
    if not stated:                                              # unstructured inputs: + rounding of the candidate
        tol += (X.shape[1] + 4) * 2.0 ** -24 * max(np.abs(U).max(), np.abs(Lo).max())
    for a, b, o in zip(got, ref, (U, Lo, G)):
        a, b = a.cpu().numpy(), b.cpu().numpy()
        assert np.all(np.isfinite(a))
        assert np.abs(a - b).max() <= tol, (np.abs(a - b).max(), tol)          # vs the existing path
        assert np.abs(a - o).max() <= tol, (np.abs(a - o).max(), tol)          # vs the oracle
    return got


def test_two_calls_in_a_row_share_the_scratch():
    # call 1: config 2 shape, many data chunks; call 2 right after it: fewer data, fewer queries, another norm
    # and mask -- it runs over the stale records and keys of call 1
    wl = make_workload(2, N=30000, Q=5003)
    _compare(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights, stated=True)
    wl3 = make_workload(3, N=2500, Q=777)
    _compare(wl3.X, wl3.y, wl3.Xq, wl3.M, wl3.mask, wl3.norm, wl3.weights, stated=True)
    # and the first problem again: identical bits to its first evaluation
    a = _compare(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights, stated=True)
    b = _compare(wl.X, wl.y, wl.Xq, wl.M, wl.mask, wl.norm, wl.weights, stated=True)
    for u, v in zip(a, b):
        assert bool((u == v).all())


@pytest.mark.parametrize("norm", [L1, L2, LINF])
@pytest.mark.parametrize("d,mask", [(1, [1]), (5, [1, 1, 1, 1, 1]), (7, [0, 1, 0, -1, 0, 0, 1]), (12, [1, 0] * 6),
                                    (32, [0, 1, -1, 0] * 8)])
def test_shapes_back_to_back(norm, d, mask):
    X, y, Xq = random_problem(700 + d, 1500 + d, 777 + d, d)
    w = (0.25 + np.arange(d) % 3).astype(np.float32)
    _compare(X, y, Xq, 1.25, mask, norm, w, stated=False)
    _compare(X[:301], y[:301], Xq[:130], 0.5, mask, norm, None, stated=False)


def test_no_device_memory_is_allocated_by_a_call():
    import torch
    import paper_2606_04670_b200 as L
    wl = make_workload(5, N=20000, Q=40000)
    Xd, yd, Qd = _dev(wl.X), _dev(wl.y), _dev(wl.Xq)
    outs = [torch.empty(wl.Q, dtype=torch.float32, device="cuda:0") for _ in range(3)]
    L.lipfit_bounds_noalloc(Xd, yd, Qd, wl.M, wl.mask, wl.norm, None, out=outs)   # set-up: symbol address, modules
    torch.cuda.synchronize()
    first = [o.clone() for o in outs]
    seen = []
    for _attempt in range(3):       # (the device-wide figure can move for reasons outside this process: retry)
        free0, _ = torch.cuda.mem_get_info()
        for _ in range(3):
            L.lipfit_bounds_noalloc(Xd, yd, Qd, wl.M, wl.mask, wl.norm, None, out=outs)
        torch.cuda.synchronize()
        free1, _ = torch.cuda.mem_get_info()
        seen.append((free0, free1))
        if free1 == free0:
            break
    assert any(a == b for a, b in seen), seen
    for u, v in zip(outs, first):
        assert bool((u == v).all())


def test_limits_and_errors():
    import torch
    import paper_2606_04670_b200 as L
    assert L.status_string(-7) not in ("ok", "unknown status")
    X, y, Xq = random_problem(3, 64, 32, 4)
    # at the limit for d <= 4 (N * 8 floats = 2^20): accepted; one datum more: rejected
    nmax = L.LIPFIT_NOALLOC_MAX_RECORD_FLOATS // 8
    Xb = _dev(np.tile(X, (nmax // 64 + 1, 1))[:nmax + 1])
    yb = _dev(np.tile(y, nmax // 64 + 1)[:nmax + 1])
    up, lo, g = L.lipfit_bounds_noalloc(Xb[:nmax].contiguous(), yb[:nmax].contiguous(), _dev(Xq), 1.0)
    ub, lb, gb = L.lipfit_bounds_ex(Xb[:nmax].contiguous(), yb[:nmax].contiguous(), _dev(Xq), 1.0,
                                    policy=L.LIPFIT_BOUNDS_BRUTE)
    torch.cuda.synchronize()
    assert float((up - ub).abs().max()) <= 1e-5 * float(y.max() - y.min()) + 8 * 2.0 ** -24 * float(ub.abs().max())
    with pytest.raises(L.LipfitError) as ei:
        L.lipfit_bounds_noalloc(Xb, yb, _dev(Xq), 1.0)
    assert ei.value.code == -7
    with pytest.raises(L.LipfitError) as ei:                       # d = 5 -> DP = 8: 12 floats per record
        L.lipfit_bounds_noalloc(_dev(np.zeros((90000, 5), np.float32)), _dev(np.zeros(90000, np.float32)),
                                _dev(np.zeros((4, 5), np.float32)), 1.0)
    assert ei.value.code == -7
    with pytest.raises(L.LipfitError) as ei:                       # too many queries for one call
        L.lipfit_bounds_noalloc(_dev(X), _dev(y), _dev(np.zeros((L.LIPFIT_NOALLOC_MAX_Q + 1, 4), np.float32)), 1.0)
    assert ei.value.code == -7
    with pytest.raises(L.LipfitError) as ei:
        L.lipfit_bounds_noalloc(_dev(X), _dev(y), _dev(Xq), -1.0)
    assert ei.value.code == -4
    up, lo, g = L.lipfit_bounds_noalloc(_dev(X), _dev(y), _dev(Xq[:0]), 1.0)       # Q = 0: OK, nothing written
    assert up.numel() == 0
