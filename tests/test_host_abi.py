"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads, exports every symbol
include/lipfit.h declares, validates arguments before touching the device, and its host LBFGS (step
a5) finds the unique minimiser of Eq.(7) when driven by the oracle's objective.  No kernels run."""
import os
import re

import numpy as np
import pytest

import oracle
import paper_2606_04670_b200 as L
from inputs import L1, L2, LINF, make_workload, random_problem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = L.load()
    header = open(os.path.join(ROOT, "include", "lipfit.h")).read()
    header = re.sub(r"/\*.*?\*/", "", header, flags=re.S)
    declared = set(re.findall(r"\b(lipfit_[a-z_]+)\s*\(", header))
    declared -= {"lipfit_eval_fn"}
    assert len(declared) >= 12
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert set(L.binding.EXPORTS) == declared
    assert L.version().count(".") == 2


def test_status_strings_and_variant_names():
    assert L.status_string(0) == "ok"
    for code in range(-6, 0):
        assert L.status_string(code) not in ("ok", "unknown status")
    assert L.bounds_variant(2, None, L2) == "bounds<L2,U2,C0>"
    assert L.bounds_variant(4, [1, 1, 0, 0], L1) == "bounds<L1,U2,C2,folded>"
    assert L.bounds_variant(8, [1] + [0] * 7, LINF) == "bounds<Linf,U7,C1,packed>"
    assert L.bounds_variant(5, [1] * 5, L2) == "bounds<L2,U0,C5,packed>"
    assert L.bounds_variant(5, [-1] * 5, L2) == "bounds<L2,U0,C5,packed>"     # mirrored coordinates (R2)
    assert L.bounds_variant(9, None, L1).startswith("bounds_generic<L1,DP16")
    with pytest.raises(L.LipfitError):
        L.bounds_variant(33, None, L2)
    with pytest.raises(L.LipfitError):
        L.bounds_variant(3, [0, 5, 0], L2)


def test_argument_validation_happens_before_any_device_work():
    X, y, Xq = random_problem(0, 10, 4, 3)
    E = L.LipfitError
    cases = [
        (dict(M=-1.0), -4), (dict(M=float("nan")), -4), (dict(norm=0), -4),
        (dict(mono_mask=[0, 2, 0]), -4), (dict(weights=[1, -1, 1]), -4),
        (dict(weights=[1, float("inf"), 1]), -4),
    ]
    for kw, code in cases:
        args = dict(M=1.0, mono_mask=None, norm=L2, weights=None)
        args.update(kw)
        with pytest.raises(E) as ei:
            L.lipfit_bounds_host(X, y, Xq, args["M"], args["mono_mask"], args["norm"], args["weights"])
        assert ei.value.code == code, (kw, ei.value.code)
    with pytest.raises(E) as ei:
        L.lipfit_knn_host(X, Xq, 11)
    assert ei.value.code == -3
    with pytest.raises(E) as ei:
        L.lipfit_knn_host(X, Xq, 2, side=3)
    assert ei.value.code == -4
    with pytest.raises(E) as ei:
        L.lipfit_smooth_host(X, y, 1.0, p=0.0)
    assert ei.value.code == -4
    # Q = 0 is OK without a device: nothing to do (R9)
    up, lo, g = L.lipfit_bounds_host(X, y, Xq[:0], 1.0)
    assert up.size == 0


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a device is present")
    X, y, Xq = random_problem(0, 10, 4, 3)
    with pytest.raises(L.LipfitError) as ei:
        L.lipfit_bounds_host(X, y, Xq, 1.0)
    assert ei.value.code in (-5, -6)
    with pytest.raises(RuntimeError):
        L.lipfit_bounds(torch.zeros(3, 2), torch.zeros(3), torch.zeros(1, 2), 1.0)


def test_host_lbfgs_on_textbook_functions():
    def rosen(x):
        f = np.sum(100 * (x[1:] - x[:-1] ** 2) ** 2 + (1 - x[:-1]) ** 2)
        g = np.zeros_like(x)
        g[:-1] += -400 * x[:-1] * (x[1:] - x[:-1] ** 2) - 2 * (1 - x[:-1])
        g[1:] += 200 * (x[1:] - x[:-1] ** 2)
        return f, g
    x, info = L.lipfit_lbfgs(rosen, np.zeros(12), max_iter=1000, tol_grad=1e-9)
    np.testing.assert_allclose(x, 1.0, atol=1e-7)
    assert info["status"] == 0 and info["F"] < 1e-14
    A = np.diag(np.linspace(1, 1000, 50))
    b = np.arange(50.0)
    x, info = L.lipfit_lbfgs(lambda v: (0.5 * v @ A @ v - b @ v, A @ v - b), np.zeros(50), 500, 1e-9)
    np.testing.assert_allclose(x, b / np.diag(A), atol=1e-7)      # |g| <= 1e-9, lambda_min = 1
    # iteration cap is honoured and reported
    x, info = L.lipfit_lbfgs(rosen, np.zeros(12), max_iter=3, tol_grad=1e-12)
    assert info["iters"] == 3 and info["status"] == 1


@pytest.mark.parametrize("norm,mask", [(L2, [1] * 5), (L1, [1, 0, 0, -1, 0]), (LINF, None)])
def test_host_lbfgs_minimises_eq7_to_the_oracle_minimiser(norm, mask):
    """a5 driven by the ORACLE objective on the CPU: same unique minimiser as scipy's (R14)."""
    wl = make_workload(5, N=120)
    p = 1.0
    eps_ref, info_ref = oracle.smooth(wl.X, wl.y, wl.M, mask, norm, None, p)
    fun = lambda e: oracle.smooth_objective(wl.X, wl.y, wl.M, e, mask, norm, None, p)
    x, info = L.lipfit_lbfgs(fun, np.zeros(120), max_iter=2000, tol_grad=1e-10)
    assert info["status"] in (0, 2)
    np.testing.assert_allclose(x, eps_ref, atol=5e-8)
    assert abs(x.sum()) < 1e-8        # P14: sum eps = 0 along LBFGS from eps = 0


def test_world_size_2_gloo_query_sharding():
    """§8(e): the path shards over queries with no data-path collective; the only multi-process logic
    is the partition of Q and the max-over-ranks timing bench.py does.  Exercise both with gloo."""
    import torch.multiprocessing as mp
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_gloo_worker, args=(r, 2, q)) for r in range(2)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    got = sorted(q.get(timeout=5) for _ in range(2))
    assert got[0][0] == 0 and got[1][0] == 1
    # shards tile [0, Q) exactly, and every rank saw the same max time
    assert got[0][1] == 0 and got[0][2] == got[1][1] and got[1][2] == 1001
    assert got[0][3] == got[1][3] == 2.0


def _gloo_worker(rank, world, q):
    import os
    import sys
    sys.path.insert(0, ROOT)
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT="29611", RANK=str(rank),
                      WORLD_SIZE=str(world))
    import torch
    import torch.distributed as dist
    import bench
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = bench.shard_range(1001, rank, world)
    t = bench.max_over_ranks(float(rank + 1), device="cpu")
    q.put((rank, lo, hi, t))
    dist.destroy_process_group()


def test_bench_gpus_n_starts_n_ranks_by_itself():
    """`python bench.py --gpus N` not started by torchrun re-launches itself under torchrun with N ranks on
    127.0.0.1 (the driver's own launch line), passing its arguments through."""
    import bench
    cmd = bench.torchrun_command(8, ["--gpus", "8", "--steps", "3"], 29555)
    assert cmd[1:3] == ["-m", "torch.distributed.run"]
    assert "--nproc-per-node=8" in cmd and "--nnodes=1" in cmd
    assert cmd[cmd.index("--master-addr") + 1] == "127.0.0.1" and cmd[cmd.index("--master-port") + 1] == "29555"
    assert cmd[-4:] == ["--gpus", "8", "--steps", "3"] and cmd[-5].endswith("bench.py")
    assert 1024 <= bench.free_port() <= 65535
