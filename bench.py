#!/usr/bin/env python
"""bench.py -- measures the LipFit hot path on B200 (contract: task prompt, "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--configs 2[,1,3,4,5,6,7,8]]

One "step" = one pass of the hot path over one batch of synthetic input of the bench workload:
BASELINE.json configs[1] (d=4, N=1e5 data, Q=1e6 queries, weighted L1, mask [+1,+1,0,0], M=8) through
`lipfit_bounds` = a1 prepack + a2 fused bounds (+ finalize).  `value` = query x datum pair
evaluations per second (Gpairs/s) with inputs resident in HBM; `e2e` = the same through
`lipfit_bounds_host` (host buffers; H2D and D2H inside the timed region).  The other configs are
reported under "configs" when asked for with --configs.

Multi-GPU (N > 1, launched by torchrun): queries are independent, so every rank runs the same-size
batch of its own (seeded by rank) with NO data-path collective ("weak" scaling); time = max over ranks.

`--impl reference` times the CPU oracle (oracle/, fp64, OpenMP) on a bounded sample of the same
workload on the host cores; only rank 0 works.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from inputs import make_workload, oracle_subset  # noqa: E402

METRIC = "query x datum pair evaluations per second (bounds, config 2)"
UNIT = "Gpairs/s"
# Algorithmic lane-ops per pair: 1 lane-op = one fp32
# add/sub/mul/fma, one min/max/relu/compare, or one sqrt.
# Config 2 (weighted L1, 2 free + 2 constrained coordinates) runs the FOLDED form (bounds.cu FoldL1Core):
# 4 sub + 4 add + 2 relu + 1 sub + min + max = 13 executed lane-ops per pair (SURVEY.md's plain form: 18).
# Config 4 (symmetric L2) selects on the cross-term key ||x||^2 - 2 q.x: 16 FFMA + 1 compare = 17 executed
# lane-ops per pair (the direct-difference form of SURVEY.md is 33).  Smoothing visits each UNORDERED pair
# once with a one-sided distance: 5 sub + 5 relu + 5 fma + dz + dz^2 + compare = 18 executed lane-ops
# per visit (SURVEY.md credits 26 per ORDERED pair).  Rooflines are reported on EXECUTED work.
LANE_OPS = {1: 9, 2: 13, "2survey": 18, 3: 21, 4: 17, "4direct": 33, "5s": 18, "5s_survey": 26, "5b": 31}
# dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the committed
# `ncu --set full` captures (profiles/*.md); null where no capture of this kernel version exists.
NCU_TRAFFIC_BYTES = {"bounds<L1,U2,C2,folded>": 30_431_744, "knn_tc_select": 2_853_554_000, "knn_select<dot>": 5_975_622_000,
                     "smooth_pairs<L2,U0,C5>": 14_425_600}
FP32_LANES_PER_SM = 128


# ------------------------------------------------------------------------------------------------
# helpers shared with the gloo test (tests/test_host_abi.py)
# ------------------------------------------------------------------------------------------------
def shard_range(Q: int, rank: int, world: int):
    """Contiguous slice [lo, hi) of Q units owned by `rank` (strong-scaling helper, §8(e))."""
    base, rem = divmod(Q, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(t: float, device="cuda") -> float:
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return t
    x = torch.tensor([t], dtype=torch.float64, device=device)
    dist.all_reduce(x, op=dist.ReduceOp.MAX)
    return float(x.item())


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except OSError:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100",
                 "-i", str(self.index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc:
            self.proc.terminate()
            try:
                self.proc.wait(2)
            except Exception:
                self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[1]))
                mx.append(float(r[2]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown",
                                "sw_power_cap"), r[4:8]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "reasons": sorted(reasons),
                "samples": len(sm)}


def flush_l2(buf):
    buf.add_(1.0)          # read+write of a buffer larger than the 126 MB L2


# ------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on a bounded sample
# ------------------------------------------------------------------------------------------------
def oracle_sample_rate(wl, budget_s: float = 12.0):
    """Times oracle.bounds on a bounded query sample of `wl`; returns (Gpairs/s, sample text,
    cores, sample indices, oracle outputs)."""
    import oracle
    cores = oracle.num_threads()
    probe = min(wl.Q, max(64, 4 * cores))
    t0 = time.perf_counter()
    oracle.bounds(wl.X, wl.y, wl.Xq[:probe], wl.M, wl.mask, wl.norm, wl.weights)
    dt = max(time.perf_counter() - t0, 1e-6)
    qo = int(min(wl.Q, max(probe, budget_s * probe / dt)))
    sel = oracle_subset(wl.Q, qo)
    xs = np.ascontiguousarray(wl.Xq[sel])
    t0 = time.perf_counter()
    out = oracle.bounds(wl.X, wl.y, xs, wl.M, wl.mask, wl.norm, wl.weights)
    dt = time.perf_counter() - t0
    rate = len(sel) * wl.N / dt / 1e9
    return rate, f"{len(sel)} of {wl.Q} queries (first half + evenly strided) x all {wl.N} data", cores, sel, out


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import oracle
    wl = make_workload(2)
    cores = oracle.num_threads()
    # one "step" = a bounded sample sized for ~6 s of CPU work
    probe = 8 * cores
    t0 = time.perf_counter()
    oracle.bounds(wl.X, wl.y, wl.Xq[:probe], wl.M, wl.mask, wl.norm, wl.weights)
    dt = max(time.perf_counter() - t0, 1e-6)
    per_step = max(1.0, min(6.0, 120.0 / max(1, args.steps + args.warmup)))
    qo = int(min(wl.Q, max(probe, per_step * probe / dt)))
    sel = oracle_subset(wl.Q, qo)
    xs = np.ascontiguousarray(wl.Xq[sel])
    times = []
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        oracle.bounds(wl.X, wl.y, xs, wl.M, wl.mask, wl.norm, wl.weights)
        if i >= args.warmup:
            times.append(time.perf_counter() - t0)
    ms = 1e3 * float(np.mean(times))
    value = len(sel) * wl.N / (ms * 1e-3) / 1e9
    sample = f"{len(sel)} of {wl.Q} queries x all {wl.N} data per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: bounds d=4 N=100000 Q=1000000 L1 mask[+1,+1,0,0] M=8",
                   "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
def _time_steps(torch, fn, steps, warmup, l2buf):
    """W untimed steps, then K steps each bracketed by CUDA events on the launching (current)
    stream, L2 flushed between steps.  Returns per-step milliseconds."""
    for _ in range(warmup):
        fn()
    torch.cuda.synchronize()
    out = []
    for _ in range(steps):
        flush_l2(l2buf)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn()
        e1.record()
        e1.synchronize()
        out.append(e0.elapsed_time(e1))
    return out


def _kernel_ms(L, which, fn, reps):
    """Average device time of dominant kernel `which` alone (library-side CUDA events)."""
    L.set_timing(True)
    try:
        for _ in range(reps):
            fn()
        ms, n = L.get_timing(which)
    finally:
        L.set_timing(False)
    return (ms / n if n else None), n


def _roofline(pairs, lane_ops, kernel_ms, sms, peaks, kernel=None):
    peak = sms * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12    # T lane-ops/s
    ach = pairs * lane_ops / (kernel_ms * 1e-3) / 1e12 if kernel_ms else None
    return {"bound": "alu", "achieved": ach, "peak": peak, "unit": "Tlane-op/s",
            "frac": (ach / peak) if ach else None, "traffic": NCU_TRAFFIC_BYTES.get(kernel),
            "lane_ops_per_pair": lane_ops, "kernel_ms": kernel_ms,
            "peak_how": f"{sms} SMs x {FP32_LANES_PER_SM} fp32 lanes x {peaks['sm_max_mhz']:.0f} MHz (clocks.max.sm)"}


def bench_bounds(torch, L, wl, steps, warmup, l2buf, dev, lane_ops, do_e2e=True):
    t = lambda a: torch.from_numpy(a).to(dev)
    X, y, Xq = t(wl.X), t(wl.y), t(wl.Xq)
    fn = lambda: L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
    n0 = L.launch_count()
    ms = _time_steps(torch, fn, steps, warmup, l2buf)
    launches = (L.launch_count() - n0) * steps // (steps + warmup)
    kms, _ = _kernel_ms(L, 0, fn, max(1, min(3, steps)))
    pairs = wl.N * wl.Q
    res = {"ms_per_step": float(np.mean(ms)), "ms_min": float(np.min(ms)), "pairs": pairs,
           "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "gpu_launches": int(launches),
           "kernel": L.bounds_variant(wl.d, wl.mask, wl.norm), "kernel_ms": kms,
           "lane_ops": lane_ops, "outputs": fn()}
    if do_e2e:
        pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
        Xh, yh, Xqh = pin(wl.X), pin(wl.y), pin(wl.Xq)
        outs = tuple(torch.empty(wl.Q, dtype=torch.float32).pin_memory().numpy() for _ in range(3))
        sp = torch.cuda.current_stream().cuda_stream
        hfn = lambda: L.lipfit_bounds_host(Xh, yh, Xqh, wl.M, wl.mask, wl.norm, wl.weights, outs, sp)
        hms = _time_steps(torch, hfn, max(1, steps), warmup, l2buf)
        res["e2e"] = {"value": pairs / (np.mean(hms) * 1e-3) / 1e9, "unit": UNIT,
                      "ms_per_step": float(np.mean(hms)),
                      "h2d_bytes_per_step": int(Xh.nbytes + yh.nbytes + Xqh.nbytes),
                      "d2h_bytes_per_step": int(sum(o.nbytes for o in outs))}
    return res


def bench_knn(torch, L, wl, steps, warmup, l2buf, dev, tensor_cores=True):
    t = lambda a: torch.from_numpy(a).to(dev)
    X, Xq = t(wl.X), t(wl.Xq)
    fn = lambda: L.lipfit_knn(X, Xq, wl.k, None, 0, wl.norm, wl.weights)
    L.knn_set_tensor_cores(tensor_cores)
    try:
        variant = L.knn_variant(wl.d, 0, wl.norm)
        ms = _time_steps(torch, fn, steps, warmup, l2buf)
        kms, _ = _kernel_ms(L, 1, fn, 1)
        out = fn()
        torch.cuda.synchronize()
        res = {"fallbacks": L.knn_fallbacks(), "key_error_over_bound": L.knn_key_error_ratio()}
    finally:
        L.knn_set_tensor_cores(True)
    pairs = wl.N * wl.Q
    res.update({"ms_per_step": float(np.mean(ms)), "pairs": pairs, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                "kernel_ms": kms, "kernel": variant, "outputs": out})
    return res


def _roofline_tensor(pairs, k_dim, kernel_ms, peaks):
    """bf16 GEMM roofline of the tensor-core selection: 2 * K flop per pair (K = 64 operand columns)."""
    peak = peaks.get("bf16_tflops", 1590.0)
    ach = pairs * 2.0 * k_dim / (kernel_ms * 1e-3) / 1e12 if kernel_ms else None
    return {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
            "frac": (ach / peak) if ach else None, "traffic": NCU_TRAFFIC_BYTES.get("knn_tc_select"),
            "flop_per_pair": 2 * k_dim, "kernel_ms": kernel_ms,
            "peak_how": "MEASURED_PEAKS.json bf16_tflops (cuBLAS bf16, burst; the kernel is timed alone)"}


def bench_smooth(torch, L, wl, l2buf, dev):
    """Config 5: host LBFGS (<= 200 iterations) over the device all-pairs pass, then bounds."""
    t = lambda a: torch.from_numpy(a).to(dev)
    X, y = t(wl.X), t(wl.y.copy())
    L.set_timing(True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    eps, info = L.lipfit_smooth(X, y, wl.M, wl.mask, wl.norm, wl.weights, wl.p, wl.max_iter, 1e-6)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    kms, n = L.get_timing(2)
    L.set_timing(False)
    pairs_eval = wl.N * (wl.N - 1)          # ordered pairs of Eq.(7) covered by one evaluation
    return {"wall_s": wall, "info": info, "evals": n, "kernel_ms_per_eval": kms / max(n, 1),
            "pairs_per_eval": pairs_eval, "visits_per_eval": pairs_eval // 2,
            "value": pairs_eval / (kms / max(n, 1) * 1e-3) / 1e9,
            "lane_ops": LANE_OPS["5s"], "z": y, "X": X}


def bench_local(torch, L, l2buf, dev, sms, peaks, args):
    """NEXT-1 (local Lipschitz interpolation) on config 5's data: knots from 1e6 sampled
    pairs, step tables for N = 2e5 (4e10 ordered pairs), evaluation at Q = 1e6 (2e11 pairs)."""
    import oracle
    from inputs import sample_pairs
    wl = make_workload(5)
    t = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    X, y, Xq = t(wl.X), t(wl.y), t(wl.Xq)
    pi, pk = sample_pairs(3, wl.N, 1_000_000)
    pi_d, pk_d = t(pi), t(pk)
    knots = L.lipfit_distance_quantiles(X, pi_d, pk_d, L.LIPFIT_LOCAL_KNOTS, wl.norm)
    f_tab = lambda: L.lipfit_local_lipschitz(X, y, knots, wl.norm)
    ms_tab = _time_steps(torch, f_tab, max(1, min(args.steps, 3)), 3, l2buf)
    k_tab, _ = _kernel_ms(L, 4, f_tab, 1)
    table = f_tab()
    f_ev = lambda: L.lipfit_values_local(X, y, Xq, knots, table, wl.norm)
    ms_ev = _time_steps(torch, f_ev, max(1, min(args.steps, 3)), 3, l2buf)
    k_ev, _ = _kernel_ms(L, 5, f_ev, 1)
    # executed lane-ops per pair (d = 5 padded to 8 coordinates, J = 16 knots):
    #   table: 8 sub + 8 fma + |dy| 2 + two-level knot search (6 compares + 5 adds) + MUFU sqrt + 2 mul + raise test
    #          + nearest-neighbour test 3 ~ 36 on the fast path (IEEE sqrt / divide only for pairs that raise a bin)
    #   eval : 8 sub + 8 fma + knot search 11 + MUFU sqrt + guard 2 + mul + add + sub + min + max + index math ~ 39
    #          (counted in the SASS of local_eval_kernel<2,8,4>: 157 arithmetic instructions per record of 4 pairs)
    out = {"workload": "config 5 data (d=5, N=200000), Q=1000000, L2, J=16 knots from 1e6 sampled pairs",
           "table": {"ms_per_step": float(np.mean(ms_tab)), "kernel_ms": k_tab,
                     "value": wl.N * (wl.N - 1) / (np.mean(ms_tab) * 1e-3) / 1e9, "unit": "G ordered pairs/s",
                     "roofline": _roofline(wl.N * wl.N, 36, k_tab, sms, peaks)},
           "evaluate": {"ms_per_step": float(np.mean(ms_ev)), "kernel_ms": k_ev,
                        "value": wl.N * wl.Q / (np.mean(ms_ev) * 1e-3) / 1e9, "unit": UNIT,
                        "roofline": _roofline(wl.N * wl.Q, 39, k_ev, sms, peaks)}}
    if not args.no_cpu:
        sel = oracle_subset(wl.Q, 400)
        rows = oracle_subset(wl.N, 64)
        tb = table.cpu().numpy()
        up, lo, g = (v.cpu().numpy() for v in f_ev())
        U, Lo, G = oracle.values_local(wl.X, wl.y, wl.Xq[sel], knots.astype(np.float64), tb.astype(np.float64), wl.norm)
        tol = 1e-5 * wl.y_range
        frac_ok = float(np.mean((np.abs(up[sel] - U) <= tol) & (np.abs(lo[sel] - Lo) <= tol)))
        out["evaluate"]["parity"] = {"queries": int(len(sel)), "fraction_within_tol": frac_ok, "tol": tol,
                                     "note": "queries off a knot boundary must match; tests/test_gpu_local.py sandwiches the rest"}
    return out


def parity_bounds(wl, outs, sel, ref):
    """max |gpu - oracle| / (1e-5 * range) on the oracle's query sample (<= 1 passes)."""
    tol = 1e-5 * wl.y_range
    worst = 0.0
    for o, r in zip(outs, ref):
        worst = max(worst, float(np.abs(o.cpu().numpy()[sel].astype(np.float64) - r).max()))
    return {"max_abs_err": worst, "tol": tol, "ok": bool(worst <= tol), "queries": int(len(sel))}


def run_gpu(args):
    import torch
    import torch.distributed as dist
    import paper_2606_04670_b200 as L
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    L.load()
    peaks, peaks_how = measured_peaks()
    sms = torch.cuda.get_device_properties(dev).multi_processor_count
    l2buf = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device=dev)   # 256 MB > 126 MB L2
    cfgs = [int(c) for c in args.configs.split(",")]

    # ---- the bench line: config 2 ----
    wl = make_workload(2, query_seed=1 + 1000 * rank)   # weak scaling: each rank its own batch
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    r2 = bench_bounds(torch, L, wl, args.steps, args.warmup, l2buf, dev, LANE_OPS[2])
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(r2["ms_per_step"])
    e2e_ms = max_over_ranks(r2["e2e"]["ms_per_step"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    line = {
        "metric": METRIC, "value": world * r2["pairs"] / (ms * 1e-3) / 1e9, "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": "BASELINE.json configs[1]: bounds d=4 N=100000 Q=1000000 L1 mask[+1,+1,0,0] M=8",
                   "kernel": r2["kernel"], "l2": "flushed between timed steps (256 MB write)",
                   "step": "lipfit_bounds = a1 prepack + a2 fused bounds + finalize",
                   "parallelism": f"query-sharded replicas x{world}, no collective"},
        "clocks": clocks,
        "e2e": {"value": world * r2["pairs"] / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": r2["e2e"]["h2d_bytes_per_step"],
                "d2h_bytes_per_step": r2["e2e"]["d2h_bytes_per_step"], "ms_per_step": e2e_ms},
        "gpu_launches": r2["gpu_launches"],
        "roofline": _roofline(r2["pairs"], LANE_OPS[2], r2["kernel_ms"], sms, peaks, r2["kernel"]),
        "peaks": peaks_how,
    }
    line["roofline"]["frac_survey_18ops"] = (
        r2["pairs"] * LANE_OPS["2survey"] / (r2["kernel_ms"] * 1e-3) / 1e12 / line["roofline"]["peak"])
    if clocks and clocks.get("sm_mhz"):
        rf = line["roofline"]
        rf["frac_at_observed_clock"] = rf["achieved"] / (sms * FP32_LANES_PER_SM * clocks["sm_mhz"] * 1e6 / 1e12)
    # ---- CPU baseline: the oracle on a bounded sample, with parity on exactly that sample ----
    if not args.no_cpu:
        rate, sample, cores, sel, ref = oracle_sample_rate(wl)
        line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        line["parity"] = parity_bounds(wl, r2["outputs"], sel, ref)
    # ---- the other configs on request ----
    extra = {}
    for c in cfgs:
        if c == 2:
            continue
        try:
            extra[f"config{c}"] = run_other_config(torch, L, c, args, l2buf, dev, sms, peaks)
        except Exception as e:  # report, do not hide
            extra[f"config{c}"] = {"error": repr(e)}
    if extra:
        line["configs"] = extra
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_other_config(torch, L, c, args, l2buf, dev, sms, peaks):
    import oracle
    wl = make_workload({6: 5, 7: 2, 8: 5, 9: 2, 10: 3, 11: 5, 12: 5}.get(c, c))
    steps = max(1, min(args.steps, 3)) if c in (3, 4) else args.steps
    out = {}
    if c in (1, 3):
        r = bench_bounds(torch, L, wl, steps, 3, l2buf, dev, LANE_OPS[c], do_e2e=False)
        out.update({k: r[k] for k in ("ms_per_step", "ms_min", "value", "kernel", "kernel_ms")})
        out["unit"] = UNIT
        out["roofline"] = _roofline(r["pairs"], LANE_OPS[c], r["kernel_ms"], sms, peaks)
        if c == 1:
            # latency-bound config: an isolated, L2-flushed step exposes the host launch latency; also report the
            # steady state of back-to-back calls (inputs stay in L2; 200 calls between two events)
            t = lambda a: torch.from_numpy(a).to(dev)
            X, y, Xq = t(wl.X), t(wl.y), t(wl.Xq)
            for _ in range(20):
                L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(200):
                L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
            e1.record()
            e1.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / 200
            out["back_to_back"] = {"us_per_step": us, "value": r["pairs"] / (us * 1e-6) / 1e9, "unit": UNIT,
                                   "note": "200 consecutive lipfit_bounds calls, no L2 flush"}
        if not args.no_cpu:
            rate, sample, cores, sel, ref = oracle_sample_rate(wl, 8.0)
            out["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "sample": sample}
            out["parity"] = parity_bounds(wl, r["outputs"], sel, ref)
    elif c == 4:
        r = bench_knn(torch, L, wl, steps, max(3, args.warmup), l2buf, dev, tensor_cores=True)
        out.update({k: r[k] for k in ("ms_per_step", "value", "kernel_ms", "kernel")})
        out["unit"] = UNIT
        out["step"] = "lipfit_knn = operand images + tensor-core selection + fp64 re-rank / certificate + exact fallback"
        out["exact_fallback_queries"] = r["fallbacks"]
        out["key_error_over_bound"] = r["key_error_over_bound"]
        out["roofline"] = _roofline_tensor(r["pairs"], 16 * ((3 * wl.d + 3 + 15) // 16), r["kernel_ms"], peaks)
        # the CUDA-core selection kernel (tensor cores switched off), same outputs
        rc = bench_knn(torch, L, wl, max(1, min(steps, 2)), max(3, args.warmup), l2buf, dev, tensor_cores=False)
        out["cuda_core_selection"] = {k: rc[k] for k in ("ms_per_step", "value", "kernel_ms", "kernel")}
        out["cuda_core_selection"]["roofline"] = _roofline(rc["pairs"], LANE_OPS[4], rc["kernel_ms"], sms, peaks)
        out["cuda_core_selection"]["roofline"]["frac_direct_difference_form_33ops"] = (
            rc["pairs"] * LANE_OPS["4direct"] / (rc["kernel_ms"] * 1e-3) / 1e12
            / out["cuda_core_selection"]["roofline"]["peak"])
        out["cuda_core_selection"]["same_outputs"] = bool(
            torch.equal(r["outputs"][0], rc["outputs"][0]) and torch.equal(r["outputs"][1], rc["outputs"][1]))
        if not args.no_cpu:
            sel = oracle_subset(wl.Q, 64)
            t0 = time.perf_counter()
            oi, od = oracle.knn(wl.X, wl.Xq[sel], wl.k, None, 0, wl.norm)
            dt = time.perf_counter() - t0
            gi = r["outputs"][0].cpu().numpy()[sel]
            gd = r["outputs"][1].cpu().numpy()[sel]
            out["cpu_baseline"] = {"value": len(sel) * wl.N / dt / 1e9, "unit": UNIT,
                                   "cores": oracle.num_threads(), "sample": f"{len(sel)} queries x all data"}
            out["parity"] = {"index_sets_equal": bool(all(set(a) == set(b) for a, b in zip(gi, oi))),
                             "max_dist_err_ulps": float(np.max(np.abs(gd - od.astype(np.float32))
                                                               / np.spacing(od.astype(np.float32)))),
                             "queries": int(len(sel))}
    elif c == 6:
        out.update(bench_local(torch, L, l2buf, dev, sms, peaks, args))
    elif c == 7:
        # NEXT-2: weighted sums of the k = 4 best bound values on the config 2 workload
        wk = np.array([0.4, 0.3, 0.2, 0.1], dtype=np.float32)
        t = lambda a: torch.from_numpy(a).to(dev)
        X, y, Xq = t(wl.X), t(wl.y), t(wl.Xq)
        fn = lambda: L.lipfit_bounds_topk(X, y, Xq, wl.M, wk, wl.mask, wl.norm, wl.weights)
        ms = _time_steps(torch, fn, steps, 3, l2buf)
        pairs = wl.N * wl.Q
        out.update({"workload": "config 2 data and queries, k = 4 best bounds with weights [0.4, 0.3, 0.2, 0.1]",
                    "ms_per_step": float(np.mean(ms)), "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "unit": UNIT,
                    "kernel": "bounds_topk<L1,DP4> (generic distance, 2 x 8 sorted lists in registers)"})
        if not args.no_cpu:
            sel = oracle_subset(wl.Q, 2000)
            ref = oracle.bounds_topk(wl.X, wl.y, wl.Xq[sel], wl.M, wk, wl.mask, wl.norm, wl.weights)
            out["parity"] = parity_bounds(wl, fn(), sel, ref)
    elif c in (9, 10, 11):
        # NEXT-4(ii): bounds with EXACT spatial pruning on the config 2 / 3 / 5 workloads.  "Effective" pairs/s =
        # Q N / step time (the work the unpruned path would do), reported beside the pairs actually evaluated;
        # never mixed into the brute-force roofline numbers above.
        t = lambda a: torch.from_numpy(a).to(dev)
        X, y, Xq = t(wl.X), t(wl.y), t(wl.Xq)
        fn = lambda: L.lipfit_bounds_pruned(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
        steps_p = max(1, min(args.steps, 3)) if c == 10 else args.steps
        ms = _time_steps(torch, fn, steps_p, 3, l2buf)
        kms, _ = _kernel_ms(L, 6, fn, 1)
        *outs, evaluated = L.lipfit_bounds_pruned(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights, count_pairs=True)
        pairs = wl.N * wl.Q
        fb = lambda: L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
        ms_b = _time_steps(torch, fb, 1 if c == 10 else 2, 1, l2buf)
        ub = fb()
        d_async = max(float((a - b).abs().max()) for a, b in zip(outs, ub))
        torch.cuda.synchronize()
        d_sync = max(float((a - b).abs().max()) for a, b in zip(outs, ub))
        if d_async != d_sync:
            print(f"bench.py: config {c}: unpruned outputs changed after a synchronize ({d_async} -> {d_sync})",
                  file=sys.stderr)
        out.update({"workload": "config %d data and queries" % {9: 2, 10: 3, 11: 5}[c],
                    "ms_per_step": float(np.mean(ms)), "kernel_ms": kms,
                    "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "unit": "effective " + UNIT,
                    "pairs_evaluated": int(evaluated), "fraction_evaluated": evaluated / pairs,
                    "evaluated_rate_gpairs_s": evaluated / (kms * 1e-3) / 1e9,
                    "unpruned_ms_per_step": float(np.mean(ms_b)),
                    "speedup_over_unpruned": float(np.mean(ms_b) / np.mean(ms)),
                    "max_abs_diff_vs_unpruned": d_sync,
                    "kernel": "bounds_pruned<norm,DP> (Morton-sorted 32-datum tiles, box tests, generic distance)"})
        if not args.no_cpu:
            sel = oracle_subset(wl.Q, 2000 if c != 10 else 96)
            ref = oracle.bounds(wl.X, wl.y, wl.Xq[sel], wl.M, wl.mask, wl.norm, wl.weights)
            out["parity"] = parity_bounds(wl, outs, sel, ref)
    elif c == 12:
        # Eq.(7) objective / gradient of config 5 with exact pruning (the exact counterpart of the M/3 heuristic,
        # PAPER.md:214-218), beside the unpruned all-pairs pass, at eps = 0 and at a random eps (sigma 0.05)
        t = lambda a: torch.from_numpy(a).to(dev)
        X, y = t(wl.X), t(wl.y)
        eps = t((0.05 * np.random.default_rng(7).standard_normal(wl.N)).astype(np.float32))
        pairs = wl.N * (wl.N - 1)
        out.update({"workload": "config 5 data (d=5, N=200000, L2, all coordinates monotone, M=3, p=1)",
                    "unit": "effective G ordered pairs of Eq.(7) per second"})
        for name, e in (("eps0", None), ("eps_random", eps)):
            fn = lambda: L.lipfit_smooth_objective_pruned(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p)
            fu = lambda: L.lipfit_smooth_objective(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p)
            ms = _time_steps(torch, fn, args.steps, 3, l2buf)
            kms, _ = _kernel_ms(L, 7, fn, 1)
            ms_u = _time_steps(torch, fu, 2, 1, l2buf)
            F, g, evaluated = L.lipfit_smooth_objective_pruned(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p,
                                                               count_pairs=True)
            Fu, gu = fu()
            torch.cuda.synchronize()
            out[name] = {"ms_per_step": float(np.mean(ms)), "kernel_ms": kms,
                         "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                         "pairs_evaluated": int(evaluated), "fraction_evaluated": evaluated / pairs,
                         "unpruned_ms_per_step": float(np.mean(ms_u)),
                         "speedup_over_unpruned": float(np.mean(ms_u) / np.mean(ms)),
                         "F": F, "F_rel_diff_vs_unpruned": abs(F - Fu) / Fu,
                         "grad_rel_diff_vs_unpruned": float((g - gu).abs().max() / gu.abs().max())}
        out["value"] = out["eps0"]["value"]
        out["ms_per_step"] = out["eps0"]["ms_per_step"]
        # the same data without the monotone mask (symmetric distance): only near pairs can violate
        fs = lambda: L.lipfit_smooth_objective_pruned(X, y, wl.M, None, None, wl.norm, None, wl.p)
        fsu = lambda: L.lipfit_smooth_objective(X, y, wl.M, None, None, wl.norm, None, wl.p)
        ms = _time_steps(torch, fs, args.steps, 3, l2buf)
        ms_u = _time_steps(torch, fsu, 2, 1, l2buf)
        Fs, gs, ev = L.lipfit_smooth_objective_pruned(X, y, wl.M, None, None, wl.norm, None, wl.p, count_pairs=True)
        Fsu, gsu = fsu()
        torch.cuda.synchronize()
        out["eps0_no_mask"] = {"ms_per_step": float(np.mean(ms)), "unpruned_ms_per_step": float(np.mean(ms_u)),
                               "speedup_over_unpruned": float(np.mean(ms_u) / np.mean(ms)),
                               "fraction_evaluated": ev / pairs, "F_rel_diff_vs_unpruned": abs(Fs - Fsu) / Fsu,
                               "grad_rel_diff_vs_unpruned": float((gs - gsu).abs().max() / gsu.abs().max())}
        # lipfit_smooth on the same data without a mask runs the pruned pass (N >= 8192, no constrained coordinate)
        ys = y.clone()
        t0 = time.perf_counter()
        _, info_s = L.lipfit_smooth(X, ys, wl.M, None, wl.norm, None, wl.p, wl.max_iter, 1e-6)
        torch.cuda.synchronize()
        out["smooth_no_mask"] = {"wall_s": time.perf_counter() - t0, "info": info_s,
                                 "ms_per_evaluation_incl_host": 1e3 * (time.perf_counter() - t0) / max(info_s["evals"], 1)}
        if not args.no_cpu:
            rows = oracle_subset(wl.N, 64)
            g_ref, _ = oracle.smooth_rows(wl.X, wl.y, wl.M, np.zeros(wl.N), rows, wl.mask, wl.norm, None, wl.p)
            _, g0 = L.lipfit_smooth_objective_pruned(X, y, wl.M, None, wl.mask, wl.norm, None, wl.p)
            err = float(np.abs(g0.cpu().numpy()[rows] - g_ref).max() / np.abs(g_ref).max())
            out["parity"] = {"gradient_rows": int(len(rows)), "max_rel_err": err, "tol": 1e-5, "ok": bool(err <= 1e-5)}
    elif c == 8:
        # NEXT-3: smallest consistent Lipschitz constant of the config 5 data
        t = lambda a: torch.from_numpy(a).to(dev)
        X, y = t(wl.X), t(wl.y)
        # (symmetric distance: under the config's monotone mask the noisy data violate monotonicity, L = +inf)
        fn = lambda: L.lipfit_lipschitz_constant(X, y, None, wl.norm, wl.weights)
        ms = _time_steps(torch, fn, steps, 3, l2buf)
        kms, _ = _kernel_ms(L, 3, fn, 1)
        pairs = wl.N * (wl.N - 1)
        out.update({"workload": "config 5 data (d=5, N=200000, L2), symmetric distance",
                    "ms_per_step": float(np.mean(ms)), "kernel_ms": kms, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                    "unit": "G ordered pairs/s (each unordered pair is visited once)",
                    "L": float(fn().cpu().numpy()[0]),
                    # fast path per visited unordered pair (source count, d = 5 symmetric L2): 5 sub + 5 fma + dy +
                    # |dy| + 2 mul + 1 compare of dy^2 against L^2 D^2 + loop share ~ 16; survivors take the fp64 ratio
                    "roofline": _roofline(pairs // 2, 16, kms, sms, peaks)})
        if not args.no_cpu:
            # the oracle is O(N^2) on the host: compare on the first 20000 data (4e8 ordered pairs)
            n = 20000
            ref = oracle.lipschitz_constant(wl.X[:n], wl.y[:n], None, wl.norm, wl.weights)
            got = float(L.lipfit_lipschitz_constant(t(wl.X[:n]), t(wl.y[:n]), None, wl.norm, wl.weights).cpu().numpy()[0])
            out["parity"] = {"data": n, "oracle": ref, "gpu": got, "ok": bool(got == float(np.float32(ref)))}
    elif c == 5:
        r = bench_smooth(torch, L, wl, l2buf, dev)
        out.update({"smooth_wall_s": r["wall_s"], "info": r["info"], "evals": r["evals"],
                    "kernel_ms_per_eval": r["kernel_ms_per_eval"], "value": r["value"],
                    "unit": "G ordered pairs of Eq.(7) per second (each unordered pair is visited once)",
                    "roofline": _roofline(r["visits_per_eval"], LANE_OPS["5s"], r["kernel_ms_per_eval"], sms, peaks)})
        out["roofline"]["frac_survey_26ops_per_ordered_pair"] = (
            r["pairs_per_eval"] * LANE_OPS["5s_survey"] / (r["kernel_ms_per_eval"] * 1e-3) / 1e12
            / out["roofline"]["peak"])
        Xq = torch.from_numpy(wl.Xq).to(dev)
        fn = lambda: L.lipfit_bounds(r["X"], r["z"], Xq, wl.M, wl.mask, wl.norm, wl.weights)
        ms = _time_steps(torch, fn, max(1, min(args.steps, 3)), 2, l2buf)
        kms, _ = _kernel_ms(L, 0, fn, 1)
        pairs = wl.N * wl.Q
        out["bounds_after"] = {"ms_per_step": float(np.mean(ms)), "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                               "roofline": _roofline(pairs, LANE_OPS["5b"], kms, sms, peaks)}
        if not args.no_cpu:
            z = r["z"].cpu().numpy()
            sel = oracle_subset(wl.Q, 2000)
            ref = oracle.bounds(wl.X, z, wl.Xq[sel], wl.M, wl.mask, wl.norm, wl.weights)
            wl.y = z
            out["bounds_after"]["parity"] = parity_bounds(wl, fn(), sel, ref)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--configs", default="2",
                    help="comma list of BASELINE.json configs to report (2 always); 6 = local Lipschitz (NEXT-1), "
                         "7 = top-k bounds (NEXT-2), 8 = Lipschitz constant (NEXT-3), 9 / 10 / 11 = exactly pruned bounds on the "
                         "config 2 / 3 / 5 workloads, 12 = exactly pruned smoothing objective (NEXT-4(ii))")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline / parity leg")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
