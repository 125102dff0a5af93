#!/usr/bin/env python
"""bench.py -- measures the LipFit hot path on B200 (contract: task prompt, "Measurement").

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--configs all|LIST] [--no-cpu]

One "step" = one pass of the hot path over one batch of synthetic input of the bench workload:
BASELINE.json configs[1] (d=4, N=1e5 data, Q=1e6 queries, weighted L1, mask [+1,+1,0,0], M=8) through
`lipfit_bounds_ex(LIPFIT_BOUNDS_BRUTE)` = a1 prepack + a2 fused all-pairs bounds (+ finalize): every one of the
Q N pairs is evaluated, which is what BASELINE.json's metric (pair evaluations per second, % of the FP32
CUDA-core peak) counts.  `value` = pairs/s with inputs resident in HBM; `e2e` = the same through
`lipfit_bounds_host_ex` (host buffers; H2D and D2H inside the timed region).  What the plain entry point
`lipfit_bounds` does on this workload (LIPFIT_BOUNDS_AUTO -> exact pruning, the same upper/lower/g from a
fraction of the pairs) is printed BESIDE it under "effective", never mixed into `value`.

With no --configs flag (N = 1) the line also carries, under "configs", the other BASELINE.json configs
(1, 3, 4, 5: smoothing + bounds after) and the NEXT rows (6 local Lipschitz, 7 top-k bounds, 8 Lipschitz
constant, 9/10/11 exactly pruned bounds on the config 2/3/5 workloads, 12 exactly pruned smoothing pass,
13 region monotonicity, 14 off-table shapes: even-rounded and generic kernels), each with ms_per_step, value,
roofline (kernel time from CUDA events), cpu_baseline (cores, sample, compiler flags) and a pass/fail parity
on exactly the oracle's sample.  Config 3 is the LARGEST workload (1e12 pairs); config 2 stays the top-level
line because it is the full-size BASELINE config the metric is quoted on.

Multi-GPU: `--gpus N` (N > 1) re-launches itself under torchrun when it was not started by it; queries are
independent, so every rank runs the same-size batch of its own (seeded by rank) with NO data-path collective
("weak" scaling); time = max over ranks.  Only the main line is measured at N > 1.

`--impl reference` times the CPU oracle (oracle/, fp64, OpenMP) on a bounded sample of the same workload on
the host cores; only rank 0 works.
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import socket
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from inputs import make_workload, oracle_subset, random_problem, sample_pairs  # noqa: E402

METRIC = "query x datum pair evaluations per second (bounds, config 2)"
UNIT = "Gpairs/s"
WORKLOAD = ("BASELINE.json configs[1]: bounds d=4 N=100000 Q=1000000 L1 mask[+1,+1,0,0] M=8 (every pair evaluated); "
            "configs[2] (1e12 pairs) is the largest workload and is reported under configs.config3")
# Algorithmic lane-ops per unit (1 lane-op = one fp32 add/sub/mul/fma, one min/max/relu/compare,
# or one sqrt; FMA counts once) and the lane-ops the kernels actually execute:
#   config 2: folded L1 form, 11 executed;  config 4: cross-term key 17 on the CUDA cores (direct-difference
#   form 33);  smoothing: 18 per VISITED unordered pair = 9 per ordered pair (SURVEY credits 26 per ordered
#   pair);  config 3: 20 (the chain of maxima over the 7 unconstrained coordinates starts from |delta_0|);  the
#   others execute the survey's plain form.
SURVEY_OPS = {1: 9, 2: 18, 3: 21, 4: 33, "5s": 26, "5b": 31}
EXECUTED_OPS = {1: 9, 2: 11, 3: 20, 4: 17, "5s": 9, "5b": 31}
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


def torchrun_command(gpus: int, argv, port: int):
    """The command `bench.py --gpus N` re-executes itself with when it was not started by torchrun."""
    return [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={gpus}",
            "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__), *argv]


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured (MEASURED_PEAKS.json)"
    except OSError:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0, "bf16_tflops": 1590.0}, "fallback (B200_PROFILING.md)"


def ncu_table():
    """Per-kernel ncu counters of the committed captures (profiles/r2_ncu_kernels.csv): kernel key ->
    {issue_active, pipe_fma, pipe_alu, sm_throughput (all % of peak), dram_bytes}.  Values are COPIES of
    captured numbers, valid while profiles/ holds the capture of the same kernel version."""
    out = {}
    try:
        with open(os.path.join(ROOT, "profiles", "r2_ncu_kernels.csv")) as f:
            for row in csv.DictReader(l for l in f if not l.startswith("#")):
                key = row.pop("kernel")
                out[key] = {k: (float(v) if v not in ("", "null") else None) for k, v in row.items()}
    except OSError:
        pass
    return out


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


def oracle_flags():
    from oracle import build as obuild
    return "gcc " + " ".join(obuild.FLAGS)


# ------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on a bounded sample
# ------------------------------------------------------------------------------------------------
def oracle_sample_rate(wl, budget_s: float = 8.0, fn=None):
    """Times the oracle (default oracle.bounds) on a bounded query sample of `wl`; returns
    (cpu_baseline dict, sample indices, oracle outputs)."""
    import oracle
    fn = fn or (lambda xs: oracle.bounds(wl.X, wl.y, xs, wl.M, wl.mask, wl.norm, wl.weights))
    cores = oracle.num_threads()
    probe = min(wl.Q, max(64, 4 * cores))
    t0 = time.perf_counter()
    fn(np.ascontiguousarray(wl.Xq[:probe]))
    dt = max(time.perf_counter() - t0, 1e-6)
    qo = int(min(wl.Q, max(probe, budget_s * probe / dt)))
    sel = oracle_subset(wl.Q, qo)
    xs = np.ascontiguousarray(wl.Xq[sel])
    t0 = time.perf_counter()
    out = fn(xs)
    dt = time.perf_counter() - t0
    base = {"value": len(sel) * wl.N / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "sample": f"{len(sel)} of {wl.Q} queries (first half + evenly strided) x all {wl.N} data",
            "flags": oracle_flags(), "seconds": dt}
    return base, sel, out


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
        "config": {"workload": WORKLOAD, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                         "flags": oracle_flags()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------
# GPU arm
# ------------------------------------------------------------------------------------------------
class Bench:
    def __init__(self, torch, L, dev, args, sms, peaks, peaks_how):
        self.torch, self.L, self.dev, self.args = torch, L, dev, args
        self.sms, self.peaks, self.peaks_how = sms, peaks, peaks_how
        self.l2buf = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device=dev)   # 256 MB > 126 MB L2
        self.ncu = ncu_table()
        self.alu_peak = sms * FP32_LANES_PER_SM * peaks["sm_max_mhz"] * 1e6 / 1e12      # T lane-ops/s

    def t(self, a):
        return self.torch.from_numpy(np.ascontiguousarray(a)).to(self.dev)

    def time_steps(self, fn, steps, warmup):
        """W untimed steps, then K steps each bracketed by CUDA events on the launching (current)
        stream, L2 flushed between steps.  Returns per-step milliseconds."""
        torch = self.torch
        for _ in range(warmup):
            fn()
        torch.cuda.synchronize()
        out = []
        for _ in range(steps):
            flush_l2(self.l2buf)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            fn()
            e1.record()
            e1.synchronize()
            out.append(e0.elapsed_time(e1))
        return out

    def kernel_ms(self, which, fn, reps=1):
        """Average device time of dominant kernel `which` alone (library-side CUDA events on its stream)."""
        L = self.L
        L.set_timing(True)
        try:
            for _ in range(reps):
                fn()
            ms, n = L.get_timing(which)
        finally:
            L.set_timing(False)
        return (ms / n if n else None), n

    def roofline(self, units, ops_survey, ops_executed, kernel_ms, kernel=None, unit_name="pair"):
        """"alu" roofline: achieved = units x SURVEY.md §8(d) lane-ops / kernel time; peak = SMs x 128 fp32
        lanes x clocks.max.sm.  `frac` is that algorithmic fraction (it may exceed the pipe
        utilisation and even 1: FADD2 / FMNMX3 retire two lane-ops per issue slot, the ALU pipe runs beside the
        FMA pipe, and folded forms execute fewer ops than the plain formulation credits); `frac_executed`
        counts the lane-ops the kernel really executes; `ncu` = issue / pipe percentages of the committed
        capture of this kernel version (profiles/), the honest utilisation."""
        ach = units * ops_survey / (kernel_ms * 1e-3) / 1e12 if kernel_ms else None
        ex = units * ops_executed / (kernel_ms * 1e-3) / 1e12 if kernel_ms and ops_executed else None
        n = self.ncu.get(kernel or "", {})
        return {"bound": "alu", "achieved": ach, "peak": self.alu_peak, "unit": "Tlane-op/s",
                "frac": (ach / self.alu_peak) if ach else None,
                "frac_executed": (ex / self.alu_peak) if ex else None,
                "traffic": n.get("dram_bytes"),
                "lane_ops_per_%s" % unit_name: ops_survey, "lane_ops_executed_per_%s" % unit_name: ops_executed,
                "kernel_ms": kernel_ms, "kernel": kernel,
                "ncu": ({k: n.get(k) for k in ("issue_active", "pipe_fma", "pipe_alu", "sm_throughput")}
                        if n else None),
                "peak_how": f"{self.sms} SMs x {FP32_LANES_PER_SM} fp32 lanes x {self.peaks['sm_max_mhz']:.0f} MHz "
                            f"(clocks.max.sm, {self.peaks_how})"}

    def roofline_tensor(self, pairs, d, k_dim, kernel_ms, kernel):
        """bf16 tensor roofline of the kNN selection: `frac` on the method's 2 d flop per pair, `frac_executed`
        on the 2 K flop per pair the bf16x3 split multiplies (K = 16 ceil((3 d + 3) / 16) operand columns)."""
        peak = self.peaks.get("bf16_tflops", 1590.0)
        ach = pairs * 2.0 * d / (kernel_ms * 1e-3) / 1e12 if kernel_ms else None
        ex = pairs * 2.0 * k_dim / (kernel_ms * 1e-3) / 1e12 if kernel_ms else None
        n = self.ncu.get(kernel or "", {})
        return {"bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s",
                "frac": (ach / peak) if ach else None, "frac_executed": (ex / peak) if ex else None,
                "traffic": n.get("dram_bytes"), "flop_per_pair": 2 * d, "flop_executed_per_pair": 2 * k_dim,
                "kernel_ms": kernel_ms, "kernel": kernel,
                "ncu": ({k: n.get(k) for k in ("issue_active", "pipe_tensor", "pipe_alu", "sm_throughput")}
                        if n else None),
                "peak_how": f"bf16_tflops ({self.peaks_how}; cuBLAS bf16, burst: the kernel is timed alone)"}

    # ---- bounds (configs 1, 2, 3, 5-after) -------------------------------------------------------------
    def bounds_brute(self, wl, steps, warmup, cfg_key, do_e2e=False, y_dev=None, policy=None):
        L, torch = self.L, self.torch
        X, y, Xq = self.t(wl.X), (y_dev if y_dev is not None else self.t(wl.y)), self.t(wl.Xq)
        policy = L.LIPFIT_BOUNDS_BRUTE if policy is None else policy
        fn = lambda: L.lipfit_bounds_ex(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights, policy=policy)
        n0 = L.launch_count()
        ms = self.time_steps(fn, steps, warmup)
        launches = (L.launch_count() - n0) * steps // (steps + warmup)
        kms, _ = self.kernel_ms(0, fn, max(1, min(3, steps)))
        pairs = wl.N * wl.Q
        kernel = L.bounds_variant(wl.d, wl.mask, wl.norm)
        res = {"ms_per_step": float(np.mean(ms)), "ms_min": float(np.min(ms)), "pairs": pairs,
               "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "unit": UNIT, "gpu_launches": int(launches),
               "kernel": kernel, "kernel_ms": kms, "policy": "LIPFIT_BOUNDS_BRUTE (every pair evaluated)",
               "roofline": self.roofline(pairs, SURVEY_OPS[cfg_key], EXECUTED_OPS[cfg_key], kms, kernel)}
        outputs = fn()
        if do_e2e:
            pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
            Xh, yh, Xqh = pin(wl.X), pin(wl.y), pin(wl.Xq)
            outs = tuple(torch.empty(wl.Q, dtype=torch.float32).pin_memory().numpy() for _ in range(3))
            sp = torch.cuda.current_stream().cuda_stream
            hfn = lambda: L.lipfit_bounds_host_ex(Xh, yh, Xqh, wl.M, wl.mask, wl.norm, wl.weights, outs, sp,
                                                  L.LIPFIT_BOUNDS_BRUTE)
            hms = self.time_steps(hfn, max(1, steps), warmup)
            res["e2e"] = {"value": pairs / (np.mean(hms) * 1e-3) / 1e9, "unit": UNIT,
                          "ms_per_step": float(np.mean(hms)),
                          "h2d_bytes_per_step": int(Xh.nbytes + yh.nbytes + Xqh.nbytes),
                          "d2h_bytes_per_step": int(sum(o.nbytes for o in outs))}
            afn = lambda: L.lipfit_bounds_host_ex(Xh, yh, Xqh, wl.M, wl.mask, wl.norm, wl.weights, outs, sp, None)
            ams = self.time_steps(afn, max(1, steps), warmup)
            res["e2e_effective_ms"] = float(np.mean(ams))
        return res, outputs, (X, y, Xq)

    def bounds_effective(self, wl, dev_arrays, steps, warmup, brute_outputs=None, brute_ms=None):
        """What the plain entry point lipfit_bounds (LIPFIT_BOUNDS_AUTO) does on this workload."""
        L = self.L
        X, y, Xq = dev_arrays
        fn = lambda: L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
        ms = self.time_steps(fn, steps, warmup)
        kms, n = self.kernel_ms(6, fn, 1)
        *outs, counts = L.lipfit_bounds_ex(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights, policy=L.LIPFIT_BOUNDS_AUTO,
                                           count_pairs=True)
        pairs = wl.N * wl.Q
        res = {"entry_point": "lipfit_bounds (LIPFIT_BOUNDS_AUTO)",
               "path": "exact pruning" if n else "all pairs", "ms_per_step": float(np.mean(ms)),
               "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "unit": "effective " + UNIT,
               "pairs_asked": pairs, "pairs_evaluated": int(counts[0]), "fraction_evaluated": counts[0] / pairs,
               "kernel_ms": kms,
               "evaluated_rate_gpairs_s": (counts[0] / (kms * 1e-3) / 1e9) if kms else None,
               "kernel": "bounds_pruned<norm,DP,DC> (Morton-sorted 32-datum tiles, box tests)"}
        if brute_ms:
            res["all_pairs_ms_per_step"] = brute_ms
            res["speedup_over_all_pairs"] = brute_ms / float(np.mean(ms))
        if brute_outputs is not None:
            self.torch.cuda.synchronize()
            res["max_abs_diff_vs_all_pairs"] = max(float((a - b).abs().max()) for a, b in zip(outs, brute_outputs))
        return res, outs

    def parity_bounds(self, wl, outs, sel, ref, y_range=None):
        """max |gpu - oracle| against 1e-5 * range on exactly the oracle's query sample."""
        tol = 1e-5 * (wl.y_range if y_range is None else y_range)
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
    B = Bench(torch, L, dev, args, sms, peaks, peaks_how)
    if args.configs == "all":
        cfgs = [1, 3, 4, 5, 6, 7, 8, 9, 10, 11, 12, 13, 14] if world == 1 else []
    elif args.configs in ("", "main", "2"):
        cfgs = []
    else:
        cfgs = [int(c) for c in args.configs.split(",") if int(c) != 2]

    # ---- the bench line: config 2, every pair evaluated ----
    wl = make_workload(2, query_seed=1 + 1000 * rank)   # weak scaling: each rank its own batch
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    r2, outputs, dev_arrays = B.bounds_brute(wl, args.steps, args.warmup, 2, do_e2e=True)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    clocks = sampler.stop() if rank == 0 else None
    ms = max_over_ranks(r2["ms_per_step"])
    e2e_ms = max_over_ranks(r2["e2e"]["ms_per_step"])
    eff, eff_outs = B.bounds_effective(wl, dev_arrays, args.steps, args.warmup, outputs, r2["ms_per_step"])
    eff_ms = max_over_ranks(eff["ms_per_step"])
    eff_e2e_ms = max_over_ranks(r2["e2e_effective_ms"])
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    pairs = r2["pairs"]
    line = {
        "metric": METRIC, "value": world * pairs / (ms * 1e-3) / 1e9, "unit": UNIT,
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
        "data": "synthetic",
        "config": {"workload": WORKLOAD, "kernel": r2["kernel"], "l2": "flushed between timed steps (256 MB write)",
                   "step": "lipfit_bounds_ex(LIPFIT_BOUNDS_BRUTE) = a1 prepack + a2 fused all-pairs bounds + finalize",
                   "parallelism": f"query-sharded replicas x{world}, no collective"},
        "clocks": clocks,
        "e2e": {"value": world * pairs / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                "h2d_bytes_per_step": r2["e2e"]["h2d_bytes_per_step"],
                "d2h_bytes_per_step": r2["e2e"]["d2h_bytes_per_step"], "ms_per_step": e2e_ms,
                "entry_point": "lipfit_bounds_host_ex(LIPFIT_BOUNDS_BRUTE), pinned host buffers"},
        "gpu_launches": r2["gpu_launches"],
        "roofline": r2["roofline"],
        "peaks": peaks_how,
    }
    eff.update({"ms_per_step": eff_ms, "value": world * pairs / (eff_ms * 1e-3) / 1e9,
                "e2e": {"ms_per_step": eff_e2e_ms, "value": world * pairs / (eff_e2e_ms * 1e-3) / 1e9,
                        "unit": "effective " + UNIT, "entry_point": "lipfit_bounds_host (LIPFIT_BOUNDS_AUTO)"},
                "note": "same upper/lower/g (min / max over ALL data) from a fraction of the pairs; reported "
                        "beside the all-pairs numbers, never mixed into value / roofline"})
    line["effective"] = eff
    if clocks and clocks.get("sm_mhz"):
        rf = line["roofline"]
        rf["frac_at_observed_clock"] = rf["achieved"] / (sms * FP32_LANES_PER_SM * clocks["sm_mhz"] * 1e6 / 1e12)
    # ---- CPU baseline: the oracle on a bounded sample, with parity on exactly that sample ----
    if not args.no_cpu:
        base, sel, ref = oracle_sample_rate(wl, 10.0)
        line["cpu_baseline"] = base
        line["parity"] = B.parity_bounds(wl, outputs, sel, ref)
        line["effective"]["parity"] = B.parity_bounds(wl, eff_outs, sel, ref)
    del outputs, eff_outs, dev_arrays
    # ---- the other configs ----
    extra = {}
    for c in cfgs:
        t0 = time.perf_counter()
        try:
            extra[f"config{c}"] = run_other_config(B, c)
        except Exception as e:  # report, do not hide
            extra[f"config{c}"] = {"error": repr(e)}
        extra[f"config{c}"]["wall_s"] = time.perf_counter() - t0
        torch.cuda.empty_cache()
    if extra:
        line["configs"] = extra
        par = [v.get("parity", {}).get("ok") for v in extra.values() if isinstance(v.get("parity"), dict)]
        line["all_parity_ok"] = bool(line.get("parity", {}).get("ok", True) and all(p is not False for p in par))
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


CONFIG_DATA = {6: 5, 7: 2, 8: 5, 9: 2, 10: 3, 11: 5, 12: 5, 13: 2, 14: 2}


def run_other_config(B, c):
    import oracle
    torch, L, args = B.torch, B.L, B.args
    wl = make_workload(CONFIG_DATA.get(c, c))
    few = max(1, min(args.steps, 3))
    cpu = not args.no_cpu
    out = {}
    if c in (1, 3):
        # config 1 is latency-bound: timed through the plain entry point (AUTO -> the single-launch kernel, which
        # visits every pair as well); config 3 through the all-pairs kernels
        r, outputs, dev_arrays = B.bounds_brute(wl, few if c == 3 else args.steps, 3, c,
                                                policy=L.LIPFIT_BOUNDS_AUTO if c == 1 else None)
        out.update({k: r[k] for k in ("ms_per_step", "ms_min", "value", "unit", "kernel", "kernel_ms", "policy",
                                      "roofline")})
        out["workload"] = f"BASELINE.json configs[{c - 1}]"
        if c == 1:
            out["kernel"] = "bounds_small<L2,D2>"   # one launch: a1 inside the kernel, all data in shared memory
            out["roofline"] = B.roofline(r["pairs"], SURVEY_OPS[1], EXECUTED_OPS[1], r["kernel_ms"], out["kernel"])
            out["policy"] = "LIPFIT_BOUNDS_AUTO (every pair evaluated)"
            # latency-bound config: an isolated, L2-flushed step exposes the host launch latency; also report the
            # steady state of back-to-back calls (inputs stay in L2; 200 calls between two events)
            X, y, Xq = dev_arrays
            fn = lambda: L.lipfit_bounds(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights)
            for _ in range(20):
                fn()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for _ in range(200):
                fn()
            e1.record()
            e1.synchronize()
            us = e0.elapsed_time(e1) * 1e3 / 200
            out["back_to_back"] = {"us_per_step": us, "value": r["pairs"] / (us * 1e-6) / 1e9, "unit": UNIT,
                                   "note": "200 consecutive lipfit_bounds calls, no L2 flush"}
            moved = wl.X.nbytes + wl.y.nbytes + wl.Xq.nbytes + 3 * 4 * wl.Q
            out["regime"] = ("latency-bound: 1e7 pairs are ~3 us of arithmetic at peak; the 60 percent target does "
                             f"not apply (SURVEY.md §8(d)); bytes moved per step = {moved}")
            out["hbm_gbs_at_step_time"] = moved / (out["ms_per_step"] * 1e-3) / 1e9
        if cpu:
            base, sel, ref = oracle_sample_rate(wl, 4.0)
            out["cpu_baseline"] = base
            out["parity"] = B.parity_bounds(wl, outputs, sel, ref)
    elif c == 4:
        X, Xq = B.t(wl.X), B.t(wl.Xq)
        pairs = wl.N * wl.Q
        res = {}
        for tc in (True, False):
            fn = lambda: L.lipfit_knn(X, Xq, wl.k, None, 0, wl.norm, wl.weights) if tc else \
                L.lipfit_knn_ex(X, Xq, wl.k, None, 0, wl.norm, wl.weights, tensor_cores=False, want_info=False)
            ms = B.time_steps(fn, few if tc else 1, 3 if tc else 1)
            kms, _ = B.kernel_ms(1, fn, 1)
            rms, _ = B.kernel_ms(8, fn, 1)
            idx, dist_, info = L.lipfit_knn_ex(X, Xq, wl.k, None, 0, wl.norm, wl.weights, tensor_cores=tc)
            res[tc] = {"ms_per_step": float(np.mean(ms)), "value": pairs / (np.mean(ms) * 1e-3) / 1e9, "unit": UNIT,
                       "kernel": L.knn_variant(wl.d, 0, wl.norm, tensor_cores=tc), "kernel_ms": kms,
                       "rerank_kernel_ms": rms, "exact_fallback_queries": info["fallbacks"],
                       "key_error_over_bound": info["key_error_ratio"], "outputs": (idx, dist_)}
        r = res[True]
        out.update({k: r[k] for k in r if k != "outputs"})
        out["workload"] = "BASELINE.json configs[3]"
        out["step"] = "lipfit_knn = operand images + tensor-core selection + fp64 re-rank / certificate + exact fallback"
        out["roofline"] = B.roofline_tensor(pairs, wl.d, 16 * ((3 * wl.d + 3 + 15) // 16), r["kernel_ms"], r["kernel"])
        rc = res[False]
        out["cuda_core_selection"] = {k: rc[k] for k in rc if k != "outputs"}
        out["cuda_core_selection"]["roofline"] = B.roofline(pairs, SURVEY_OPS[4], EXECUTED_OPS[4], rc["kernel_ms"],
                                                            rc["kernel"])
        out["cuda_core_selection"]["same_outputs"] = bool(
            torch.equal(r["outputs"][0], rc["outputs"][0]) and torch.equal(r["outputs"][1], rc["outputs"][1]))
        if cpu:
            sel = oracle_subset(wl.Q, 96)
            t0 = time.perf_counter()
            oi, od = oracle.knn(wl.X, wl.Xq[sel], wl.k, None, 0, wl.norm)
            dt = time.perf_counter() - t0
            gi = r["outputs"][0].cpu().numpy()[sel]
            gd = r["outputs"][1].cpu().numpy()[sel]
            out["cpu_baseline"] = {"value": len(sel) * wl.N / dt / 1e9, "unit": UNIT, "cores": oracle.num_threads(),
                                   "kind": "oracle", "sample": f"{len(sel)} of {wl.Q} queries x all {wl.N} data",
                                   "flags": oracle_flags(), "seconds": dt}
            sets_ok = bool(all(set(a) == set(b) for a, b in zip(gi, oi)))
            ulps = float(np.max(np.abs(gd - od.astype(np.float32)) / np.spacing(od.astype(np.float32))))
            out["parity"] = {"index_sets_equal": sets_ok, "max_dist_err_ulps": ulps, "queries": int(len(sel)),
                             "ok": bool(sets_ok and ulps <= 1.0)}
    elif c == 5:
        X, y = B.t(wl.X), B.t(wl.y.copy())
        L.set_timing(True)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        eps, info = L.lipfit_smooth(X, y, wl.M, wl.mask, wl.norm, wl.weights, wl.p, wl.max_iter, 1e-6)
        torch.cuda.synchronize()
        wall = time.perf_counter() - t0
        kms_tot, n = L.get_timing(2)
        L.set_timing(False)
        kms = kms_tot / max(n, 1)
        pairs_eval = wl.N * (wl.N - 1)          # ordered pairs of Eq.(7) covered by one evaluation
        out.update({"workload": "BASELINE.json configs[4]: smoothing (host LBFGS <= 200 iterations), then bounds",
                    "smooth_wall_s": wall, "info": info, "evals": n, "kernel_ms_per_eval": kms,
                    "ms_per_step": kms, "host_share_of_wall": 1.0 - kms_tot * 1e-3 / wall,
                    "value": pairs_eval / (kms * 1e-3) / 1e9,
                    "unit": "G ordered pairs of Eq.(7) per second (each unordered pair is visited once)",
                    "kernel": "smooth_pairs_packed<L2,U0,C5>",
                    "roofline": B.roofline(pairs_eval, SURVEY_OPS["5s"], EXECUTED_OPS["5s"], kms,
                                           "smooth_pairs_packed<L2,U0,C5>", unit_name="ordered_pair")})
        if cpu:
            # objective / gradient at eps = 0 against the oracle's rows (4e10 pairs are unaffordable in full)
            rows = oracle_subset(wl.N, 96)
            t0 = time.perf_counter()
            g_ref, _ = oracle.smooth_rows(wl.X, wl.y, wl.M, np.zeros(wl.N), rows, wl.mask, wl.norm, None, wl.p)
            dt = time.perf_counter() - t0
            _, g0 = L.lipfit_smooth_objective(X, B.t(wl.y), wl.M, None, wl.mask, wl.norm, None, wl.p)
            err = float(np.abs(g0.cpu().numpy()[rows] - g_ref).max() / np.abs(g_ref).max())
            out["cpu_baseline"] = {"value": 2 * len(rows) * (wl.N - 1) / dt / 1e9, "unit": "G ordered pairs/s",
                                   "cores": oracle.num_threads(), "kind": "oracle", "flags": oracle_flags(),
                                   "sample": f"{len(rows)} of {wl.N} gradient rows x all data (both sums of Eq.(7))",
                                   "seconds": dt}
            out["parity"] = {"gradient_rows": int(len(rows)), "max_rel_err": err, "tol": 1e-5, "ok": bool(err <= 1e-5)}
        # a6: bounds on the smoothed z (all pairs), parity against the oracle on the SAME z
        wl_after = make_workload(5)
        z = y.cpu().numpy()
        rb, outputs, dev_arrays = B.bounds_brute(wl_after, few, 2, "5b", y_dev=y)
        out["bounds_after"] = {k: rb[k] for k in ("ms_per_step", "value", "unit", "kernel", "kernel_ms", "policy",
                                                  "roofline")}
        eff, eff_outs = B.bounds_effective(wl_after, dev_arrays, few, 2, outputs, rb["ms_per_step"])
        out["bounds_after"]["effective"] = eff
        if cpu:
            wl_after.y = z
            base, sel, ref = oracle_sample_rate(wl_after, 4.0)
            out["bounds_after"]["cpu_baseline"] = base
            out["bounds_after"]["parity"] = B.parity_bounds(wl_after, outputs, sel, ref, y_range=wl.y_range)
            out["bounds_after"]["effective"]["parity"] = B.parity_bounds(wl_after, eff_outs, sel, ref,
                                                                         y_range=wl.y_range)
            out["parity"]["ok"] = bool(out["parity"]["ok"] and out["bounds_after"]["parity"]["ok"]
                                       and out["bounds_after"]["effective"]["parity"]["ok"])
    elif c == 6:
        out.update(bench_local(B, wl))
    elif c == 7:
        # NEXT-2: weighted sums of the k = 4 best bound values on the config 2 workload
        wk = np.array([0.4, 0.3, 0.2, 0.1], dtype=np.float32)
        X, y, Xq = B.t(wl.X), B.t(wl.y), B.t(wl.Xq)
        fn = lambda: L.lipfit_bounds_topk(X, y, Xq, wl.M, wk, wl.mask, wl.norm, wl.weights)
        ms = B.time_steps(fn, few, 3)
        kms, _ = B.kernel_ms(9, fn, 1)
        pairs = wl.N * wl.Q
        out.update({"workload": "config 2 data and queries, k = 4 best bounds with weights [0.4, 0.3, 0.2, 0.1]",
                    "ms_per_step": float(np.mean(ms)), "kernel_ms": kms, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                    "unit": UNIT, "kernel": "bounds_topk",
                    # the k = 1 work (18 lane-ops per pair in the plain form, 13 in the folded form the kernel
                    # executes) + one compare per side against the worst kept value
                    "roofline": B.roofline(pairs, SURVEY_OPS[2] + 2, EXECUTED_OPS[2] + 2, kms, "bounds_topk")})
        if cpu:
            base, sel, ref = oracle_sample_rate(
                wl, 3.0, lambda xs: oracle.bounds_topk(wl.X, wl.y, xs, wl.M, wk, wl.mask, wl.norm, wl.weights))
            out["cpu_baseline"] = base
            out["parity"] = B.parity_bounds(wl, fn(), sel, ref)
    elif c == 8:
        # NEXT-3: smallest consistent Lipschitz constant of the config 5 data
        X, y = B.t(wl.X), B.t(wl.y)
        # (symmetric distance: under the config's monotone mask the noisy data violate monotonicity, L = +inf)
        fn = lambda: L.lipfit_lipschitz_constant(X, y, None, wl.norm, wl.weights)
        ms = B.time_steps(fn, few, 3)
        kms, _ = B.kernel_ms(3, fn, 1)
        pairs = wl.N * (wl.N - 1)
        out.update({"workload": "config 5 data (d=5, N=200000, L2), symmetric distance",
                    "ms_per_step": float(np.mean(ms)), "kernel_ms": kms, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                    "unit": "G ordered pairs/s (each unordered pair is visited once)",
                    "L": float(fn().cpu().numpy()[0]), "kernel": "smooth_pairs<L2,U5,C0,lipconst>",
                    # plain form per ORDERED pair: 5 sub + 5 fma + sqrt + |dy| + divide + max = 14; executed per
                    # VISITED unordered pair (exact-d symmetric kernel): 5 sub + 5 fma + dy + 2 mul + compare = 14
                    # (7 per ordered pair); survivors of the filter take the fp64 ratio
                    "roofline": B.roofline(pairs, 14, 7, kms, "smooth_pairs<L2,U5,C0,lipconst>",
                                           unit_name="ordered_pair")})
        if cpu:
            n = 20000      # the oracle is O(N^2) on the host: the first 20000 data (4e8 ordered pairs)
            t0 = time.perf_counter()
            ref = oracle.lipschitz_constant(wl.X[:n], wl.y[:n], None, wl.norm, wl.weights)
            dt = time.perf_counter() - t0
            got = float(L.lipfit_lipschitz_constant(B.t(wl.X[:n]), B.t(wl.y[:n]), None, wl.norm,
                                                    wl.weights).cpu().numpy()[0])
            out["cpu_baseline"] = {"value": n * (n - 1) / dt / 1e9, "unit": "G ordered pairs/s",
                                   "cores": oracle.num_threads(), "kind": "oracle", "flags": oracle_flags(),
                                   "sample": f"first {n} of {wl.N} data, all pairs", "seconds": dt}
            out["parity"] = {"data": n, "oracle": ref, "gpu": got, "ok": bool(got == float(np.float32(ref)))}
    elif c in (9, 10, 11):
        # NEXT-4(ii): what lipfit_bounds (LIPFIT_BOUNDS_AUTO -> exact pruning) does on the config 2 / 3 / 5
        # workloads.  "Effective" pairs/s = Q N / step time (the work the all-pairs path would do), reported
        # beside the pairs actually evaluated; never mixed into the all-pairs roofline numbers above.
        X, y, Xq = B.t(wl.X), B.t(wl.y), B.t(wl.Xq)
        steps_p = few if c == 10 else args.steps
        fb = lambda: L.lipfit_bounds_ex(X, y, Xq, wl.M, wl.mask, wl.norm, wl.weights, policy=L.LIPFIT_BOUNDS_BRUTE)
        ms_b = B.time_steps(fb, 1 if c == 10 else 2, 1)
        eff, outs = B.bounds_effective(wl, (X, y, Xq), steps_p, 3, fb(), float(np.mean(ms_b)))
        out.update(eff)
        out["workload"] = "config %d data and queries" % CONFIG_DATA[c]
        kname = {9: "bounds_pruned<L1,DP4,DC2>", 10: "bounds_pruned<Linf,DP8,DC1>", 11: "bounds_pruned<L2,DP8,DC5>"}[c]
        out["kernel"] = kname
        n = B.ncu.get(kname)
        if n:
            out["ncu"] = {k: n.get(k) for k in ("issue_active", "pipe_fma", "pipe_alu", "sm_throughput")}
        # e2e through the public host entry point (H2D + sorts + pruned pass + D2H)
        pin = lambda a: torch.from_numpy(a).pin_memory().numpy()
        Xh, yh, Xqh = pin(wl.X), pin(wl.y), pin(wl.Xq)
        houts = tuple(torch.empty(wl.Q, dtype=torch.float32).pin_memory().numpy() for _ in range(3))
        sp = torch.cuda.current_stream().cuda_stream
        hfn = lambda: L.lipfit_bounds_host(Xh, yh, Xqh, wl.M, wl.mask, wl.norm, wl.weights, houts, sp)
        hms = B.time_steps(hfn, few, 2)
        out["e2e"] = {"ms_per_step": float(np.mean(hms)), "value": wl.N * wl.Q / (np.mean(hms) * 1e-3) / 1e9,
                      "unit": "effective " + UNIT, "entry_point": "lipfit_bounds_host (LIPFIT_BOUNDS_AUTO)",
                      "h2d_bytes_per_step": int(Xh.nbytes + yh.nbytes + Xqh.nbytes),
                      "d2h_bytes_per_step": int(sum(o.nbytes for o in houts))}
        if cpu:
            base, sel, ref = oracle_sample_rate(wl, 3.0)
            out["cpu_baseline"] = base
            out["parity"] = B.parity_bounds(wl, outs, sel, ref)
    elif c == 12:
        out.update(bench_smooth_pruned(B, wl))
    elif c == 13:
        # NEXT-4(iii): monotonicity on parts of the domain on the config 2 workload:
        # case III on x1 (a = 0.3, b = 0.6), case I on x2 (a = b = 0.4), x3, x4 unrestricted
        mon, a, b = [3, 1, 0, 0], [0.3, 0.4, 0.0, 0.0], [0.6, 0.4, 0.0, 0.0]
        X, y, Xq = B.t(wl.X), B.t(wl.y), B.t(wl.Xq)
        fn = lambda: L.lipfit_bounds_region(X, y, Xq, wl.M, mon, a, b, wl.norm, wl.weights)
        ms = B.time_steps(fn, few, 3)
        kms, _ = B.kernel_ms(10, fn, 1)
        pairs = wl.N * wl.Q
        out.update({"workload": "config 2 data and queries; case III on x1 (a=.3, b=.6), case I on x2 (a=b=.4)",
                    "ms_per_step": float(np.mean(ms)), "kernel_ms": kms, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                    "unit": UNIT, "kernel": "bounds_region<L1,DP4>",
                    # restricted coordinate: 2 sub + max + min + 2 accumulate = 6 (two transformed values), free
                    # coordinate: sub + add = 2, epilogue 4 + 2: 2 x 6 + 2 x 2 + 6 = 22 lane-ops per pair here
                    "roofline": B.roofline(pairs, 22, 22, kms, "bounds_region<L1,DP4>")})
        if cpu:
            base, sel, ref = oracle_sample_rate(
                wl, 3.0, lambda xs: oracle.bounds_region(wl.X, wl.y, xs, wl.M, mon, a, b, wl.norm, wl.weights))
            out["cpu_baseline"] = base
            out["parity"] = B.parity_bounds(wl, fn(), sel, ref)
    elif c == 14:
        # OFF-TABLE shapes (no tuned kernel), unstructured normal data (inputs.random_problem), N = 1e5, Q = 1e6:
        #   d = 6, mask [+1,0,0,-1,0,0], L2 -> even-rounded compile-time arithmetic "bounds<L2,U4,C2,padded>"
        #   d = 12, mask [+1,0,-1,0,...], L2 -> the generic kernel "bounds_generic<L2,DP16>" (flag arithmetic)
        def leg(d, mask, ops_plain, ops_exec):
            Xn, yn, Xqn = random_problem(14 + d, 100_000, 1_000_000, d)
            X, y, Xq = B.t(Xn), B.t(yn), B.t(Xqn)
            fn = lambda: L.lipfit_bounds_ex(X, y, Xq, 1.5, mask, 2, None, policy=L.LIPFIT_BOUNDS_BRUTE)
            ms = B.time_steps(fn, few, 3)
            kms, _ = B.kernel_ms(0, fn, 1)
            pairs = Xn.shape[0] * Xqn.shape[0]
            kernel = L.bounds_variant(d, mask, 2)
            res = {"workload": f"off-table shape: d={d} mask {mask} L2 M=1.5, N=1e5 Q=1e6 normal data",
                   "ms_per_step": float(np.mean(ms)), "kernel_ms": kms, "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                   "unit": UNIT, "kernel": kernel, "roofline": B.roofline(pairs, ops_plain, ops_exec, kms, kernel)}
            if cpu:
                sel = oracle_subset(Xqn.shape[0], 600)
                ref = oracle.bounds(Xn, yn, Xqn[sel], 1.5, mask, 2, None)
                worst = max(float(np.abs(o.cpu().numpy()[sel].astype(np.float64) - r).max()) for o, r in zip(fn(), ref))
                mag = max(float(np.abs(r).max()) for r in ref[:2])
                tol = 1e-5 * float(yn.max() - yn.min()) + (d + 4) * 2.0 ** -24 * mag
                res["parity"] = {"max_abs_err": worst, "tol": tol, "ok": bool(worst <= tol), "queries": int(len(sel)),
                                 "note": "unstructured inputs: the stated bar + the fp32 rounding of the candidate "
                                         "(DESIGN.md §6)"}
            return res
        # plain form: 2 per free + 5 per constrained coordinate + epilogue 4 + 2 sqrt: d=6 (4+2): 24; executed the same
        out.update(leg(6, [1, 0, 0, -1, 0, 0], 24, 24))
        # d=12 (6 free + 6 constrained): plain 12 + 30 + 6 = 48; executed by the chunked generic arithmetic over
        # DP = 16 padded coordinates: one chunk of 4 free coordinates (8) + two chunks of flag arithmetic
        # (8 x (sub, mul, 2 max, 2 fma) = 48), the padding chunk skipped, + 2 sqrt + 2 fma + min + max = 62
        out["generic_kernel"] = leg(12, [1, 0, -1, 0] * 3, 48, 62)
        if cpu:
            out["parity"]["ok"] = bool(out["parity"]["ok"] and out["generic_kernel"]["parity"]["ok"])
    return out


def bench_local(B, wl):
    """NEXT-1 (local Lipschitz interpolation) on config 5's data: knots from 1e6 sampled
    pairs, step tables for N = 2e5 (4e10 ordered pairs), evaluation at Q = 1e6 (2e11 pairs)."""
    import oracle
    torch, L, args = B.torch, B.L, B.args
    few = max(1, min(args.steps, 3))
    X, y, Xq = B.t(wl.X), B.t(wl.y), B.t(wl.Xq)
    pi, pk = sample_pairs(3, wl.N, 1_000_000)
    pi_d, pk_d = B.t(pi), B.t(pk)
    J = L.LIPFIT_LOCAL_KNOTS
    knots = L.lipfit_distance_quantiles(X, pi_d, pk_d, J, wl.norm)
    f_tab = lambda: L.lipfit_local_lipschitz(X, y, knots, wl.norm)
    ms_tab = B.time_steps(f_tab, few, 3)
    k_tab, _ = B.kernel_ms(4, f_tab, 1)
    table = f_tab()
    f_ev = lambda: L.lipfit_values_local(X, y, Xq, knots, table, wl.norm)
    ms_ev = B.time_steps(f_ev, few, 3)
    k_ev, _ = B.kernel_ms(5, f_ev, 1)
    # plain formulation per pair (d = 5, J = 16): table: 5 sub + 5 fma + sqrt + |dy| + divide + searchsorted 4 +
    # max = 18 per ordered pair; evaluation: 5 sub + 5 fma + sqrt + searchsorted 4 + table fetch + 2 fma + min + max
    # = 20.  Executed (the d = 5 existing coordinates, knot lookup through the cell table on the float bits of the
    # squared distance, guards; evaluation packed f32x2): ~31 / ~26 lane-ops.
    out = {"workload": "config 5 data (d=5, N=200000), Q=1000000, L2, J=16 knots from 1e6 sampled pairs",
           "table": {"ms_per_step": float(np.mean(ms_tab)), "kernel_ms": k_tab, "kernel": "local_table<L2,DP8>",
                     "value": wl.N * (wl.N - 1) / (np.mean(ms_tab) * 1e-3) / 1e9, "unit": "G ordered pairs/s",
                     "roofline": B.roofline(wl.N * wl.N, 18, 31, k_tab, "local_table<L2,DP8>",
                                            unit_name="ordered_pair")},
           "evaluate": {"ms_per_step": float(np.mean(ms_ev)), "kernel_ms": k_ev, "kernel": "local_eval<L2,DP8>",
                        "value": wl.N * wl.Q / (np.mean(ms_ev) * 1e-3) / 1e9, "unit": UNIT,
                        "roofline": B.roofline(wl.N * wl.Q, 20, 26, k_ev, "local_eval<L2,DP8>")}}
    out["ms_per_step"] = out["evaluate"]["ms_per_step"]
    out["value"] = out["evaluate"]["value"]
    out["unit"] = UNIT
    if not args.no_cpu:
        # pass/fail on exactly the oracle's sample, with the knot-band sandwich of R22 (fp32 rounding of a
        # distance may decide the side of a knot: both neighbours are correct): 64 table rows, 400 queries on
        # a SYNTHETIC seeded table (the oracle never sees a GPU result)
        EPS, TOL = 4e-6, 2e-5
        k64 = knots.astype(np.float64)
        rows = oracle_subset(wl.N, 64)
        t0 = time.perf_counter()
        lo = oracle.local_lipschitz_rows(wl.X, wl.y, k64 * (1 - EPS), rows, wl.norm)
        dt = time.perf_counter() - t0
        hi = oracle.local_lipschitz_rows(wl.X, wl.y, k64 * (1 + EPS), rows, wl.norm)
        got = table.cpu().numpy()[rows].astype(np.float64)
        ok_tab = bool(np.all(got >= lo * (1 - TOL)) and np.all(got <= hi * (1 + TOL)))
        syn = np.maximum.accumulate(np.random.default_rng(5).uniform(0.2, 6.0, (wl.N, J)), axis=1).astype(np.float32)
        sel = oracle_subset(wl.Q, 400)
        up, lw, _ = (v.cpu().numpy()[sel].astype(np.float64)
                     for v in L.lipfit_values_local(X, y, Xq, knots, B.t(syn), wl.norm))
        t64 = syn.astype(np.float64)
        t0 = time.perf_counter()
        Ua, La, _ = oracle.values_local(wl.X, wl.y, wl.Xq[sel], k64 * (1 - EPS), t64, wl.norm)
        dte = time.perf_counter() - t0
        Ub, Lb, _ = oracle.values_local(wl.X, wl.y, wl.Xq[sel], k64 * (1 + EPS), t64, wl.norm)
        tol = 1e-5 * wl.y_range
        ok_ev = bool(np.all(up <= np.maximum(Ua, Ub) + tol) and np.all(up >= np.minimum(Ua, Ub) - tol)
                     and np.all(lw <= np.maximum(La, Lb) + tol) and np.all(lw >= np.minimum(La, Lb) - tol))
        out["cpu_baseline"] = {"table": {"value": len(rows) * (wl.N - 1) / dt / 1e9, "unit": "G ordered pairs/s",
                                         "sample": f"{len(rows)} of {wl.N} rows x all data", "seconds": dt},
                               "evaluate": {"value": len(sel) * wl.N / dte / 1e9, "unit": UNIT,
                                            "sample": f"{len(sel)} of {wl.Q} queries x all data", "seconds": dte},
                               "cores": oracle.num_threads(), "kind": "oracle", "flags": oracle_flags()}
        out["parity"] = {"table_rows": int(len(rows)), "table_ok": ok_tab, "queries": int(len(sel)),
                         "evaluate_ok": ok_ev, "ok": bool(ok_tab and ok_ev),
                         "rule": "sandwich between the oracle with knots * (1 -+ 4e-6) (R22), tol 1e-5 * range "
                                 "(evaluation) / 2e-5 relative (table)"}
    return out


def bench_smooth_pruned(B, wl):
    """Eq.(7) objective / gradient of config 5 with exact pruning (the exact counterpart of the M/3 heuristic,
    PAPER.md:214-218), beside the all-pairs pass, at eps = 0 and at a random eps (sigma 0.05)."""
    import oracle
    torch, L, args = B.torch, B.L, B.args
    few = max(1, min(args.steps, 3))
    X, y = B.t(wl.X), B.t(wl.y)
    eps = B.t((0.05 * np.random.default_rng(7).standard_normal(wl.N)).astype(np.float32))
    pairs = wl.N * (wl.N - 1)
    out = {"workload": "config 5 data (d=5, N=200000, L2, all coordinates monotone, M=3, p=1)",
           "unit": "effective G ordered pairs of Eq.(7) per second", "kernel": "smooth_pruned<L2,DP8,DC5>"}
    for name, e in (("eps0", None), ("eps_random", eps)):
        fn = lambda: L.lipfit_smooth_objective_pruned(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p)
        fu = lambda: L.lipfit_smooth_objective(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p)
        ms = B.time_steps(fn, few, 3)
        kms, _ = B.kernel_ms(7, fn, 1)
        ms_u = B.time_steps(fu, 2, 1)
        F, g, evaluated = L.lipfit_smooth_objective_pruned(X, y, wl.M, e, wl.mask, wl.norm, None, wl.p,
                                                           count_pairs=True)
        Fu, gu = fu()
        torch.cuda.synchronize()
        out[name] = {"ms_per_step": float(np.mean(ms)), "kernel_ms": kms,
                     "value": pairs / (np.mean(ms) * 1e-3) / 1e9,
                     "pairs_evaluated": int(evaluated), "fraction_evaluated": evaluated / pairs,
                     "all_pairs_ms_per_step": float(np.mean(ms_u)),
                     "speedup_over_all_pairs": float(np.mean(ms_u) / np.mean(ms)),
                     "F": F, "F_rel_diff_vs_all_pairs": abs(F - Fu) / Fu,
                     "grad_rel_diff_vs_all_pairs": float((g - gu).abs().max() / gu.abs().max())}
    out["value"] = out["eps0"]["value"]
    out["ms_per_step"] = out["eps0"]["ms_per_step"]
    # the same data without the monotone mask (symmetric distance): only near pairs can violate
    fs = lambda: L.lipfit_smooth_objective_pruned(X, y, wl.M, None, None, wl.norm, None, wl.p)
    fsu = lambda: L.lipfit_smooth_objective(X, y, wl.M, None, None, wl.norm, None, wl.p)
    ms = B.time_steps(fs, few, 3)
    ms_u = B.time_steps(fsu, 2, 1)
    Fs, gs, ev = L.lipfit_smooth_objective_pruned(X, y, wl.M, None, None, wl.norm, None, wl.p, count_pairs=True)
    Fsu, gsu = fsu()
    torch.cuda.synchronize()
    out["eps0_no_mask"] = {"ms_per_step": float(np.mean(ms)), "all_pairs_ms_per_step": float(np.mean(ms_u)),
                           "speedup_over_all_pairs": float(np.mean(ms_u) / np.mean(ms)),
                           "fraction_evaluated": ev / pairs, "F_rel_diff_vs_all_pairs": abs(Fs - Fsu) / Fsu,
                           "grad_rel_diff_vs_all_pairs": float((gs - gsu).abs().max() / gsu.abs().max())}
    # lipfit_smooth on the same data without a mask runs the pruned pass (N >= 8192, no constrained coordinate)
    ys = y.clone()
    t0 = time.perf_counter()
    _, info_s = L.lipfit_smooth(X, ys, wl.M, None, wl.norm, None, wl.p, wl.max_iter, 1e-6)
    torch.cuda.synchronize()
    out["smooth_no_mask"] = {"wall_s": time.perf_counter() - t0, "info": info_s,
                             "ms_per_evaluation_incl_host": 1e3 * (time.perf_counter() - t0) / max(info_s["evals"], 1)}
    if not args.no_cpu:
        rows = oracle_subset(wl.N, 64)
        t0 = time.perf_counter()
        g_ref, _ = oracle.smooth_rows(wl.X, wl.y, wl.M, np.zeros(wl.N), rows, wl.mask, wl.norm, None, wl.p)
        dt = time.perf_counter() - t0
        _, g0 = L.lipfit_smooth_objective_pruned(X, y, wl.M, None, wl.mask, wl.norm, None, wl.p)
        err = float(np.abs(g0.cpu().numpy()[rows] - g_ref).max() / np.abs(g_ref).max())
        out["cpu_baseline"] = {"value": 2 * len(rows) * (wl.N - 1) / dt / 1e9, "unit": "G ordered pairs/s",
                               "cores": oracle.num_threads(), "kind": "oracle", "flags": oracle_flags(),
                               "sample": f"{len(rows)} of {wl.N} gradient rows x all data", "seconds": dt}
        out["parity"] = {"gradient_rows": int(len(rows)), "max_rel_err": err, "tol": 1e-5, "ok": bool(err <= 1e-5)}
    return out


def free_port() -> int:
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--configs", default="all",
                    help="'all' (default; at N = 1 every config below rides on the line), 'main' (config 2 only) or a "
                         "comma list: 1, 3, 4, 5 = BASELINE.json configs; 6 = local Lipschitz (NEXT-1), 7 = top-k "
                         "bounds (NEXT-2), 8 = Lipschitz constant (NEXT-3), 9 / 10 / 11 = exactly pruned bounds on "
                         "the config 2 / 3 / 5 workloads, 12 = exactly pruned smoothing objective (NEXT-4(ii)), "
                         "13 = region monotonicity (NEXT-4(iii)), 14 = off-table shapes (even-rounded / generic kernels)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline / parity legs")
    ap.add_argument("--pipes", action="store_true",
                    help="print the measured issue rates of the fp32 instruction classes (lipfit_pipe_throughput) "
                         "behind DESIGN.md's 'alu' peak, then exit")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    if args.impl == "reference":
        return run_reference(args)
    if args.pipes:
        import paper_2606_04670_b200 as L
        rows = []
        for which in range(16):
            name, lanes, instr = L.pipe_throughput(which)
            rows.append({"instruction": name, "lane_results_per_clk_per_sm": round(lanes, 2),
                         "warp_instr_per_clk_per_sm": round(instr, 3)})
        print(json.dumps({"pipes": rows, "how": "32 warps / SM, 8 independent chains each, clock64 span of the "
                                                "slowest CTA (csrc/pipes.cu)"}))
        return 0
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # not started by torchrun: start the N ranks ourselves (one process per GPU, NCCL for the timing scalar)
        env = dict(os.environ)
        env.setdefault("NCCL_DEBUG", "WARN")
        return subprocess.call(torchrun_command(args.gpus, sys.argv[1:], free_port()), env=env)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
