"""Generators for the five synthetic workloads of BASELINE.json `configs`.

Recipe:
  * `numpy.random.default_rng(seed)`: data seed 0, query seed 1, noise seed 2.
  * coordinates are drawn in float64 and rounded to fp32;
  * y = f(x) is evaluated in float64 FROM THE fp32-ROUNDED x, noise (if any) is
    added in float64, and the sum is rounded to fp32;
  * "N(0, s)" in BASELINE.json is read as standard deviation s;
  * "clipped to [-3,3]" is `np.clip`, not rejection.
The paper measures on no dataset; these stand in for nothing else.

Nothing here computes a distance, a bound, a neighbour or a penalty.
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Callable, Optional

import numpy as np

L1, L2, LINF = 1, 2, 3


@dataclass
class Workload:
    name: str
    kind: str                 # "bounds" | "knn" | "smooth"
    X: np.ndarray             # [N, d] fp32
    y: np.ndarray             # [N]    fp32
    Xq: np.ndarray            # [Q, d] fp32
    M: float
    mask: np.ndarray          # [d] int32 in {-1,0,+1}
    norm: int                 # 1=L1 2=L2 3=Linf
    weights: np.ndarray       # [d] fp32
    k: int = 0                # kNN only
    p: float = 1.0            # smoothing penalty (R11)
    max_iter: int = 0         # smoothing LBFGS cap
    f: Optional[Callable[[np.ndarray], np.ndarray]] = field(default=None, repr=False)

    @property
    def N(self) -> int:
        return int(self.X.shape[0])

    @property
    def Q(self) -> int:
        return int(self.Xq.shape[0])

    @property
    def d(self) -> int:
        return int(self.X.shape[1])

    @property
    def y_range(self) -> float:
        return float(self.y.astype(np.float64).max() - self.y.astype(np.float64).min())


def _f1(x):  # config 1: y = sin(3 x1) + x2^2
    return np.sin(3.0 * x[:, 0]) + x[:, 1] ** 2


def _f2(x):  # config 2: y = x1 + 2 x2 + 0.5 sin(4 x3) + x4^2
    return x[:, 0] + 2.0 * x[:, 1] + 0.5 * np.sin(4.0 * x[:, 2]) + x[:, 3] ** 2


def _f3(x):  # config 3: y = sum_i tanh(x_i)/i
    i = np.arange(1, x.shape[1] + 1, dtype=np.float64)
    return (np.tanh(x) / i).sum(axis=1)


def _f4(x):  # config 4: y = exp(-||x-0.5||^2) + 0.1 x1
    return np.exp(-((x - 0.5) ** 2).sum(axis=1)) + 0.1 * x[:, 0]


def _f5(x):  # config 5: y = prod_i x_i^0.3
    return np.prod(x ** 0.3, axis=1)


def _uniform(rng, n, d):
    return rng.random((n, d)).astype(np.float32)


def _clipped_normal(rng, n, d):
    return np.clip(rng.standard_normal((n, d)), -3.0, 3.0).astype(np.float32)


# name -> (kind, d, N, Q, draw, f, noise_sigma, M, mask, norm, k, p, max_iter)
CONFIGS = {
    1: dict(kind="bounds", d=2, N=1_000, Q=10_000, draw=_uniform, f=_f1, sigma=0.0,
            M=4.0, mask=[0, 0], norm=L2),
    2: dict(kind="bounds", d=4, N=100_000, Q=1_000_000, draw=_uniform, f=_f2, sigma=0.01,
            M=8.0, mask=[1, 1, 0, 0], norm=L1),
    3: dict(kind="bounds", d=8, N=1_000_000, Q=1_000_000, draw=_clipped_normal, f=_f3, sigma=0.0,
            M=2.0, mask=[1, 0, 0, 0, 0, 0, 0, 0], norm=LINF),
    4: dict(kind="knn", d=16, N=1_000_000, Q=500_000, draw=_uniform, f=_f4, sigma=0.0,
            M=0.0, mask=[0] * 16, norm=L2, k=32),
    5: dict(kind="smooth", d=5, N=200_000, Q=1_000_000, draw=_uniform, f=_f5, sigma=0.05,
            M=3.0, mask=[1] * 5, norm=L2, p=1.0, max_iter=200),
}


def make_workload(config: int, N: Optional[int] = None, Q: Optional[int] = None,
                  data_seed: int = 0, query_seed: int = 1, noise_seed: int = 2) -> Workload:
    """Build config `config` (1..5); N/Q override the sizes (scaled-down parity cases)."""
    c = CONFIGS[config]
    n = int(c["N"] if N is None else N)
    q = int(c["Q"] if Q is None else Q)
    d = c["d"]
    X = c["draw"](np.random.default_rng(data_seed), n, d)
    Xq = c["draw"](np.random.default_rng(query_seed), q, d)
    y64 = c["f"](X.astype(np.float64))
    if c["sigma"] > 0.0:
        y64 = y64 + c["sigma"] * np.random.default_rng(noise_seed).standard_normal(n)
    return Workload(
        name=f"config{config}", kind=c["kind"], X=np.ascontiguousarray(X),
        y=np.ascontiguousarray(y64.astype(np.float32)), Xq=np.ascontiguousarray(Xq),
        M=float(c["M"]), mask=np.asarray(c["mask"], dtype=np.int32), norm=int(c["norm"]),
        weights=np.ones(d, dtype=np.float32), k=int(c.get("k", 0)), p=float(c.get("p", 1.0)),
        max_iter=int(c.get("max_iter", 0)), f=c["f"])


def oracle_subset(Q: int, Qo: int) -> np.ndarray:
    """Deterministic query subset the oracle is run on when the full config is
    unaffordable: the first Qo/2 queries plus Qo/2 evenly strided ones
    (BASELINE.md §3).  Returns sorted unique int64 indices."""
    if Qo >= Q:
        return np.arange(Q, dtype=np.int64)
    h = Qo // 2
    head = np.arange(h, dtype=np.int64)
    strided = np.linspace(h, Q - 1, Qo - h).astype(np.int64)
    return np.unique(np.concatenate([head, strided]))


def random_problem(seed: int, N: int, Q: int, d: int, spread: float = 1.0):
    """Unstructured random problem for hypothesis-style parity cases: returns
    X, y, Xq (fp32), y being an arbitrary (inconsistent) normal draw."""
    rng = np.random.default_rng(seed)
    X = (spread * rng.standard_normal((N, d))).astype(np.float32)
    Xq = (spread * rng.standard_normal((Q, d))).astype(np.float32)
    y = rng.standard_normal(N).astype(np.float32)
    return np.ascontiguousarray(X), np.ascontiguousarray(y), np.ascontiguousarray(Xq)


def sample_pairs(seed: int, N: int, S: int):
    """S random index pairs (i != k) for the inter-point distance sample of local Lipschitz
    interpolation: the random numbers the method draws, passed in as inputs."""
    rng = np.random.default_rng(seed)
    i = rng.integers(0, N, S, dtype=np.int64)
    k = (i + 1 + rng.integers(0, max(N - 1, 1), S, dtype=np.int64)) % max(N, 1)
    return i.astype(np.int32), k.astype(np.int32)

