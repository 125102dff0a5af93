"""Seeded synthetic inputs for the five BASELINE.json configs.

This package holds NONE of the method's arithmetic (no distances, bounds,
selection or smoothing): it only draws the scattered data, evaluates the
generator function f that BASELINE.json names for each config, and draws the
queries.  It is the one module that both the CPU oracle (`oracle/`) and the
CUDA path (`paper_2606_04670_b200/`) are fed from.
"""
from .gen import (CONFIGS, L1, L2, LINF, Workload, make_workload, sample_pairs,  # noqa: F401
                  oracle_subset, random_problem)
