"""Builds paper_2606_04670_b200/liblipfit.so (the C-ABI library of include/lipfit.h) in-tree with
nvcc for sm_100a only.  `python -m paper_2606_04670_b200.build [--force]`.

The .so is git-ignored but travels to the GPU box with the gpurun snapshot; a hash of the sources
is stored beside it so a stale library is rebuilt on demand (nvcc is present on the GPU box too).
"""
from __future__ import annotations

import concurrent.futures as cf
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "liblipfit.so")
STAMP = LIB + ".srchash"
OBJDIR = os.path.join(HERE, "build")

UNITS = ["prepack.cu", "bounds.cu", "knn.cu", "knn_tc.cu", "smooth.cu", "local.cu", "prune.cu", "region.cu", "pipes.cu", "noalloc.cu", "small.cu", "api.cu", "api_smooth.cu", "lbfgs.cpp"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-I", INCLUDE]


def _sources():
    files = sorted(os.path.join(CSRC, f) for f in os.listdir(CSRC))
    files.append(os.path.join(INCLUDE, "lipfit.h"))
    return files


def _hash() -> str:
    h = hashlib.sha256()
    for p in _sources():
        h.update(os.path.basename(p).encode())
        with open(p, "rb") as f:
            h.update(f.read())
    h.update(" ".join(NVCC_FLAGS[:6]).encode())
    return h.hexdigest()


def is_fresh() -> bool:
    try:
        with open(STAMP) as f:
            return os.path.exists(LIB) and f.read().strip() == _hash()
    except OSError:
        return False


def _compile(unit: str) -> str:
    obj = os.path.join(OBJDIR, unit.rsplit(".", 1)[0] + ".o")
    extra = ["-Xcompiler", "-fopenmp"] if unit.endswith(".cpp") else []    # host LBFGS vector kernels
    cmd = ["nvcc", *NVCC_FLAGS, *extra, "-c", os.path.join(CSRC, unit), "-o", obj]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"nvcc failed for {unit}:\n{r.stdout}\n{r.stderr}")
    return obj


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and is_fresh():
        return LIB
    os.makedirs(OBJDIR, exist_ok=True)
    with cf.ThreadPoolExecutor(max_workers=min(8, len(UNITS))) as ex:
        objs = list(ex.map(_compile, UNITS))
    cmd = ["nvcc", "-shared", "-gencode", "arch=compute_100a,code=sm_100a", "-o", LIB + ".tmp",
           *objs, "-cudart", "static", "-ldl", "-lgomp"]
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError(f"link failed:\n{r.stdout}\n{r.stderr}")
    os.replace(LIB + ".tmp", LIB)
    with open(STAMP, "w") as f:
        f.write(_hash())
    if verbose:
        print("built", LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
