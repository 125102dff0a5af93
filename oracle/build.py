"""Builds oracle/liblipfit_oracle.so from lipfit_oracle.c with gcc (TEST INFRASTRUCTURE).

Usage: python -m oracle.build      (also called by __graft_entry__.build() and,
on demand, by oracle.load() when the library is missing or stale).
No -march=native: the .so travels to a different host with the gpurun snapshot.
FLAGS is what bench.py reports beside the cpu_baseline.
"""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "lipfit_oracle.c"), os.path.join(HERE, "lipfit_oracle.h")]
LIB = os.path.join(HERE, "liblipfit_oracle.so")
STAMP = LIB + ".srchash"


def _hash() -> str:
    h = hashlib.sha256()
    for p in SRC:
        with open(p, "rb") as f:
            h.update(f.read())
    return h.hexdigest()


def is_fresh() -> bool:
    try:
        with open(STAMP) as f:
            return os.path.exists(LIB) and f.read().strip() == _hash()
    except OSError:
        return False


FLAGS = ["-O2", "-std=c11", "-fopenmp", "-fno-fast-math"]


def build(force: bool = False) -> str:
    if not force and is_fresh():
        return LIB
    cmd = ["gcc", *FLAGS, "-shared", "-fPIC", "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC[0], "-lm"]
    subprocess.run(cmd, check=True, cwd=HERE)
    os.replace(LIB + ".tmp", LIB)
    with open(STAMP, "w") as f:
        f.write(_hash())
    return LIB


if __name__ == "__main__":
    print(build(force=True))
