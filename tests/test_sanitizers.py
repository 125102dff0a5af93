"""ASan + UBSan over the host-only code: the plain-C oracle and the product's host LBFGS
(csrc/lbfgs.cpp).  compute-sanitizer is not available on this pool, so the device code is covered by the
parity tests only; everything that runs on the host cores is covered here.  CPU only."""
import os
import shutil
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.skipif(shutil.which("g++") is None, reason="needs g++")
def test_oracle_and_lbfgs_under_asan_ubsan(tmp_path):
    exe = str(tmp_path / "sanitize_driver")
    obj = str(tmp_path / "oracle.o")
    san = ["-fsanitize=address,undefined", "-fno-sanitize-recover=all", "-fno-omit-frame-pointer", "-g", "-O1"]
    subprocess.run(["gcc", "-std=c11", "-fopenmp", *san, "-c", os.path.join(ROOT, "oracle", "lipfit_oracle.c"),
                    "-o", obj], check=True)
    subprocess.run(["g++", "-std=c++17", "-fopenmp", *san, os.path.join(ROOT, "tests", "sanitize_driver.cpp"),
                    os.path.join(ROOT, "paper_2606_04670_b200", "csrc", "lbfgs.cpp"), obj, "-o", exe, "-lm"],
                   check=True)
    env = dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1",
               OMP_NUM_THREADS="4")
    r = subprocess.run([exe], capture_output=True, text=True, env=env, timeout=600)
    assert r.returncode == 0, r.stdout + r.stderr
    assert "sanitize_driver ok" in r.stdout
    assert "runtime error" not in r.stderr and "AddressSanitizer" not in r.stderr, r.stderr
