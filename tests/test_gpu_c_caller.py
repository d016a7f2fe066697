"""-m gpu: the C ABI called from a plain C99 program (no Python binding, no torch) -- tests/c_caller/zmc_c_caller.c is built
with gcc against include/zmc.h, libzmc.so and libcudart, run, and its output compared with the CPU oracle."""
import os
import subprocess

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import build as zbuild, workloads as wl

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_a_c99_program_calls_the_library(tmp_path):
    lib = zbuild.build()
    cuda = os.environ.get("CUDA_HOME", "/usr/local/cuda")
    exe, out = str(tmp_path / "zmc_c_caller"), str(tmp_path / "out.bin")
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-O1", "-I", os.path.join(ROOT, "include"), "-I", os.path.join(cuda, "include"),
                    os.path.join(ROOT, "tests", "c_caller", "zmc_c_caller.c"), "-o", exe, lib,
                    "-L", os.path.join(cuda, "lib64"), "-lcudart", "-Wl,-rpath," + os.path.dirname(lib),
                    "-Wl,-rpath," + os.path.join(cuda, "lib64")], check=True)
    L, n = 53, 1000
    r = subprocess.run([exe, out, str(L), str(n)], capture_output=True, text=True, timeout=300)
    assert r.returncode == 0, r.stdout + r.stderr
    got = np.fromfile(out, dtype=np.float64).reshape(4, L)
    w = wl.config(1, n_samples=n)
    w.lists[0] = wl.linspace(0.1, 10.0, L)
    rc, mean_o, err_o = orc.scan_workload(w, 0, L, n_threads=4)
    assert rc == 0
    for mean, err in ((got[0], got[1]), (got[2], got[3])):          # zmc_scan (device outputs), zmc_scan_ex (host, 8 batches)
        assert np.all(np.abs(mean - mean_o) <= 1e-10 * np.maximum(np.abs(mean_o), err_o))
        assert np.all(np.abs(err - err_o) <= 1e-10 * err_o)
    # both calls took the same schedule (AUTO by count), so they agree bit for bit whatever the batching
    assert np.array_equal(got[0], got[2]) and np.array_equal(got[1], got[3])
