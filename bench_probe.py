"""bench_probe.py -- builds and calls libzmc_probe.so (bench_probe.cu), bench.py's micro-benchmark of the SM dispatch costs.

A measurement tool kept beside bench.py, outside the product package: `pipe_rates` in bench.py's JSON line and the sanity
bands of tests/test_gpu_edges.py come from here.  `python bench_probe.py` builds the library (nvcc, sm_100a; no GPU needed)
and, when a GPU is present, prints the table.
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess

ROOT = os.path.dirname(os.path.abspath(__file__))
SRC, HDR, LIB = (os.path.join(ROOT, n) for n in ("bench_probe.cu", "bench_probe.h", "libzmc_probe.so"))
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
         "-Xcompiler", "-fvisibility=hidden", "-Wno-deprecated-gpu-targets", "-shared"]
MAX_ROWS = 48


class _Row(ctypes.Structure):
    _fields_ = [("name", ctypes.c_char * 72), ("cycles", ctypes.c_double), ("parallel", ctypes.c_double),
                ("serial", ctypes.c_double)]


class _Report(ctypes.Structure):
    _fields_ = [("sm_mhz", ctypes.c_double), ("sm_count", ctypes.c_int32), ("n_rows", ctypes.c_int32), ("rows", _Row * MAX_ROWS)]


def build(force: bool = False) -> str:
    """Content-stamped like the main library (a snapshot copied to a GPU box arrives with shuffled file times)."""
    stamp = hashlib.sha256(open(SRC, "rb").read() + open(HDR, "rb").read() + " ".join(FLAGS).encode()).hexdigest()
    stamp_path = LIB + ".stamp"
    if not force and os.path.exists(LIB) and os.path.exists(stamp_path) and open(stamp_path).read().strip() == stamp:
        return LIB
    subprocess.run([NVCC] + FLAGS + ["-I", ROOT, "-o", LIB + ".tmp", SRC], check=True)
    os.replace(LIB + ".tmp", LIB)
    with open(stamp_path, "w") as f:
        f.write(stamp + "\n")
    return LIB


_lib = None


def measure_pipes(stream_handle: int = 0) -> dict:
    """bench_probe.h bench_measure_pipes on the current device; `stream_handle` is a cudaStream_t as an integer."""
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        _lib.bench_measure_pipes.argtypes = [ctypes.POINTER(_Report), ctypes.c_void_p]
        _lib.bench_measure_pipes.restype = ctypes.c_int
    rep = _Report()
    rc = _lib.bench_measure_pipes(ctypes.byref(rep), ctypes.c_void_p(stream_handle))
    if rc != 0:
        raise RuntimeError(f"bench_measure_pipes failed: cudaError {rc}")
    return {"sm_mhz": rep.sm_mhz, "sm_count": rep.sm_count,
            "rows": [{"name": rep.rows[i].name.decode(), "cycles": rep.rows[i].cycles, "parallel": rep.rows[i].parallel,
                      "serial": rep.rows[i].serial} for i in range(rep.n_rows)]}


if __name__ == "__main__":
    print(build())
    import torch
    if torch.cuda.is_available():
        r = measure_pipes(torch.cuda.current_stream().cuda_stream)
        print(f"# SM clock {r['sm_mhz']:.0f} MHz, {r['sm_count']} SMs; SMSP-cycles per group per warp: measured / parallel / serial")
        for row in r["rows"]:
            print(f"{row['cycles']:8.3f} {row['parallel']:8.3f} {row['serial']:8.3f}  {row['name']}")
