"""Build and run tools/pipe_rates.cu: the measured dispatch costs behind the ALU roofline.

    python -m paper_1910_01965_b200.pipe_rates          # needs a GPU; prints the table
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tools", "pipe_rates.cu")
EXE = os.path.join(HERE, "build", "pipe_rates")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")


def build() -> str:
    os.makedirs(os.path.dirname(EXE), exist_ok=True)
    if not os.path.exists(EXE) or os.path.getmtime(EXE) < os.path.getmtime(SRC):
        subprocess.run([NVCC, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-o", EXE, SRC], check=True)
    return EXE


if __name__ == "__main__":
    sys.exit(subprocess.run([build()]).returncode)
