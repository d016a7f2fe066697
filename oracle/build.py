"""Build the CPU oracle (TEST INFRASTRUCTURE): gcc -> oracle/libzmc_oracle.so."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
# ZMC_ORACLE_SRC / ZMC_ORACLE_LIB: build and load another copy of the source instead -- used only by
# tests/test_oracle_mutations.py, which checks that a deliberately broken oracle turns the pin tests red.
SRC = os.environ.get("ZMC_ORACLE_SRC") or os.path.join(HERE, "zmc_oracle.c")
LIB = os.environ.get("ZMC_ORACLE_LIB") or os.path.join(HERE, "libzmc_oracle.so")


def build(force: bool = False) -> str:
    import hashlib
    cmd = ["gcc", "-O2", "-std=c11", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-o", LIB + ".tmp", SRC, "-lm"]
    flags = " ".join(c for c in cmd if c not in (SRC, LIB + ".tmp"))                        # not the checkout's absolute paths
    stamp = hashlib.sha256(open(SRC, "rb").read() + flags.encode()).hexdigest()             # content, not file times
    stamp_path = LIB + ".stamp"
    if not force and os.path.exists(LIB) and os.path.exists(stamp_path) and open(stamp_path).read().strip() == stamp:
        return LIB
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    with open(stamp_path, "w") as f:
        f.write(stamp + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force=True))
