"""Build libzmc.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1910_01965_b200.build [--force]

Every .cu under csrc/ is compiled to an object (in parallel) and linked into
paper_1910_01965_b200/libzmc.so.  nvcc cross-compiles without a GPU.
"""
from __future__ import annotations

import concurrent.futures
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
# ZMC_VARIANT=<name> builds an experimental copy (extra nvcc flags in ZMC_EXTRA_FLAGS) next to the product library
VARIANT = os.environ.get("ZMC_VARIANT", "")
OBJ = os.path.join(HERE, "build" + ("_" + VARIANT if VARIANT else ""))
LIB = os.path.join(HERE, "libzmc" + ("_" + VARIANT if VARIANT else "") + ".so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
INCLUDE = os.path.normpath(os.path.join(HERE, "..", "include"))
FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-I", INCLUDE, "-I", OBJ,
         "-Xcompiler", "-fPIC", "-Xcompiler", "-fvisibility=hidden"] + os.environ.get("ZMC_EXTRA_FLAGS", "").split()
# headers handed to NVRTC when a user integrand is compiled at run time (zmc_register_integrand): embedded as strings
RTC_HEADERS = ["zmc_compat.h", "zmc_params.h", "zmc_math.cuh", "zmc_families.cuh", "zmc_kernel.cuh"]


def _write_rtc_headers():
    """build/zmc_rtc_headers.inc: {name, text} pairs of the kernel headers (+ zmc.h) as raw string literals."""
    out = os.path.join(OBJ, "zmc_rtc_headers.inc")
    parts = []
    for name, path in [(h, os.path.join(CSRC, h)) for h in RTC_HEADERS] + [("zmc.h", os.path.join(INCLUDE, "zmc.h"))]:
        text = open(path).read()
        chunks = [text[i:i + 8000] for i in range(0, len(text), 8000)]       # stay below the literal length limit
        parts.append('{"%s", %s},' % (name, " ".join('R"ZMCHDR(%s)ZMCHDR"' % c for c in chunks)))
    new = "\n".join(parts) + "\n"
    if not os.path.exists(out) or open(out).read() != new:
        with open(out, "w") as f:
            f.write(new)
    return out


def _newest(paths):
    return max(os.path.getmtime(p) for p in paths)


def _source_stamp(srcs, deps) -> str:
    """Hash of everything the library is built from.  File times are not trusted alone: a snapshot copied to another
    machine (gpurun) arrives with shuffled mtimes, and a rebuild there costs half a minute of GPU time."""
    import hashlib
    # the flags without the checkout's absolute paths: the same sources at another path (the GPU box's scratch copy) are the same build
    h = hashlib.sha256(" ".join("<include>" if f == INCLUDE else "<obj>" if f == OBJ else f for f in FLAGS).encode())
    for path in sorted(set(srcs + deps)):
        h.update(os.path.basename(path).encode())
        h.update(open(path, "rb").read())
    return h.hexdigest()


def build(force: bool = False, verbose: bool = False) -> str:
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    deps = glob.glob(os.path.join(CSRC, "*.cuh")) + glob.glob(os.path.join(CSRC, "*.h")) + \
        [os.path.join(HERE, "..", "include", "zmc.h")]
    os.makedirs(OBJ, exist_ok=True)
    deps.append(_write_rtc_headers())
    stamp_path = LIB + ".stamp"
    stamp = _source_stamp(srcs, deps)
    if not force and os.path.exists(LIB) and os.path.exists(stamp_path) and open(stamp_path).read().strip() == stamp:
        return LIB                                   # built from exactly these sources, whatever the file times say
    if os.path.exists(stamp_path):
        force = True                                 # sources changed since the stamped build: do not trust object times
    dep_time = _newest(deps)
    jobs = []
    objs = []
    for src in srcs:
        obj = os.path.join(OBJ, os.path.basename(src)[:-3] + ".o")
        objs.append(obj)
        if force or not os.path.exists(obj) or os.path.getmtime(obj) < max(os.path.getmtime(src), dep_time):
            jobs.append([NVCC] + FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", src, "-o", obj])
    if jobs:
        with concurrent.futures.ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for res in ex.map(lambda c: subprocess.run(c, capture_output=True, text=True), jobs):
                if verbose or res.returncode:
                    sys.stderr.write(res.stdout + res.stderr)
                if res.returncode:
                    raise RuntimeError("nvcc failed: " + " ".join(res.args))
    if jobs or not os.path.exists(LIB) or os.path.getmtime(LIB) < _newest(objs):
        cmd = [NVCC, "-Wno-deprecated-gpu-targets", "-shared", "-o", LIB + ".tmp"] + objs + ["-ldl"]
        subprocess.run(cmd, check=True)
        os.replace(LIB + ".tmp", LIB)
    with open(stamp_path, "w") as f:
        f.write(stamp + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
