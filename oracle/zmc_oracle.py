"""ctypes face of the CPU oracle (oracle/zmc_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this module.  It does not import the product
package and the product package does not import it.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

from . import build as _build

MODE_F64 = 0
MODE_F32_MIRROR = 1

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(_build.build())
        _lib.zmc_oracle_word.restype = ctypes.c_uint32
        _lib.zmc_oracle_word.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64]
        _lib.zmc_oracle_uniform.restype = ctypes.c_double
        _lib.zmc_oracle_uniform.argtypes = [ctypes.c_uint32, ctypes.c_int]
        _lib.zmc_oracle_philox.restype = None
    return _lib


def philox(ctr: Sequence[int], key: Sequence[int]):
    c = (ctypes.c_uint32 * 4)(*ctr)
    k = (ctypes.c_uint32 * 2)(*key)
    o = (ctypes.c_uint32 * 4)()
    lib().zmc_oracle_philox(c, k, o)
    return [int(v) for v in o]


def word(seed: int, t: int, q: int) -> int:
    return int(lib().zmc_oracle_word(seed, t, q))


def uniform(w: int, mode: int) -> float:
    return float(lib().zmc_oracle_uniform(w, mode))


USER_FN = ctypes.CFUNCTYPE(ctypes.c_double, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double),
                           ctypes.POINTER(ctypes.c_double))
_user_keepalive = []


def set_user_integrand(c_body: str, N: int, M: int, n_consts: int = 0):
    """Compile `double g(const double* y, const double* x, const double* c) { <c_body> }` with gcc (R = double) and
    make it the integrand of every id >= 1000.  The same body text is what zmc_register_integrand hands to NVRTC."""
    import hashlib
    import subprocess
    import tempfile
    # the helper names include/zmc.h offers to user bodies (zmc_register_integrand), by their plain definitions
    helpers = ("static double zmc_sin(double v) { return sin(v); }\nstatic double zmc_cos(double v) { return cos(v); }\n"
               "static double zmc_sinpi(double v) { return sin(3.141592653589793 * v); }\n"
               "static double zmc_cospi(double v) { return cos(3.141592653589793 * v); }\n"
               "static double zmc_exp(double v) { return exp(v); }\nstatic double zmc_exp2(double v) { return exp2(v); }\n")
    src = ("#include <math.h>\n#define R double\n" + helpers +
           "double zmc_user_g(const double* y, const double* x, const double* c) {\n" + c_body + "\n}\n")
    d = os.path.join(tempfile.gettempdir(), "zmc_oracle_user")
    os.makedirs(d, exist_ok=True)
    base = os.path.join(d, hashlib.sha1(src.encode()).hexdigest()[:16])
    if not os.path.exists(base + ".so"):
        with open(base + ".c", "w") as f:
            f.write(src)
        subprocess.run(["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-Wno-unused-function", "-shared", "-fPIC", base + ".c",
                        "-o", base + ".so", "-lm"],
                       check=True)
    so = ctypes.CDLL(base + ".so")
    fn = ctypes.cast(so.zmc_user_g, USER_FN)
    _user_keepalive.append((so, fn))
    lib().zmc_oracle_set_user.restype = None
    lib().zmc_oracle_set_user.argtypes = [USER_FN, ctypes.c_int, ctypes.c_int, ctypes.c_int]
    lib().zmc_oracle_set_user(fn, N, M, n_consts)


def _marshal(bounds, lists, consts):
    b = np.ascontiguousarray(bounds, dtype=np.float64)
    ls = [np.ascontiguousarray(l, dtype=np.float64) for l in lists]
    ptrs = (ctypes.POINTER(ctypes.c_double) * len(ls))(
        *[l.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) for l in ls])
    counts = (ctypes.c_int64 * len(ls))(*[len(l) for l in ls])
    c = np.ascontiguousarray(consts if consts is not None else [], dtype=np.float64)
    return b, ls, ptrs, counts, c


def _dp(a):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def scan(integrand_id: int, bounds, lists, n_samples: int, seed: int, mode: int = MODE_F64,
         consts=None, first_index: int = 0, count: Optional[int] = None, n_threads: int = 1):
    """Contiguous flat range; returns (status, mean[count], stderr[count]) as float64."""
    b, ls, ptrs, counts, c = _marshal(bounds, lists, consts)
    if count is None:
        count = 1
        for l in ls:
            count *= len(l)
        count -= first_index
    mean = np.full(max(count, 0), np.nan)
    err = np.full(max(count, 0), np.nan)
    rc = lib().zmc_oracle_scan(
        ctypes.c_int(integrand_id), ctypes.c_int(len(b) // 2), _dp(b), ctypes.c_int(len(ls)), ptrs, counts,
        ctypes.c_uint64(n_samples), ctypes.c_uint64(seed), ctypes.c_int(mode), _dp(c), ctypes.c_int(len(c)),
        ctypes.c_uint64(first_index), ctypes.c_uint64(max(count, 0)), _dp(mean), _dp(err),
        ctypes.c_int(n_threads))
    return int(rc), mean, err


def points(integrand_id: int, bounds, lists, n_samples: int, seed: int, indices, mode: int = MODE_F64,
           consts=None, n_threads: int = 1):
    """Arbitrary subset of flat indices; returns (status, mean, stderr)."""
    b, ls, ptrs, counts, c = _marshal(bounds, lists, consts)
    idx = np.ascontiguousarray(indices, dtype=np.uint64)
    mean = np.full(len(idx), np.nan)
    err = np.full(len(idx), np.nan)
    rc = lib().zmc_oracle_points(
        ctypes.c_int(integrand_id), ctypes.c_int(len(b) // 2), _dp(b), ctypes.c_int(len(ls)), ptrs, counts,
        ctypes.c_uint64(n_samples), ctypes.c_uint64(seed), ctypes.c_int(mode), _dp(c), ctypes.c_int(len(c)),
        idx.ctypes.data_as(ctypes.POINTER(ctypes.c_uint64)), ctypes.c_uint64(len(idx)),
        _dp(mean), _dp(err), ctypes.c_int(n_threads))
    return int(rc), mean, err


def samples(integrand_id: int, bounds, lists, n_samples: int, seed: int, t: int, mode: int = MODE_F64,
            consts=None):
    """The n_samples values g_s of one grid point, in sample order."""
    b, ls, ptrs, counts, c = _marshal(bounds, lists, consts)
    g = np.full(n_samples, np.nan)
    rc = lib().zmc_oracle_samples(
        ctypes.c_int(integrand_id), ctypes.c_int(len(b) // 2), _dp(b), ctypes.c_int(len(ls)), ptrs, counts,
        ctypes.c_uint64(n_samples), ctypes.c_uint64(seed), ctypes.c_int(mode), _dp(c), ctypes.c_int(len(c)),
        ctypes.c_uint64(t), _dp(g))
    return int(rc), g


def scan_workload(w, first_index: int = 0, count: Optional[int] = None, n_threads: int = 1):
    """Run a paper_1910_01965_b200.workloads.Workload-shaped object (duck-typed)."""
    return scan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, w.precision, w.consts,
                first_index, count, n_threads)


def points_workload(w, indices, n_threads: int = 1):
    return points(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, indices, w.precision,
                  w.consts, n_threads)
