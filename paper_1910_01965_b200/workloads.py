"""Seeded synthetic input generators shared by tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Philox, no decode, no
integrand, no estimator): it only builds the *inputs* of a scan -- the box, the
per-parameter value lists, the sample count and the seed -- for the five
workloads of BASELINE.json `configs` and for the
paper's own workloads (Eq. 2, Eq. 4).
Both the CUDA path and the CPU oracle receive exactly these arrays.

All inputs are synthetic by construction (the paper's workloads are synthetic
closed-form integrands on integer lists {0..99}).
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence

import numpy as np

# Integrand family ids.  Mirrored -- as plain numbers -- by
# include/zmc.h (product) and oracle/zmc_oracle.c (oracle); no code is shared.
C1_COS_XY = 1
C2_SIN_XY2 = 2
C3_OSCILLATORY = 3
C4_GAUSS_PEAK = 4
C5_DAMPED_COS = 5
P6_SIN_SUM = 6          # the paper's Eq. (2)/(4): sin(sum_j y_j + sum_l x_l)
D_CONST_ONE = 100
D_PARAM_ECHO = 101      # consts[0] = i (0-based parameter index)
D_LIN_Y = 102           # consts[0] = k (0-based dimension index)
D_POLY = 103            # prod_k y_k

PREC_F64 = 0            # everything in fp64
PREC_F32E = 1           # fp32 evaluate / fp64 accumulate (oracle: "mirror" mode)

PI = 3.141592653589793


def linspace(lo: float, hi: float, count: int) -> np.ndarray:
    """S8: v_j = lo + j*((hi-lo)/(count-1)) in double, v_{count-1} = hi exactly."""
    if count == 1:
        return np.array([lo], dtype=np.float64)
    step = (hi - lo) / (count - 1)
    v = np.array([lo + j * step for j in range(count)], dtype=np.float64)
    v[-1] = hi
    return v


@dataclasses.dataclass
class Workload:
    name: str
    integrand_id: int
    bounds: np.ndarray            # 2N doubles: a_0,b_0,...,a_{N-1},b_{N-1}
    lists: List[np.ndarray]       # M value lists (float64)
    n_samples: int
    seed: int
    precision: int                # PREC_F64 | PREC_F32E
    consts: np.ndarray            # family constants (float64, may be empty)
    out_f32: bool = False         # fp32 results (cfg 5)
    batch_points: int = 0         # 0 = one batch
    host_out: bool = False        # results streamed to pinned host memory

    @property
    def N(self) -> int:
        return len(self.bounds) // 2

    @property
    def M(self) -> int:
        return len(self.lists)

    @property
    def counts(self) -> List[int]:
        return [len(l) for l in self.lists]

    @property
    def G(self) -> int:
        g = 1
        for l in self.lists:
            g *= len(l)
        return g

    @property
    def evals(self) -> int:
        return self.G * self.n_samples


def _box(lo: float, hi: float, N: int) -> np.ndarray:
    return np.array([lo, hi] * N, dtype=np.float64)


def config(k: int, scale: Optional[Sequence[int]] = None, n_samples: Optional[int] = None) -> Workload:
    """BASELINE.json configs[k-1] (k = 1..5).  `scale` overrides the list lengths
    (same ranges) and `n_samples` the sample count, for reduced parity cases."""
    none = np.zeros(0, dtype=np.float64)
    if k == 1:
        L = list(scale or [1000])
        return Workload("cfg1", C1_COS_XY, _box(0.0, 1.0, 1), [linspace(0.1, 10.0, L[0])],
                        n_samples or 10_000, 1, PREC_F64, none)
    if k == 2:
        L = list(scale or [1000, 1000])
        return Workload("cfg2", C2_SIN_XY2, _box(0.0, PI, 2),
                        [linspace(0.5, 5.0, L[0]), linspace(0.5, 5.0, L[1])],
                        n_samples or 10_000, 2, PREC_F64, none)
    if k == 3:
        L = list(scale or [200, 200, 200])
        return Workload("cfg3", C3_OSCILLATORY, _box(0.0, 1.0, 4),
                        [linspace(0.1, 3.0, c) for c in L],
                        n_samples or 2000, 3, PREC_F32E, np.array([0.25]))
    if k == 4:
        L = list(scale or [100, 100, 100, 100])
        return Workload("cfg4", C4_GAUSS_PEAK, _box(0.0, 1.0, 6),
                        [linspace(1.0, 20.0, L[0])] + [linspace(0.0, 1.0, c) for c in L[1:]],
                        n_samples or 1000, 4, PREC_F32E, none)
    if k == 5:
        L = list(scale or [100] * 5)
        return Workload("cfg5", C5_DAMPED_COS, _box(-1.0, 1.0, 3),
                        [linspace(0.1, 4.0, c) for c in L],
                        n_samples or 256, 5, PREC_F32E, none,
                        out_f32=True, batch_points=1 << 28, host_out=True)
    raise ValueError("config index must be 1..5")


def paper_eq2(M: int, N: int, n_samples: int = 10_000, seed: int = 6, L: int = 100,
              precision: int = PREC_F64) -> Workload:
    """PAPER.md:73-77 Eq. (2): sin(sum y + sum x) on [0,10]^N, x_l in {0..L-1}."""
    return Workload(f"eq2_M{M}_N{N}", P6_SIN_SUM, _box(0.0, 10.0, N),
                    [np.arange(L, dtype=np.float64) for _ in range(M)],
                    n_samples, seed, precision, np.zeros(0))


def paper_eq4(n_samples: int = 100_000, seed: int = 7, L: int = 100,
              precision: int = PREC_F64) -> Workload:
    """PAPER.md:118-122 Eq. (4): the same integrand on [0,1]^6, M=4."""
    return Workload("eq4", P6_SIN_SUM, _box(0.0, 1.0, 6),
                    [np.arange(L, dtype=np.float64) for _ in range(4)],
                    n_samples, seed, precision, np.zeros(0))


def subset_indices_seed_words(count: int):
    """Q17 helper: returns the (counter, key) pairs whose Philox output selects the
    r-th sampled grid point.  The Philox evaluation itself is NOT done here (no
    method arithmetic in this module): callers feed these to their own Philox."""
    return [((r & 0xFFFFFFFF, 0, 0, 0), (0x5EED, 0)) for r in range(count)]


def forced_indices(G: int, batch_points: int) -> List[int]:
    """Q17 forced points: 0, G-1, every batch edge, and the 2^32 overflow traps."""
    pts = {0, G - 1}
    if batch_points:
        m = 1
        while m * batch_points < G:
            pts.add(m * batch_points - 1)
            pts.add(m * batch_points)
            m += 1
    for p in ((1 << 32) - 1, 1 << 32, 1 << 33):
        if p < G:
            pts.add(p)
    return sorted(pts)


def shard_range(G: int, rank: int, world: int):
    """Contiguous flat-index range of `rank` among `world` ranks:
    the first G % world ranks get one extra point.  Returns (first, count)."""
    base, rem = divmod(G, world)
    first = rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)
