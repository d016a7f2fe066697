"""Third, independent piece: a pure-Python brute-force enumerator for tiny grids.

Written from the definitions, sharing nothing with oracle/ or the CUDA
path: Philox4x32-10 in Python integers, M nested loops over the value lists with a running
counter (no mixed-radix decode), words generated one at a time, sums left to right in Python
floats, exact rational arithmetic where a test asks for it.
"""
from __future__ import annotations

import itertools
import math
from fractions import Fraction

M32 = 0xFFFFFFFF


def philox4x32_10(ctr, key):
    c0, c1, c2, c3 = ctr
    k0, k1 = key
    for r in range(10):
        if r:
            k0 = (k0 + 0x9E3779B9) & M32
            k1 = (k1 + 0xBB67AE85) & M32
        p0 = 0xD2511F53 * c0
        p1 = 0xCD9E8D57 * c2
        c0, c1, c2, c3 = ((p1 >> 32) ^ c1 ^ k0) & M32, p1 & M32, ((p0 >> 32) ^ c3 ^ k1) & M32, p0 & M32
    return [c0, c1, c2, c3]


def word(seed, t, q):
    j = q >> 2
    out = philox4x32_10((j & M32, j >> 32, t & M32, t >> 32), (seed & M32, seed >> 32))
    return out[q & 3]


def uniform_exact(w, f32_mirror=False) -> Fraction:
    if f32_mirror:
        return Fraction(2 * (w >> 9) + 1, 1 << 24)
    return Fraction(2 * w + 1, 1 << 33)


def f32(v: float) -> float:
    import struct
    return struct.unpack("f", struct.pack("f", v))[0]


FAMILIES = {
    1: lambda y, x, c: math.cos(x[0] * y[0]),
    2: lambda y, x, c: math.sin(x[0] * y[0] + x[1] * y[1]),
    100: lambda y, x, c: 1.0,
    101: lambda y, x, c: x[int(c[0])],
    102: lambda y, x, c: y[int(c[0])],
    103: lambda y, x, c: math.prod(y),
}


def _p6(y, x, c):
    arg = 0.0
    for v in y:
        arg += v
    for v in x:
        arg += v
    return math.sin(arg)


def _c3(y, x, c):
    phase = 2.0 * 3.141592653589793 * c[0]
    for k, yk in enumerate(y):
        phase += (x[k % 3] * float(k + 1)) * yk
    return math.cos(phase)


def _poly(y, x, c):
    p = 1.0
    for v in y:
        p *= v
    return p


def _c4(y, x, c):
    """BASELINE.json configs[3]: g = exp(-sum_k a^2 (y_k - w_k)^2), a = x1,
    w_k = x2 for k < 2, x3 for 2 <= k < 4, x4 for k >= 4 (k 0-based, reading Q9)."""
    a = x[0]
    total = 0.0
    for k, yk in enumerate(y):
        if k < 2:
            wk = x[1]
        elif k < 4:
            wk = x[2]
        else:
            wk = x[3]
        total += a * a * (yk - wk) * (yk - wk)
    return math.exp(-total)


def _c5(y, x, c):
    """BASELINE.json configs[4]: g = exp(-x1 |y|^2) cos(x2 y1 + x3 y2 + x4 y3) (1 + x5 y1 y2 y3) (paper's 1-based y)."""
    y1, y2, y3 = y
    x1, x2, x3, x4, x5 = x
    norm2 = y1 * y1 + y2 * y2 + y3 * y3
    return math.exp(-x1 * norm2) * math.cos(x2 * y1 + x3 * y2 + x4 * y3) * (1.0 + x5 * y1 * y2 * y3)


FAMILIES[6] = _p6
FAMILIES[3] = _c3
FAMILIES[4] = _c4
FAMILIES[5] = _c5
FAMILIES[103] = _poly


def enumerate_grid(fid, bounds, lists, n, seed, consts=(), f32_mirror=False):
    """Returns [(mean, stderr, [g_s...])] for every grid point in nested-loop order
    (first list outermost = row-major, last fastest)."""
    N = len(bounds) // 2
    rnd = f32 if f32_mirror else (lambda v: v)
    a = [rnd(bounds[2 * k]) for k in range(N)]
    width = [rnd(bounds[2 * k + 1] - bounds[2 * k]) for k in range(N)]
    V = 1.0
    for wk in width:
        V *= wk
    cs = [rnd(c) for c in consts]
    g_fn = FAMILIES[fid]
    out = []
    t = 0                                   # running counter, no decode
    for xs in itertools.product(*[list(l) for l in lists]):
        x = [rnd(float(v)) for v in xs]
        g = []
        q = 0
        for s in range(n):
            y = []
            for k in range(N):
                u = float(uniform_exact(word(seed, t, q), f32_mirror))   # exact: dyadic, <=33 bits
                y.append(math.fma(u, width[k], a[k]) if hasattr(math, "fma") else _fma(u, width[k], a[k]))
                q += 1
            g.append(g_fn(y, x, cs))
        mean_g = math.fsum(g) / n
        ss = math.fsum((v - mean_g) ** 2 for v in g)
        out.append((V * mean_g, V * math.sqrt(ss / (n - 1) / n), g))
        t += 1
    return out


def _fma(u, w, a):
    """Exactly rounded u*w+a via rationals (Python < 3.13 has no math.fma)."""
    return float(Fraction(u) * Fraction(w) + Fraction(a))
