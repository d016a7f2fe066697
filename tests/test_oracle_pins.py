"""Pins of the CPU oracle against things other than itself (CPU-only, -m "not gpu").

T1 Philox known answers + S3 stream values (tests/golden), T2 uniform extremes and exactness,
T3 decode via param_echo (incl. t >= 2^32), T4 const_one, T5 brute force on tiny grids +
batch-cut invariance + prefix property, T6 the n=4 worked example.  (SURVEY.md 8(c) pins.)
"""
import os
from fractions import Fraction

import numpy as np
import pytest

import brute_force as bf
from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


# ---- T1 -----------------------------------------------------------------------------------
def test_philox_known_answer_vectors():
    for r in _rows("philox_kat.txt"):
        v = [int(h, 16) for h in r]
        assert orc.philox(v[0:4], v[4:6]) == v[6:10]
        assert bf.philox4x32_10(v[0:4], v[4:6]) == v[6:10]


def test_stream_layout_s3_values():
    for r in _rows("stream_s3.txt"):
        seed, t, block = int(r[0], 16), int(r[1]), int(r[2])
        want = [int(h, 16) for h in r[3:7]]
        got = [orc.word(seed, t, 4 * block + lane) for lane in range(4)]
        assert got == want
        assert [bf.word(seed, t, 4 * block + lane) for lane in range(4)] == want


def test_packed_words_n3():
    for r in _rows("n3_words.txt"):
        seed, t, N, s = int(r[0]), int(r[1]), int(r[2]), int(r[3])
        want = [int(h, 16) for h in r[4:4 + N]]
        assert [orc.word(seed, t, s * N + k) for k in range(N)] == want


def test_word_counter_is_64bit_clean():
    # block index above 2^32 must land in counter word 1, t above 2^32 in counter word 3
    q = (1 << 34) + 5 * 4 + 2
    t = (3 << 32) + 17
    seed = 0xABCDEF0123456789
    j = q >> 2
    ref = bf.philox4x32_10((j & bf.M32, j >> 32, t & bf.M32, t >> 32), (seed & bf.M32, seed >> 32))
    assert orc.word(seed, t, q) == ref[2]


# ---- T2 -----------------------------------------------------------------------------------
def test_uniform_extremes_and_exactness():
    assert orc.uniform(0, orc.MODE_F64) == 2.0 ** -33
    assert orc.uniform(0xFFFFFFFF, orc.MODE_F64) == 1.0 - 2.0 ** -33
    assert orc.uniform(0x80000000, orc.MODE_F64) == 0.5 + 2.0 ** -33
    assert orc.uniform(0, orc.MODE_F32_MIRROR) == 2.0 ** -24
    assert orc.uniform(0xFFFFFFFF, orc.MODE_F32_MIRROR) == 1.0 - 2.0 ** -24
    assert orc.uniform(0x80000000, orc.MODE_F32_MIRROR) == 0.5 + 2.0 ** -24
    rng = np.random.default_rng(7)
    for w in [int(v) for v in rng.integers(0, 1 << 32, size=200)] + [1, 0x1FF, 0x200, 0xFFFFFE00]:
        u64 = orc.uniform(w, orc.MODE_F64)
        u32 = orc.uniform(w, orc.MODE_F32_MIRROR)
        assert Fraction(u64) == Fraction(2 * w + 1, 1 << 33)
        assert Fraction(u32) == Fraction(2 * (w >> 9) + 1, 1 << 24)
        assert float(np.float32(u32)) == u32            # exactly representable in float
        assert 0.0 < u32 < 1.0 and 0.0 < u64 < 1.0
        # symmetric about 1/2: complementing the word mirrors the uniform
        assert orc.uniform(w ^ 0xFFFFFFFF, orc.MODE_F64) == 1.0 - u64


def test_lin_y_mean_in_exact_integer_arithmetic():
    # lin_y: estimate = V * (a + width * sum(2 w_s + 1) / (n 2^33)), V = width, in exact rationals (S4 pin)
    a, b, n, seed, t = -1.5, 2.25, 37, 11, 3
    lists = [np.arange(5.0)]
    rc, mean, _ = orc.scan(wl.D_LIN_Y, [a, b], lists, n, seed, consts=[0.0], first_index=t, count=1)
    assert rc == 0
    tot = sum(2 * bf.word(seed, t, s) + 1 for s in range(n))
    # y_s = fma(u, width, a) is exact here? not in general -> compare to 1 ulp of the rational value
    exact = Fraction(b - a) * (Fraction(a) + Fraction(b - a) * Fraction(tot, n << 33))
    assert abs(Fraction(mean[0]) - exact) <= abs(exact) * Fraction(1, 1 << 50)


# ---- T3 -----------------------------------------------------------------------------------
@pytest.mark.parametrize("counts", [(3,), (2, 3), (3, 2, 2), (4, 1, 3, 2)])
def test_decode_param_echo_small(counts):
    lists = [np.array([10.0 * (i + 1) + j for j in range(c)]) for i, c in enumerate(counts)]
    G = int(np.prod(counts))
    mesh = np.meshgrid(*lists, indexing="ij")
    for i in range(len(counts)):
        rc, mean, err = orc.scan(wl.D_PARAM_ECHO, [0.0, 1.0], lists, 3, 9, consts=[float(i)])
        assert rc == 0
        assert np.array_equal(mean, mesh[i].reshape(-1))
        assert np.all(err == 0.0)
        assert len(mean) == G


def test_decode_above_2_pow_32():
    counts = (70000, 70000, 3)               # G = 1.47e10 > 2^32
    lists = [np.arange(c, dtype=np.float64) + 0.5 * i for i, c in enumerate(counts)]
    idx = [0, (1 << 32) - 1, 1 << 32, (1 << 33) + 12345, 70000 * 70000 * 3 - 1]
    for i in range(3):
        rc, mean, err = orc.points(wl.D_PARAM_ECHO, [0.0, 1.0], lists, 2, 1, idx, consts=[float(i)])
        assert rc == 0
        for t, m in zip(idx, mean):
            digits = np.unravel_index(t, counts)    # numpy's C-order unravel = S1
            assert m == lists[i][digits[i]]
        assert np.all(err == 0.0)


# ---- T4 -----------------------------------------------------------------------------------
def test_const_one_gives_volume_and_zero_stderr():
    bounds = [0.0, 2.0, -1.0, 0.5, 3.0, 3.25]
    rc, mean, err = orc.scan(wl.D_CONST_ONE, bounds, [np.arange(4.0), np.arange(3.0)], 17, 5)
    assert rc == 0
    assert np.all(mean == 2.0 * 1.5 * 0.25)
    assert np.all(err == 0.0)


# ---- T5 -----------------------------------------------------------------------------------
S5_BOX = [0.1, 0.7, -0.3, 1.9]
BF_CASES = [
    # fid, bounds, lists, n, consts, bit_exact
    (wl.D_POLY, [0.0, 1.0, -1.0, 2.0], [[1.0, 2.0], [0.5, 1.5, 2.5]], 5, (), True),
    (wl.D_POLY, [0.0, 1.0, -1.0, 2.0, 0.25, 0.75], [[1.0, 2.0, 3.0], [0.5, 1.5], [7.0, 8.0]], 9, (), True),
    (wl.D_LIN_Y, [0.0, 1.0, -1.0, 2.0, 0.25, 0.75], [[1.0, 2.0], [0.5, 1.5, 2.5]], 4, (2.0,), True),
    (wl.D_PARAM_ECHO, [0.0, 1.0], [[1.0, 2.0], [0.5, 1.5, 2.5]], 4, (1.0,), True),
    (wl.C1_COS_XY, [0.0, 1.0], [[0.1, 3.0, 10.0]], 9, (), False),
    (wl.C2_SIN_XY2, [0.0, wl.PI, 0.0, wl.PI], [[0.5, 5.0], [0.5, 2.0, 5.0]], 5, (), False),
    (wl.C3_OSCILLATORY, [0.0, 1.0] * 3, [[0.1, 3.0], [1.0, 2.0], [0.3, 0.7]], 4, (0.25,), False),
    (wl.P6_SIN_SUM, [0.0, 10.0] * 3, [[0.0, 1.0, 2.0], [5.0, 99.0]], 5, (), False),
    # c4 / c5 with every parameter different (and boxes that differ between the dimension pairs), so that a swapped
    # parameter, a dropped y_k or a wrong sign changes every sample value
    (wl.C4_GAUSS_PEAK, [0.0, 1.0, 0.0, 1.0, 0.0, 1.0, 0.0, 1.0, 0.0, 0.5, 0.0, 0.5],
     [[1.0, 2.5], [0.2], [0.45, 0.7], [0.9, 0.1]], 5, (), False),
    (wl.C5_DAMPED_COS, [-1.0, 1.0, -1.0, 1.0, -1.0, 1.0], [[0.1, 1.3], [0.7], [2.9, 1.1], [4.0], [3.7, 0.4]], 6, (), False),
    (wl.C5_DAMPED_COS, [0.0, 1.0, -0.5, 1.0, 0.25, 2.0], [[0.3], [1.7], [0.6], [2.2], [1.9, -2.5]], 7, (), False),
    # reading S5 (Eq. 1 is silent on the sample map, so the reading is the definition):
    # boxes and constants that are NOT exactly representable in float and whose widths are not short dyadics.  F64 mode:
    # u * width needs more than 53 bits, so fma(u, width, a) and the unfused u * width + a differ in the last bit of many
    # samples (bit-exact families).  Mirror mode: float(a_k) != a_k, float(b - a) != float(b) - float(a) and
    # float(u) != u (asserted in test_s5_cases_exercise_every_rounding_site below), so leaving any of them unrounded,
    # or rounding the width the other way, moves every sample by ~1e-8.
    (wl.D_POLY, S5_BOX, [[1.0, 2.0], [0.5, 1.5, 2.5]], 9, (), True),
    (wl.D_LIN_Y, S5_BOX, [[1.0, 2.0], [0.5, 1.5]], 9, (0.0,), True),
    (wl.D_LIN_Y, S5_BOX, [[1.0, 2.0], [0.5, 1.5]], 9, (1.0,), True),
    (wl.C3_OSCILLATORY, S5_BOX, [[0.1, 3.0], [1.0, 2.0], [0.3, 0.7]], 6, (0.6,), False),
]


def test_s5_cases_exercise_every_rounding_site():
    """The S5 cases above only pin what they claim if the roundings they are meant to catch are not the identity."""
    import struct

    def f32(v):
        return struct.unpack("f", struct.pack("f", v))[0]

    for k in range(len(S5_BOX) // 2):
        a, b = S5_BOX[2 * k], S5_BOX[2 * k + 1]
        assert f32(a) != a                                   # "a_k not rounded in mirror mode" changes y
        assert f32(b - a) != f32(b) - f32(a)                 # "width = float(b) - float(a)" changes y
        assert f32(b - a) != b - a
    assert f32(0.6) != 0.6                                   # "consts not rounded in mirror mode" changes c3's phase
    # F64 mode: the product u * width is inexact for these widths, so fused and unfused sample maps differ somewhere
    differ = 0
    for t in range(4):
        for q in range(18):
            u = bf.uniform_exact(bf.word(3, t, q))
            k = q % 2
            a, w = S5_BOX[2 * k], S5_BOX[2 * k + 1] - S5_BOX[2 * k]
            differ += bf._fma(float(u), w, a) != float(u) * w + a
    assert differ >= 10


@pytest.mark.parametrize("case", BF_CASES)
@pytest.mark.parametrize("mirror", [False, True])
def test_brute_force_tiny_grids(case, mirror):
    fid, bounds, lists, n, consts, exact = case
    seed = 3
    ref = bf.enumerate_grid(fid, bounds, lists, n, seed, consts, f32_mirror=mirror)
    mode = orc.MODE_F32_MIRROR if mirror else orc.MODE_F64
    rc, mean, err = orc.scan(fid, bounds, [np.array(l) for l in lists], n, seed, mode, list(consts))
    assert rc == 0 and len(mean) == len(ref)
    for t, (m, e, g) in enumerate(ref):
        rc, gs = orc.samples(fid, bounds, [np.array(l) for l in lists], n, seed, t, mode, list(consts))
        assert rc == 0
        if exact:
            assert list(gs) == g                     # every sample value bit-exact
            # the enumerator rounds three times in double (fsum, / n, * V -- V is inexact for S5_BOX), the oracle once from
            # long double (reading S6): up to 1.5 ulp = 3.4e-16 apart
            assert abs(mean[t] - m) <= 4e-16 * abs(m)
            assert abs(err[t] - e) <= 1e-15 * abs(e) + 1e-300
        else:
            assert np.allclose(gs, g, rtol=0, atol=1e-15)
            assert abs(mean[t] - m) <= 1e-15 * max(1.0, abs(m))
            assert abs(err[t] - e) <= 1e-14 * abs(e) + 1e-18


def test_batch_cut_invariance_bit_exact():
    w = wl.config(2, scale=[7, 9], n_samples=50)
    rc, mean, err = orc.scan_workload(w)
    assert rc == 0
    parts_m, parts_e = [], []
    for first, count in [(0, 5), (5, 1), (6, 40), (46, 17)]:
        rc, m, e = orc.scan_workload(w, first, count)
        assert rc == 0
        parts_m.append(m)
        parts_e.append(e)
    assert np.array_equal(np.concatenate(parts_m), mean)
    assert np.array_equal(np.concatenate(parts_e), err)
    rc, m, e = orc.points_workload(w, [62, 0, 62, 17])
    assert np.array_equal(m, mean[[62, 0, 62, 17]]) and np.array_equal(e, err[[62, 0, 62, 17]])


def test_prefix_property():
    # an estimate with n samples uses exactly the first n*N words: g_s of a longer run extend a shorter one
    w = wl.config(5, scale=[2, 2, 2, 2, 2])
    for t in (0, 13, 31):
        _, g_long = orc.samples(w.integrand_id, w.bounds, w.lists, 40, w.seed, t, w.precision, w.consts)
        _, g_short = orc.samples(w.integrand_id, w.bounds, w.lists, 11, w.seed, t, w.precision, w.consts)
        assert np.array_equal(g_long[:11], g_short)


def test_points_are_independent_streams():
    # Q4: different grid points never share samples (keyed by t) -> lin_y means differ
    rc, mean, _ = orc.scan(wl.D_LIN_Y, [0.0, 1.0], [np.arange(6.0)], 8, 1, consts=[0.0])
    assert len(set(mean.tolist())) == 6


# ---- T6 -----------------------------------------------------------------------------------
def test_worked_example_n4():
    rows = _rows("worked_example.txt")
    lists = [np.array([0.1, 10.0])]
    rc, mean, err = orc.scan(wl.C1_COS_XY, [0.0, 1.0], lists, 4, 1)
    assert rc == 0
    for r in rows:
        t = int(r[0])
        words = [int(h, 16) for h in r[1:5]]
        assert [orc.word(1, t, s) for s in range(4)] == words
        if r[5] != "-":
            for s in range(4):
                assert abs(orc.uniform(words[s], orc.MODE_F64) - float(r[5 + s])) <= 1e-16
        assert abs(mean[t] - float(r[9])) <= 2e-15
        assert abs(err[t] - float(r[10])) <= 2e-15


# ---- Q18: argument checks -----------------------------------------------------------------
def test_oracle_rejects_degenerate_input():
    ok = dict(bounds=[0.0, 1.0], lists=[np.array([1.0, 2.0])], n_samples=4, seed=1)
    assert orc.scan(1, **ok)[0] == 0
    assert orc.scan(1, [1.0, 1.0], ok["lists"], 4, 1)[0] == 1          # a >= b
    assert orc.scan(1, [0.0, np.nan], ok["lists"], 4, 1)[0] == 1
    assert orc.scan(1, [0.0, 1.0], [np.array([1.0, np.inf])], 4, 1)[0] == 1
    assert orc.scan(1, [0.0, 1.0], ok["lists"], 1, 1)[0] == 1           # n < 2
    assert orc.scan(77, [0.0, 1.0], ok["lists"], 4, 1)[0] == 2          # unknown family
    assert orc.scan(2, [0.0, 1.0], ok["lists"], 4, 1)[0] == 3           # shape mismatch
    assert orc.scan(1, [0.0, 1.0], ok["lists"], 4, 1, first_index=1, count=2)[0] == 1
