"""T7: the oracle against the closed forms of every family (CPU-only).

north_star acceptance: |estimate - exact| <= 5*stderr at >= 99.9 % of grid points (reading Q13:
for c4 on the points with effective sample size n_eff = n E[g]^2/E[g^2] >= 30); plus z-score
moments (catches a mis-scaled stderr) and the stderr scale against the closed-form E[g^2].
Grids are reduced copies of BASELINE.json configs 1-5 (same ranges, fewer list entries) so the
CPU suite stays within minutes; cfg 1 runs at full size.
"""
import os

import numpy as np
import pytest

import closed_forms as cf
from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl

NT = min(8, os.cpu_count() or 1)


def _volume(w):
    b = np.asarray(w.bounds).reshape(-1, 2)
    return float(np.prod(b[:, 1] - b[:, 0]))


def _check(w, gate=None, cov=0.999, zvar_tol=None, scale_tol=0.03, min_frac=0.2):
    rc, mean, err = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    exact, m2 = cf.exact_for_workload(w)
    V = _volume(w)
    sel = np.ones(len(mean), bool) if gate is None else gate(exact / V, m2)
    assert sel.sum() >= min_frac * len(mean)
    z = (mean[sel] - exact[sel]) / err[sel]
    P = sel.sum()
    assert np.mean(np.abs(z) <= 5.0) >= cov
    assert abs(z.mean()) <= 4.0 / np.sqrt(P)
    tol = zvar_tol if zvar_tol is not None else 6.0 * np.sqrt(2.0 / P)
    assert abs(z.var() - 1.0) <= tol
    if m2 is not None:
        var_g = m2 - (exact / V) ** 2
        ok = sel & (var_g > 1e-12)
        ratio = w.n_samples * err[ok] ** 2 / (V * V * var_g[ok])
        assert abs(ratio.mean() - 1.0) <= scale_tol
    return mean, err, exact


def test_cfg1_full_size():
    _check(wl.config(1))


def test_cfg2_reduced():
    _check(wl.config(2, scale=[60, 60]))


def test_cfg3_reduced():
    _check(wl.config(3, scale=[20, 20, 20]))


def test_cfg3_other_N_and_u():
    w = wl.config(3, scale=[6, 6, 6], n_samples=3000)
    w.bounds = np.array([0.0, 1.0] * 5)
    w.consts = np.array([0.6])
    _check(w)


def test_cfg4_gated_by_effective_sample_size():
    w = wl.config(4, scale=[20, 8, 8, 8])

    def gate(mean_g, m2):
        return w.n_samples * mean_g ** 2 / m2 >= 30.0
    _check(w, gate=gate, cov=0.998, zvar_tol=0.5, scale_tol=0.2, min_frac=0.1)


def test_cfg4_gentle_setting_all_points():
    # Q13: validate the family once where every point qualifies (a in [1,3])
    w = wl.config(4, scale=[5, 6, 6, 6], n_samples=4000)
    w.lists[0] = wl.linspace(1.0, 3.0, 5)
    _check(w, zvar_tol=0.3, scale_tol=0.05)


def test_cfg5_reduced_and_x5_independence():
    w = wl.config(5, scale=[6, 6, 6, 6, 6])
    mean, err, exact = _check(w, cov=0.998, zvar_tol=0.2)
    # closed form cross-check: complex-erf J against quadrature
    for a, c in [(0.1, 0.1), (4.0, 4.0), (1.3, 2.9)]:
        assert abs(cf.J(a, c) - cf.J_quad(a, c)) <= 1e-13
    # stderr scale at a few points against the quadrature second moment
    xs = cf.grid_params(w.lists)
    rng = np.random.default_rng(0)
    idx = rng.choice(len(mean), 40, replace=False)
    ratios = []
    for t in idx:
        m2 = cf.c5_m2_scalar(*[float(x[t]) for x in xs])
        var_g = m2 - (exact[t] / 8.0) ** 2
        ratios.append(w.n_samples * err[t] ** 2 / (64.0 * var_g))
    assert abs(np.mean(ratios) - 1.0) <= 0.1


def test_c4_asymmetric_box_pins_which_parameter_centres_which_dimensions():
    # on [0,1]^6 the integral is symmetric in x2, x3, x4, so the closed form cannot see WHICH
    # dimensions centre on which parameter.  Box [0,1]^4 x [0,0.5]^2 and different ranges for x3 and x4 break the symmetry
    # (BASELINE.json configs[3]: w_k = x2 for k<2, x3 for 2<=k<4, x4 for k>=4).
    bounds = np.array([0.0, 1.0, 0.0, 1.0, 0.0, 1.0, 0.0, 1.0, 0.0, 0.5, 0.0, 0.5])
    lists = [wl.linspace(1.0, 3.0, 4), wl.linspace(0.1, 0.9, 3), wl.linspace(0.55, 0.95, 4), wl.linspace(0.05, 0.3, 4)]
    w = wl.Workload("c4_asym", wl.C4_GAUSS_PEAK, bounds, lists, 20000, 44, wl.PREC_F64, np.zeros(0))
    rc, mean, err = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    a, w1, w2, w3 = cf.grid_params(lists)
    exact = cf.c4_mean_box(a, w1, w2, w3, bounds)
    z = (mean - exact) / err
    assert np.all(np.abs(z) <= 5.0) and abs(z.mean()) <= 4.0 / np.sqrt(len(z)) and abs(z.var() - 1.0) <= 0.45
    # the test has teeth: with x3 and x4 swapped the closed form is many sigma away at most points
    swapped = cf.c4_mean_box(a, w1, w3, w2, bounds)
    assert np.mean(np.abs((mean - swapped) / err) > 5.0) >= 0.9


def test_c5_asymmetric_box_mean_sees_x5_and_its_sign():
    # On [-1,1]^3 the (1 + x5 y0 y1 y2) factor integrates to 1 (oddness), so the cfg 5 closed form is blind to it.
    # On a box that is not symmetric about 0 it is not: f = Re prod A_k + x5 Re prod B_k (closed_forms.c5_mean_box_scalar).
    bounds = np.array([0.0, 1.0, -0.5, 1.0, 0.25, 1.5])
    lists = [np.array([0.3, 1.1]), np.array([0.7]), np.array([1.9]), np.array([0.4, 2.6]), np.array([-3.0, 0.8, 3.5])]
    w = wl.Workload("c5_asym", wl.C5_DAMPED_COS, bounds, lists, 40000, 55, wl.PREC_F64, np.zeros(0))
    rc, mean, err = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    xs = cf.grid_params(lists)
    far = 0
    for t in range(len(mean)):
        x = [float(v[t]) for v in xs]
        exact = cf.c5_mean_box_scalar(*x, bounds)
        assert abs(mean[t] - exact) <= 5.0 * err[t], (t, x)
        flipped = cf.c5_mean_box_scalar(x[0], x[1], x[2], x[3], -x[4], bounds)        # wrong sign of the x5 term
        wrong_par = cf.c5_mean_box_scalar(x[0], x[1], x[2], x[3], x[3], bounds)       # x4 used in place of x5
        far += int(abs(mean[t] - flipped) > 5.0 * err[t]) + int(abs(mean[t] - wrong_par) > 5.0 * err[t])
    assert far >= 1.5 * len(mean)        # teeth: both mutations are > 5 sigma away at (at least) three quarters of the points


def test_c5_second_moment_per_point_depends_on_x5():
    # cfg 5's own box: only x5 varies; n stderr^2 / V^2 = Var g must follow E[g^2] = (t0 + x5^2 t2)/8 POINT BY POINT
    # (a dropped y_k, x4 in place of x5, or a missing factor changes t2's weight; the band is 4 sampling sigma of the variance)
    w = wl.config(5, scale=[1, 1, 1, 1, 9], n_samples=200_000)
    w.lists[0] = np.array([0.35]); w.lists[1] = np.array([1.3]); w.lists[2] = np.array([0.6]); w.lists[3] = np.array([2.1])
    w.lists[4] = wl.linspace(0.1, 8.0, 9)
    w.precision = wl.PREC_F64
    rc, mean, err = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    x5s = w.lists[4]
    exact = float(cf.c5_mean(0.35, 1.3, 0.6, 2.1))
    got = w.n_samples * err ** 2 / 64.0
    want = np.array([cf.c5_m2_scalar(0.35, 1.3, 0.6, 2.1, float(x5)) for x5 in x5s]) - (exact / 8.0) ** 2
    assert np.all(np.abs(got / want - 1.0) <= 0.03), got / want
    assert want[-1] / want[0] > 2.0      # the x5 term dominates at the top of the list: a version without it fails by a factor
    assert np.all(np.abs(mean - exact) <= 5.0 * err)


@pytest.mark.parametrize("M,N", [(1, 1), (2, 3), (3, 2)])
def test_paper_eq2_family(M, N):
    # PAPER.md:73-77 Eq. (2) on [0,10]^N; lists {0..L-1}
    _check(wl.paper_eq2(M, N, n_samples=4000, L=12 if M > 1 else 100))


def test_paper_eq4_family_and_error_bound():
    # PAPER.md:118-130 Eq. (4); "relative error at each parameter grid is always smaller 0.2" is a
    # statement about the grid-averaged delta_r(x1,x2) of Eq. (5) -- loose sanity bound only.
    w = wl.paper_eq4(n_samples=20000, L=5)
    mean, err, exact = _check(w)
    dr = np.abs(exact - mean) / np.abs(exact)
    assert np.median(dr) < 0.2


def test_f32_mirror_mode_tracks_f64_mode():
    # mirror mode differs from F64 mode only by input rounding and the 23-bit lattice
    w = wl.config(3, scale=[5, 5, 5])
    rc, m32, e32 = orc.scan_workload(w, n_threads=NT)
    w.precision = wl.PREC_F64
    rc, m64, e64 = orc.scan_workload(w, n_threads=NT)
    assert np.max(np.abs(m32 - m64)) < 1e-5
    assert np.max(np.abs(e32 - e64)) < 1e-5
    assert not np.array_equal(m32, m64)
