"""Closed forms of the integrand families (exact integral f and second moment E[g^2]).

Independent of both the oracle and the CUDA path: plain numpy/scipy expressions of the
integrals of SURVEY.md 8(c) row "Integrand families" (BASELINE.json configs 1-5) and of the
paper's Eq. (2)/(4) ("the theoretical value of this integration can be
obtained directly").  All take the grid as arrays of parameter values
(broadcastable) and return the integral over the box, NOT divided by the volume.
"""
from __future__ import annotations

import numpy as np
from scipy import integrate, special


def grid_params(lists):
    """Row-major (last fastest) flattening of the Cartesian product -> M flat arrays."""
    mesh = np.meshgrid(*lists, indexing="ij")
    return [m.reshape(-1) for m in mesh]


# ---- c1: cos(x1*y), y in [0,1] ------------------------------------------------------------
def c1_mean(x1):
    return np.sin(x1) / x1


def c1_m2(x1):          # E[g^2] (V = 1)
    return 0.5 + np.sin(2 * x1) / (4 * x1)


# ---- c2: sin(x1*y1 + x2*y2), y in [0,pi]^2 ------------------------------------------------
def _S(x, b):
    return (1 - np.cos(b * x)) / x


def _C(x, b):
    return np.sin(b * x) / x


def c2_mean(x1, x2, b=np.pi):
    return _S(x1, b) * _C(x2, b) + _C(x1, b) * _S(x2, b)


def c2_m2(x1, x2, b=np.pi):
    # sin^2 = (1 - cos 2arg)/2 ; int cos(2arg) = Re prod (e^{2ibx}-1)/(2ix)
    re = _C(2 * x1, b) * _C(2 * x2, b) - _S(2 * x1, b) * _S(2 * x2, b)
    return (0.5 * b * b - 0.5 * re) / (b * b)


# ---- c3: cos(2 pi u + sum_k c_k y_k), y in [0,1]^N, c_k = x_{(k mod 3)+1}*(k+1) -----------
def c3_coeffs(xs, N):
    return [xs[k % 3] * (k + 1) for k in range(N)]


def c3_mean(xs, N, u):
    c = c3_coeffs(xs, N)
    out = np.cos(2 * np.pi * u + 0.5 * sum(c))
    for ck in c:
        out = out * np.sin(ck / 2) / (ck / 2)
    return out


def c3_m2(xs, N, u):
    c = c3_coeffs(xs, N)
    prod = np.cos(4 * np.pi * u + sum(c))
    for ck in c:
        prod = prod * np.sin(ck) / ck
    return 0.5 + 0.5 * prod


# ---- c4: exp(-a^2 sum (y_k - w_k)^2), y in [0,1]^6 -----------------------------------------
def _gauss1d(a, w):
    return np.sqrt(np.pi) / (2 * a) * (special.erf(a * (1 - w)) + special.erf(a * w))


def c4_mean(a, w1, w2, w3):
    return (_gauss1d(a, w1) * _gauss1d(a, w2) * _gauss1d(a, w3)) ** 2


def c4_m2(a, w1, w2, w3):
    return c4_mean(np.sqrt(2.0) * a, w1, w2, w3)


def _gauss1d_box(a, w, lo, hi):
    """int_lo^hi exp(-a^2 (y - w)^2) dy."""
    return np.sqrt(np.pi) / (2 * a) * (special.erf(a * (hi - w)) - special.erf(a * (lo - w)))


def c4_mean_box(a, w1, w2, w3, bounds):
    """c4 over a general box: dimensions 0,1 centre on w1 (= x2), 2,3 on w2 (= x3), 4,5 on w3 (= x4)."""
    b = np.asarray(bounds, dtype=np.float64).reshape(6, 2)
    out = 1.0
    for k, w in enumerate((w1, w1, w2, w2, w3, w3)):
        out = out * _gauss1d_box(a, w, b[k, 0], b[k, 1])
    return out


# ---- c5: exp(-x1 |y|^2) cos(x2 y1 + x3 y2 + x4 y3) (1 + x5 y1 y2 y3), y in [-1,1]^3 -------
def J(alpha, c):
    """int_{-1}^{1} exp(-alpha y^2) cos(c y) dy via the complex error function."""
    alpha = np.asarray(alpha, dtype=np.float64)
    c = np.asarray(c, dtype=np.float64)
    sa = np.sqrt(alpha)
    z = sa + 1j * c / (2 * sa)
    return np.real(np.sqrt(np.pi / alpha) * np.exp(-c * c / (4 * alpha)) * special.erf(z))


def J_quad(alpha, c):
    val, _ = integrate.quad(lambda y: np.exp(-alpha * y * y) * np.cos(c * y), -1, 1, epsabs=1e-14, epsrel=1e-14)
    return val


def c5_mean(x1, x2, x3, x4, x5=None):
    # the x5 term is odd in every y_k and integrates to zero
    return J(x1, x2) * J(x1, x3) * J(x1, x4)


def _K2(alpha, c):
    """int_{-1}^{1} y^2 exp(-alpha y^2) cos(c y) dy (scalar, quadrature)."""
    val, _ = integrate.quad(lambda y: y * y * np.exp(-alpha * y * y) * np.cos(c * y), -1, 1,
                            epsabs=1e-14, epsrel=1e-14)
    return val


def c5_m2_scalar(x1, x2, x3, x4, x5):
    """E[g^2] at one parameter point (V = 8)."""
    a2 = 2 * x1
    t0 = 0.5 * (J_quad(a2, 0.0) ** 3 + J_quad(a2, 2 * x2) * J_quad(a2, 2 * x3) * J_quad(a2, 2 * x4))
    t2 = 0.5 * (_K2(a2, 0.0) ** 3 + _K2(a2, 2 * x2) * _K2(a2, 2 * x3) * _K2(a2, 2 * x4))
    return (t0 + x5 * x5 * t2) / 8.0


def _c5_1d(alpha, c, lo, hi, power):
    """int_lo^hi y^power exp(-alpha y^2 + i c y) dy (complex, quadrature)."""
    re, _ = integrate.quad(lambda y: y ** power * np.exp(-alpha * y * y) * np.cos(c * y), lo, hi, epsabs=1e-14, epsrel=1e-13)
    im, _ = integrate.quad(lambda y: y ** power * np.exp(-alpha * y * y) * np.sin(c * y), lo, hi, epsabs=1e-14, epsrel=1e-13)
    return complex(re, im)


def c5_mean_box_scalar(x1, x2, x3, x4, x5, bounds):
    """c5 over a general box (one parameter point): cos(sum c_k y_k) = Re prod exp(i c_k y_k), so
    f = Re prod_k A_k + x5 Re prod_k B_k with A_k = int exp(-x1 y^2 + i c_k y), B_k = int y exp(-x1 y^2 + i c_k y).
    On a box that is not symmetric about 0 the x5 term does NOT vanish: the mean sees x5 and its sign."""
    b = np.asarray(bounds, dtype=np.float64).reshape(3, 2)
    A = B = 1.0 + 0.0j
    for k, c in enumerate((x2, x3, x4)):
        A *= _c5_1d(x1, c, b[k, 0], b[k, 1], 0)
        B *= _c5_1d(x1, c, b[k, 0], b[k, 1], 1)
    return A.real + x5 * B.real


# ---- p6: the paper's sin(sum y + sum x) on [0,b]^N ---------------------
def p6_mean(xsum, N, b):
    return (2 * np.sin(b / 2)) ** N * np.sin(xsum + N * b / 2)


def p6_m2(xsum, N, b):
    # sin^2 = (1 - cos 2arg)/2 ; int_[0,b]^N cos(2 sum y + 2 xsum) = (sin b)^N cos(2 xsum + N b)
    return (0.5 * b ** N - 0.5 * np.sin(b) ** N * np.cos(2 * xsum + N * b)) / b ** N


def exact_for_workload(w):
    """(exact integral, E[g^2] or None) over the whole grid of a workloads.Workload."""
    xs = grid_params(w.lists)
    fid = w.integrand_id
    if fid == 1:
        return c1_mean(xs[0]), c1_m2(xs[0])
    if fid == 2:
        return c2_mean(xs[0], xs[1]), c2_m2(xs[0], xs[1])
    if fid == 3:
        return c3_mean(xs, w.N, float(w.consts[0])), c3_m2(xs, w.N, float(w.consts[0]))
    if fid == 4:
        return c4_mean(*xs), c4_m2(*xs)
    if fid == 5:
        return c5_mean(*xs), None
    if fid == 6:
        b = float(w.bounds[1])
        xsum = sum(xs)
        return p6_mean(xsum, w.N, b), p6_m2(xsum, w.N, b)
    raise ValueError(fid)
