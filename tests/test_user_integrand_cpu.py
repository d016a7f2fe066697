"""-m "not gpu": NEXT-3 (user-defined integrands) without a GPU.

NVRTC compiles without a device, so the compile step, its error reporting and the argument checks of
zmc_register_integrand are tested here; loading the compiled code needs a GPU (ZMC_ERR_CUDA on this box).
The oracle's user hook is pinned against a closed form.
"""
import numpy as np
import pytest
from scipy import special

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import binding as zb

BODY = "return exp(-x[0] * y[0] * y[0]) * cos(x[1] * y[1] + c[0]);"


def test_valid_body_compiles_for_sm_100a():
    try:
        uid = zb.zmc_register_integrand("damped", BODY, 2, 2, 1)
    except zb.ZmcError as exc:                     # no device here: compiled, but nothing to load it on
        assert exc.status == zb.ZMC_ERR_CUDA, str(exc)
        assert "cudaLibraryLoadData" in zb.zmc_last_compile_log()
    else:                                          # on a GPU box the registration goes through
        assert uid >= 1000


def test_compile_error_is_reported_with_the_nvrtc_log():
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_register_integrand("bad", "return no_such_function(y[0]);", 1, 1, 0)
    assert ei.value.status == zb.ZMC_ERR_COMPILE
    assert "no_such_function" in zb.zmc_last_compile_log()


@pytest.mark.parametrize("N,M,nc", [(0, 1, 0), (17, 1, 0), (1, 0, 0), (1, 9, 0), (1, 1, -1), (1, 1, 9)])
def test_register_argument_checks(N, M, nc):
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_register_integrand("x", "return y[0];", N, M, nc)
    assert ei.value.status == zb.ZMC_ERR_INVALID_ARG


def test_unregistered_user_id_is_unknown():
    st, _ = zb.zmc_validate(4242, [0.0, 1.0], [np.array([1.0])], 10)
    assert st == zb.ZMC_ERR_UNKNOWN_INTEGRAND


def test_oracle_user_hook_against_closed_form():
    """int_0^1 exp(-a y^2) dy * int_0^2 cos(b y + c) dy = sqrt(pi/a)/2 erf(sqrt a) * (sin(2b + c) - sin c)/b."""
    orc.set_user_integrand(BODY, 2, 2, 1)
    a = np.linspace(0.2, 3.0, 15)
    b = np.linspace(0.5, 4.0, 17)
    c = 0.3
    rc, mean, err = orc.scan(1000, [0.0, 1.0, 0.0, 2.0], [a, b], 4000, 12, orc.MODE_F64, np.array([c]), n_threads=4)
    assert rc == 0
    A, B = np.meshgrid(a, b, indexing="ij")
    exact = (np.sqrt(np.pi / A) / 2 * special.erf(np.sqrt(A)) * (np.sin(2 * B + c) - np.sin(c)) / B).reshape(-1)
    z = (mean - exact) / err
    assert np.all(np.abs(z) <= 5) and abs(z.mean()) < 4 / np.sqrt(len(z)) and 0.6 < z.var() < 1.5
    # shape other than the registered one is refused
    rc, _, _ = orc.scan(1000, [0.0, 1.0], [a], 100, 1)
    assert rc == 3
