"""-m gpu: NEXT-3, user-defined integrands compiled with NVRTC, against the CPU oracle evaluating the SAME body text
(compiled with gcc, R = double) on the same sample stream -- same tolerances as the built-in families."""
import os

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
NT = min(16, os.cpu_count() or 1)

CASES = {
    # name: (body, bounds, lists, consts, n)
    "damped_cos": ("return exp(-x[0] * y[0] * y[0]) * cos(x[1] * y[1] + c[0]);",
                   [0.0, 1.0, 0.0, 2.0], [wl.linspace(0.2, 3.0, 13), wl.linspace(0.5, 4.0, 11)], [0.3], 1003),
    "rational_3d": ("R d = (R)1 + x[0] * (y[0] * y[0] + y[1] * y[1] + y[2] * y[2]); return y[0] * y[1] / (d * d) + x[1];",
                    [-1.0, 1.0, 0.0, 2.0, 0.5, 1.5], [wl.linspace(0.1, 2.0, 7), wl.linspace(-1.0, 1.0, 5)], [], 517),
    "sum_11d": ("R s = x[0]; for (int k = 0; k < 11; ++k) s += y[k] * (R)(k + 1); return sin(s) * c[1] + c[0];",
                [0.0, 0.25] * 11, [wl.linspace(0.0, 3.0, 9)], [0.5, 2.0], 259),
}


def _workload(name, uid, precision):
    body, bounds, lists, consts, n = CASES[name]
    return wl.Workload(name, uid, np.array(bounds), [np.asarray(l, dtype=np.float64) for l in lists], n, 21, precision,
                       np.array(consts, dtype=np.float64))


@pytest.mark.parametrize("precision", [wl.PREC_F64, wl.PREC_F32E])
@pytest.mark.parametrize("name", sorted(CASES))
def test_user_integrand_parity_all_schedules(name, precision):
    from paper_1910_01965_b200 import binding as zb
    body, bounds, lists, consts, n = CASES[name]
    uid = zb.zmc_register_integrand(name, body, len(bounds) // 2, len(lists), len(consts))
    assert uid >= 1000
    orc.set_user_integrand(body, len(bounds) // 2, len(lists), len(consts))
    w = _workload(name, uid, precision)
    rc, mean_o, err_o = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    for sched in (1, 2, 3):
        mean, err = run_gpu(w, schedule=sched)
        assert_parity(w, mean, err, mean_o, err_o)
    # batch / sub-range invariance holds for user integrands too (same kernel template): bit-exact
    full, _ = run_gpu(w, schedule=1)
    part, _ = run_gpu(w, schedule=1, first_index=3, count=w.G - 5, batch_points=7)
    assert np.array_equal(part, full[3:w.G - 2])


def test_user_copy_of_a_builtin_family_matches_it():
    """The user body of cfg 2's integrand goes through the generic (unfolded) evaluation; the built-in family folds the
    affine map and uses its own sinpi: both must agree with the oracle, hence with each other, to the fp64 tolerance."""
    from paper_1910_01965_b200 import binding as zb
    uid = zb.zmc_register_integrand("c2_copy", "return sin(x[0] * y[0] + x[1] * y[1]);", 2, 2, 0)
    w = wl.config(2, scale=[19, 23], n_samples=2001)
    builtin, berr = run_gpu(w, schedule=2)
    w.integrand_id = uid
    user, uerr = run_gpu(w, schedule=2)
    assert np.all(np.abs(user - builtin) <= 1e-10 * np.maximum(np.abs(builtin), berr))
    assert np.all(np.abs(uerr - berr) <= 1e-10 * berr)


def test_user_shape_mismatch_and_unknown_id():
    import torch
    from paper_1910_01965_b200 import binding as zb
    uid = zb.zmc_register_integrand("one_d", "return y[0] * x[0];", 1, 1, 0)
    m = torch.zeros(4, dtype=torch.float64, device="cuda")
    with pytest.raises(zb.ZmcError) as ei:         # registered for N = 1, called with N = 2
        zb.zmc_scan_ex(uid, [0.0, 1.0, 0.0, 1.0], [np.arange(4.0)], 10, 1, m, m.clone())
    assert ei.value.status == zb.ZMC_ERR_SHAPE_MISMATCH
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_scan_ex(uid + 500, [0.0, 1.0], [np.arange(4.0)], 10, 1, m, m.clone())
    assert ei.value.status == zb.ZMC_ERR_UNKNOWN_INTEGRAND


HELPER_BODY = ("return zmc_sin(x[0] * y[0]) * zmc_cos(x[1] * y[1] + c[0]) + zmc_sinpi(y[0] - x[1]) * zmc_cospi(x[0] * y[1]) "
               "+ zmc_exp(-x[0] * y[1] * y[1]) - zmc_exp2(-y[0]);")


@pytest.mark.parametrize("precision,flags", [(wl.PREC_F64, 0), (wl.PREC_F32E, 0), (wl.PREC_F32E, 1), (wl.PREC_F64, 1)])
def test_library_transcendentals_in_user_bodies(precision, flags):
    """zmc_sin / zmc_cos / zmc_sinpi / zmc_cospi / zmc_exp / zmc_exp2 (include/zmc.h) against the oracle evaluating their
    plain definitions; with ZMC_USER_FAST_MATH the fp32 versions are the MUFU forms (same tolerance as the built-in families)."""
    from paper_1910_01965_b200 import binding as zb
    uid = zb.zmc_register_integrand("helpers", HELPER_BODY, 2, 2, 1, flags=flags)
    orc.set_user_integrand(HELPER_BODY, 2, 2, 1)
    w = wl.Workload("helpers", uid, np.array([0.0, 2.0, -1.0, 1.5]), [wl.linspace(0.3, 9.0, 12), wl.linspace(-2.0, 4.0, 9)],
                    1501, 33, precision, np.array([0.4]))
    rc, mean_o, err_o = orc.scan_workload(w, n_threads=NT)
    assert rc == 0
    for sched in (1, 2, 3):
        mean, err = run_gpu(w, schedule=sched)
        assert_parity(w, mean, err, mean_o, err_o)


def test_registration_is_cached_by_content_and_can_be_undone():
    """SURVEY.md 8(f) NEXT-3 "cache by hash": the same (body, N, M, n_consts, flags) is the same id and costs no compile."""
    import time
    import torch
    from paper_1910_01965_b200 import binding as zb
    body = "return x[0] * y[0] * y[0] + 0.125;"          # nothing else in the suite registers this one
    t0 = time.perf_counter()
    uid = zb.zmc_register_integrand("cached", body, 1, 1, 0)
    t_first = time.perf_counter() - t0
    t0 = time.perf_counter()
    again = zb.zmc_register_integrand("another name, same integrand", body, 1, 1, 0)
    t_again = time.perf_counter() - t0
    assert again == uid and t_again < 1e-3 < t_first
    assert zb.zmc_register_integrand("cached", body, 1, 1, 0, flags=zb.ZMC_USER_FAST_MATH) != uid      # other flags: other code
    assert zb.zmc_register_integrand("cached", body + " ", 1, 1, 0) != uid
    m = torch.zeros(3, dtype=torch.float64, device="cuda")
    e = torch.zeros_like(m)
    zb.zmc_scan_ex(uid, [0.0, 1.0], [np.array([1.0, 2.0, 3.0])], 64, 1, m, e)
    torch.cuda.synchronize()
    assert torch.all(m > 0.125)
    zb.zmc_unregister_integrand(uid)                     # registered twice above: registrations are counted ...
    zb.zmc_scan_ex(uid, [0.0, 1.0], [np.array([1.0, 2.0, 3.0])], 64, 1, m, e)
    zb.zmc_unregister_integrand(uid)                     # ... and the second unregister drops the id
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_scan_ex(uid, [0.0, 1.0], [np.array([1.0, 2.0, 3.0])], 64, 1, m, e)
    assert ei.value.status == zb.ZMC_ERR_UNKNOWN_INTEGRAND
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_unregister_integrand(uid)
    assert ei.value.status == zb.ZMC_ERR_UNKNOWN_INTEGRAND
    fresh = zb.zmc_register_integrand("cached", body, 1, 1, 0)          # compiled again, ids are never reused
    assert fresh != uid


def test_an_id_registered_twice_survives_the_first_unregister():
    """Two parts of a program register the same body and get the same id; one of them unregistering must not pull the
    code from under the other (include/zmc.h, zmc_unregister_integrand: registrations are counted)."""
    from paper_1910_01965_b200 import binding as zb
    body = "return exp(-x[0] * y[0]) + c[0] * y[1];"
    first = zb.zmc_register_integrand("owner_a", body, 2, 1, 1)
    second = zb.zmc_register_integrand("owner_b", body, 2, 1, 1)
    assert first == second
    w = wl.Workload("shared", first, np.array([0.0, 1.0, 0.0, 2.0]), [wl.linspace(0.1, 2.0, 17)], 301, 4, wl.PREC_F64,
                    np.array([0.75]))
    before, before_err = run_gpu(w, schedule=2)
    zb.zmc_unregister_integrand(first)                 # owner_a is done with it
    after, after_err = run_gpu(w, schedule=2)          # owner_b still scans
    assert np.array_equal(before, after) and np.array_equal(before_err, after_err)
    zb.zmc_unregister_integrand(second)
    with pytest.raises(zb.ZmcError) as exc:
        run_gpu(w, schedule=2)
    assert exc.value.status == zb.ZMC_ERR_UNKNOWN_INTEGRAND
    with pytest.raises(zb.ZmcError):
        zb.zmc_unregister_integrand(second)


def test_unregister_right_after_an_enqueue_only_scan():
    """zmc_scan_ex only enqueues; unregistering the integrand before the kernels have run must wait for them instead of
    unloading code that is still executing."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    body = "R s = x[0]; for (int k = 0; k < 3; ++k) s += y[k] * x[1]; return cos(s);"
    w = wl.Workload("inflight", 0, np.array([0.0, 1.0] * 3), [wl.linspace(0.1, 2.0, 400), wl.linspace(0.5, 1.5, 300)],
                    4000, 8, wl.PREC_F64, np.zeros(0))
    w.integrand_id = zb.zmc_register_integrand("inflight", body, 3, 2, 0)
    ref, ref_err = run_gpu(w, schedule=1)
    mean = torch.zeros(w.G, dtype=torch.float64, device="cuda")
    err = torch.zeros_like(mean)
    zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, schedule=1)    # ~10 ms of GPU work, not waited for
    zb.zmc_unregister_integrand(w.integrand_id)
    torch.cuda.synchronize()
    assert np.array_equal(mean.cpu().numpy(), ref) and np.array_equal(err.cpu().numpy(), ref_err)
    with pytest.raises(zb.ZmcError):
        run_gpu(w, schedule=1)
