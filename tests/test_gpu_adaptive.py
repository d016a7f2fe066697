"""-m gpu: NEXT-4, per-point adaptive sample count (zmc_scan_adaptive; PAPER.md:116 leaves the choice of the sample
count to the user).  What is unique is checked exactly: the outputs at the n the kernel stopped at are bit-identical
to a fixed-n WARP-schedule scan with that n (prefix property) and agree with the CPU oracle's fixed-n estimate; the
stopping decision itself is a floating-point comparison, so it is checked for validity with the oracle's own standard
errors and a tolerance band around the target (a point within the band may legitimately stop one checkpoint apart)."""
import os

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
NT = min(16, os.cpu_count() or 1)


def adaptive(w, n_first, n_max, target, **kw):
    import torch
    from paper_1910_01965_b200 import binding as zb
    count = kw.get("count", 0) or w.G - kw.get("first_index", 0)
    dt = torch.float32 if w.out_f32 else torch.float64
    m = torch.empty(count, dtype=dt, device="cuda")
    e = torch.empty(count, dtype=dt, device="cuda")
    n = torch.zeros(count, dtype=torch.int32, device="cuda")
    zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, m, e, n,
                         precision=w.precision, consts=w.consts, **kw)
    torch.cuda.synchronize()
    return m.cpu().numpy(), e.cpu().numpy(), n.cpu().numpy().astype(np.int64)


@pytest.mark.parametrize("cfg,scale,target", [(2, [23, 19], 0.06), (3, [7, 6, 5], 0.012), (4, [4, 5, 3, 4], 2e-3),
                                              (5, [3, 4, 3, 3, 4], 0.04)])
def test_adaptive_matches_fixed_n_scan_and_oracle(cfg, scale, target):
    w = wl.config(cfg, scale=scale)
    w.out_f32, w.host_out, w.batch_points = False, False, 0
    n_first, n_max = 256, 256 * 64 + 8 * 5                     # n_max deliberately not a power-of-two multiple
    mean, err, n_used = adaptive(w, n_first, n_max, target)
    checkpoints = [min(n_first << k, n_max) for k in range(8)]
    assert set(np.unique(n_used)) <= set(checkpoints)
    assert len(np.unique(n_used)) >= 3, "the target should make different grid points stop at different checkpoints"
    for n in np.unique(n_used):
        sel = np.nonzero(n_used == n)[0]
        w.n_samples = int(n)
        fm, fe = run_gpu(w, schedule=2)                         # fixed-n scan, WARP schedule
        assert np.array_equal(mean[sel], fm[sel]) and np.array_equal(err[sel], fe[sel])      # bit-identical
        rc, mo, eo = orc.points_workload(w, sel.astype(np.uint64), n_threads=NT)
        assert rc == 0
        assert_parity(w, mean[sel], err[sel], mo, eo)
        # validity of the decision, judged with the oracle's numbers: stopped => small enough (or out of budget) ...
        band = 1e-9 if w.precision == wl.PREC_F64 else 2e-4
        assert np.all((eo <= target * (1 + band)) | (n == n_max))
        # ... and not stopped earlier => the previous checkpoint was still too large
        if n > n_first:
            prev = max(c for c in checkpoints if c < n)
            w.n_samples = prev
            rc, _, eprev = orc.points_workload(w, sel.astype(np.uint64), n_threads=NT)
            assert np.all(eprev > target * (1 - band))


def test_adaptive_limits_batches_and_subranges():
    w = wl.config(1, scale=[64])
    # target 0: never satisfied -> every point runs to n_max; huge target: every point stops at n_first
    _, e_all, n_all = adaptive(w, 512, 4096, 0.0)
    assert np.all(n_all == 4096)
    _, _, n_one = adaptive(w, 512, 4096, 1e9)
    assert np.all(n_one == 512)
    # batching and sub-ranges do not change anything (global-index keyed), n_first == n_max is a plain fixed-n scan
    m0, e0, n0 = adaptive(w, 256, 8192, 2e-3)
    m1, e1, n1 = adaptive(w, 256, 8192, 2e-3, first_index=5, count=50, batch_points=7)
    assert np.array_equal(m1, m0[5:55]) and np.array_equal(e1, e0[5:55]) and np.array_equal(n1, n0[5:55])
    mf, ef, nf = adaptive(w, 1024, 1024, 1e-12)
    w.n_samples = 1024
    fm, fe = run_gpu(w, schedule=2)
    assert np.array_equal(mf, fm) and np.array_equal(ef, fe) and np.all(nf == 1024)


def test_adaptive_user_integrand():
    from paper_1910_01965_b200 import binding as zb
    body = "return exp(-x[0] * y[0] * y[0]) * cos(x[1] * y[1] + c[0]);"
    uid = zb.zmc_register_integrand("adaptive_user", body, 2, 2, 1)
    w = wl.Workload("u", uid, np.array([0.0, 1.0, 0.0, 2.0]), [wl.linspace(0.2, 3.0, 9), wl.linspace(0.5, 4.0, 8)], 256, 5,
                    wl.PREC_F64, np.array([0.3]))
    mean, err, n_used = adaptive(w, 256, 8192, 0.01)
    assert len(np.unique(n_used)) >= 2
    orc.set_user_integrand(body, 2, 2, 1)
    for n in np.unique(n_used):
        sel = np.nonzero(n_used == n)[0]
        w.n_samples = int(n)
        fm, fe = run_gpu(w, schedule=2)      # bit-identical to the fixed-n WARP scan for NVRTC-compiled integrands too:
        assert np.array_equal(mean[sel], fm[sel]) and np.array_equal(err[sel], fe[sel])    # g - K is never contracted
        rc, mo, eo = orc.points_workload(w, sel.astype(np.uint64), n_threads=NT)
        assert rc == 0
        assert_parity(w, mean[sel], err[sel], mo, eo)


def test_adaptive_argument_errors():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(1, scale=[8])
    m = torch.full((8,), -1.0, dtype=torch.float64, device="cuda")
    e = m.clone()
    n = torch.zeros(8, dtype=torch.int32, device="cuda")
    for n_first, n_max, target in [(100, 1024, 0.1), (255, 1024, 0.1), (256, 128, 0.1), (256, 1001, 0.1), (256, 1024, -1.0),
                                   (256, 1024, float("nan")), (256, 1 << 33, 0.1)]:
        with pytest.raises(zb.ZmcError) as ei:
            zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, m, e, n)
        assert ei.value.status == zb.ZMC_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert torch.all(m == -1.0) and torch.all(n == 0)


def test_adaptive_streams_to_pinned_host_and_through_the_farm():
    """zmc_scan_adaptive with ZMC_LOC_HOST outputs (out_n streamed with the results, batch by batch) and
    zmc_scan_farm_adaptive, on a 1.2 * 10^8-point sub-range of cfg 5's 10^10 grid cut into batches: bit-identical to the
    device-output call on the same range, which the other tests pin to the fixed-n scan and the oracle."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(5)
    first, count, bp = (1 << 32) - 7_000_001, 120_000_000, 1 << 25         # straddles 2^32; 4 batches, the last one ragged
    n_first, n_max, target = 256, 512, 0.11
    dm = torch.empty(count, dtype=torch.float32, device="cuda")
    de = torch.empty_like(dm)
    dn = torch.zeros(count, dtype=torch.int32, device="cuda")
    zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, dm, de, dn,
                         precision=w.precision, first_index=first, count=count)
    hm = torch.empty(count, dtype=torch.float32, pin_memory=True)
    he = torch.empty_like(hm).pin_memory()
    hn = torch.zeros(count, dtype=torch.int32).pin_memory()
    tm = zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, hm, he, hn,
                              precision=w.precision, first_index=first, count=count, batch_points=bp, timing=True)
    torch.cuda.synchronize()
    assert tm["n_batches"] == 4 and tm["host_out_pinned"] == 1 and tm["d2h_bytes"] == count * 12
    assert torch.equal(hm, dm.cpu()) and torch.equal(he, de.cpu()) and torch.equal(hn, dn.cpu())
    frac = float((hn == n_max).float().mean())
    assert 0.02 < frac < 0.98, "the target should split the points between the two checkpoints"
    # the same through the farm (feeder threads on the one visible device)
    fm, fe, fn = torch.empty_like(hm).pin_memory(), torch.empty_like(hm).pin_memory(), torch.zeros_like(hn).pin_memory()
    ft = zb.zmc_scan_farm_adaptive(w.integrand_id, w.bounds, w.lists, n_first, n_max, target, w.seed, fm, fe, fn, [0, 0],
                                   precision=w.precision, first_index=first, count=count, batch_points=bp)
    assert ft["n_batches"] == 4 and sum(ft["batches_done"]) == 4
    assert torch.equal(fm, hm) and torch.equal(fe, he) and torch.equal(fn, hn)
    # oracle spot check on sampled points of each checkpoint population
    rng = np.random.default_rng(5)
    n_np = hn.numpy()
    for n in (n_first, n_max):
        sel = rng.choice(np.nonzero(n_np == n)[0], 200, replace=False)
        w.n_samples = n
        rc, mo, eo = orc.points_workload(w, (sel + first).astype(np.uint64), n_threads=NT)
        assert rc == 0
        assert_parity(w, hm.numpy()[sel].astype(np.float64), he.numpy()[sel].astype(np.float64), mo, eo)
