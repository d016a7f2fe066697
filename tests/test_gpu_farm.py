"""-m gpu: NEXT-2, the single-node batch farm (Table 2).  One GPU is visible here, so the farm is
driven with device lists [0] and [0, 0] (two feeder threads on the one GPU: they share nothing but the batch counter
and never wait on each other's kernels).  The result must be bit-identical to a one-call scan with the same schedule,
whichever feeder took which batch."""
import os

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
NT = min(16, os.cpu_count() or 1)


@pytest.mark.parametrize("devices", [[0], [0, 0], [0, 0, 0]])
@pytest.mark.parametrize("cfg", [2, 5])
def test_farm_is_bit_identical_to_a_single_scan(cfg, devices):
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(cfg, scale={2: [37, 41], 5: [5, 4, 3, 6, 7]}[cfg], n_samples=300)
    w.host_out, w.batch_points = False, 0
    for sched in (1, 2):
        ref_m, ref_e = run_gpu(w, schedule=sched)
        dt = torch.float32 if w.out_f32 else torch.float64
        m = torch.full((w.G,), float("nan"), dtype=dt).pin_memory()
        e = torch.full((w.G,), float("nan"), dtype=dt).pin_memory()
        tm = zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, devices, precision=w.precision,
                              schedule=sched, batch_points=97, consts=w.consts)
        assert tm["n_batches"] == -(-w.G // 97) and sum(tm["batches_done"]) == tm["n_batches"]
        assert tm["n_devices"] == len(devices)
        assert np.array_equal(m.numpy(), ref_m) and np.array_equal(e.numpy(), ref_e)


def test_farm_default_batching_subrange_and_oracle_parity():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(3, scale=[13, 11, 17], n_samples=500)
    first, count = 101, 2003
    rc, mean_o, err_o = orc.scan_workload(w, first, count, n_threads=NT)
    assert rc == 0
    m = torch.empty(count, dtype=torch.float64).pin_memory()
    e = torch.empty(count, dtype=torch.float64).pin_memory()
    tm = zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, [0, 0], precision=w.precision,
                          first_index=first, count=count, consts=w.consts)
    assert tm["n_batches"] == 16 and tm["batch_points"] == -(-count // 16)      # about 8 batches per device
    assert_parity(w, m.numpy(), e.numpy(), mean_o, err_o)


def test_farm_argument_errors():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(1, scale=[8], n_samples=10)
    m = torch.full((8,), -1.0, dtype=torch.float64).pin_memory()
    e = m.clone().pin_memory()
    for devices in ([], [7], [-1], list(range(17))):
        with pytest.raises((zb.ZmcError, ValueError)):
            zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, devices)
    with pytest.raises(zb.ZmcError):
        zb.zmc_scan_farm(w.integrand_id, w.bounds, w.lists, 1, w.seed, m, e, [0])     # n_samples < 2
    assert torch.all(m == -1.0) and torch.all(e == -1.0)
