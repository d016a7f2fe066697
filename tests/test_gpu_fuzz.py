"""-m gpu: seeded random configurations (family, dimensions, list lengths, sample count, seed, precision, schedule,
sub-range, batch size, output type and placement) against the CPU oracle.  The draw is deterministic (numpy
default_rng with a fixed seed per case), so a failure names a reproducible case."""
import os

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl
from test_gpu_parity import assert_parity

pytestmark = pytest.mark.gpu
NT = min(16, os.cpu_count() or 1)


def draw(case):
    rng = np.random.default_rng(1000 + case)
    fam = int(rng.choice([wl.C1_COS_XY, wl.C2_SIN_XY2, wl.C3_OSCILLATORY, wl.C4_GAUSS_PEAK, wl.C5_DAMPED_COS, wl.P6_SIN_SUM,
                          wl.D_LIN_Y, wl.D_POLY]))
    N, M = {wl.C1_COS_XY: (1, 1), wl.C2_SIN_XY2: (2, 2), wl.C4_GAUSS_PEAK: (6, 4), wl.C5_DAMPED_COS: (3, 5)}.get(fam, (0, 0))
    if fam == wl.C3_OSCILLATORY:
        N, M = int(rng.integers(1, 10)), 3
    if fam in (wl.P6_SIN_SUM, wl.D_LIN_Y, wl.D_POLY):
        N, M = int(rng.integers(1, 10)), int(rng.integers(1, 5))
    lo = rng.uniform(-1.0, 0.5, N)
    bounds = np.stack([lo, lo + rng.uniform(0.3, 1.5, N)], axis=1).reshape(-1)
    lists = [np.sort(rng.uniform(0.1, 3.0, int(rng.integers(1, 9)))) for _ in range(M)]
    consts = {wl.C3_OSCILLATORY: [float(rng.uniform(0, 1))], wl.D_LIN_Y: [float(rng.integers(0, N))]}.get(fam, [])
    precision = int(rng.choice([wl.PREC_F64, wl.PREC_F32E]))
    n = int(rng.choice([2, 5, 17, 64, 100, 257, 1000, 1234]))
    w = wl.Workload(f"fuzz{case}", fam, bounds, lists, n, int(rng.integers(0, 2**63)), precision, np.array(consts))
    G = w.G
    first = int(rng.integers(0, G))
    count = int(rng.integers(1, G - first + 1))
    opts = dict(schedule=int(rng.integers(1, 4)), first_index=first, count=count,
                batch_points=int(rng.choice([0, 1, 3, 64, 1000])), host_out=bool(rng.integers(0, 2)))
    w.out_f32 = bool(rng.integers(0, 2)) and precision == wl.PREC_F32E
    return w, opts


@pytest.mark.parametrize("case", range(60))
def test_random_configuration_matches_oracle(case):
    import torch
    from paper_1910_01965_b200 import binding as zb
    w, opts = draw(case)
    rc, mean_o, err_o = orc.scan_workload(w, opts["first_index"], opts["count"], n_threads=NT)
    assert rc == 0, (w, opts)
    # outputs sit inside guard zones of NaN (compute-sanitizer is closed on this GPU pool): a write outside
    # [0, count) of either array -- on the device or, with host outputs, by the result copies -- shows up here
    pad, count = 96, opts["count"]
    dt = torch.float32 if w.out_f32 else torch.float64
    mk = (lambda: torch.full((count + 2 * pad,), float("nan"), dtype=dt).pin_memory()) if opts["host_out"] else \
         (lambda: torch.full((count + 2 * pad,), float("nan"), dtype=dt, device="cuda"))
    gm, ge = mk(), mk()
    m, e, _ = zb.scan_workload(w, out_mean=gm[pad:pad + count], out_stderr=ge[pad:pad + count], **opts)
    torch.cuda.synchronize()
    for g in (gm, ge):
        assert bool(torch.isnan(g[:pad]).all()) and bool(torch.isnan(g[pad + count:]).all()), "write outside the output range"
        assert not bool(torch.isnan(g[pad:pad + count]).any()), "an element of the range was not written"
    assert_parity(w, m.cpu().numpy(), e.cpu().numpy(), mean_o, err_o)      # one tolerance rule, from the box (test_gpu_parity.py)
