"""CPU-only checks of the C-ABI boundary: the library loads, exports every symbol include/zmc.h
declares, and its pure-host entry points (validation, schedule choice, batch cutting) behave.
No compute call is made here (there is no GPU and no CPU fallback)."""
import os
import re

import numpy as np
import pytest

from paper_1910_01965_b200 import binding as zb
from paper_1910_01965_b200 import workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    lib = zb.load()
    header = open(os.path.join(ROOT, "include", "zmc.h")).read()
    declared = set(re.findall(r"ZMC_API[^;(]*?\b(zmc_\w+)\s*\(", header))
    assert declared == set(zb.EXPORTS)
    for name in declared:
        assert hasattr(lib, name), name
    assert "sm_100a" in zb.zmc_version()


def test_struct_layouts_match_header_sizes(tmp_path):
    # the header is plain C99: compile it with gcc and compare struct sizes with the ctypes mirrors
    import ctypes
    import subprocess
    src = tmp_path / "sz.c"
    # (bench_probe.h, the header of bench.py's separate micro-benchmark library, is checked the same way against bench_probe.py)
    import bench_probe
    src.write_text('#include <stdio.h>\n#include "zmc.h"\n#include "bench_probe.h"\nint main(void){printf("%zu %zu %zu %zu %zu %zu\\n",'
                   'sizeof(zmc_options),sizeof(zmc_timing),sizeof(zmc_param_list),sizeof(zmc_integrand_info),'
                   'sizeof(bench_pipe_report),sizeof(zmc_farm_timing));return 0;}\n')
    exe = tmp_path / "sz"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", os.path.join(ROOT, "include"), "-I", ROOT, str(src), "-o", str(exe)],
                   check=True)
    sizes = [int(v) for v in subprocess.run([str(exe)], capture_output=True, text=True, check=True).stdout.split()]
    assert sizes == [ctypes.sizeof(zb.zmc_options), ctypes.sizeof(zb.zmc_timing), ctypes.sizeof(zb.zmc_param_list),
                     ctypes.sizeof(zb.zmc_integrand_info), ctypes.sizeof(bench_probe._Report), ctypes.sizeof(zb.zmc_farm_timing)]


def test_integrand_table():
    fams = {f["id"]: f for f in zb.zmc_integrands()}
    assert set(fams) == {1, 2, 3, 4, 5, 6, 100, 101, 102, 103}
    assert fams[3]["n_consts"] == 1 and fams[3]["M"] == (3, 3)
    assert fams[4]["N"] == (6, 6) and fams[5]["M"] == (5, 5)


def test_every_config_validates_with_expected_grid_size():
    sizes = {1: 10 ** 3, 2: 10 ** 6, 3: 8 * 10 ** 6, 4: 10 ** 8, 5: 10 ** 10}
    for k, G in sizes.items():
        w = wl.config(k)
        st, g = zb.zmc_validate(w.integrand_id, w.bounds, w.lists, w.n_samples, precision=w.precision,
                                consts=w.consts)
        assert (st, g) == (zb.ZMC_OK, G) and w.G == G


def test_validation_errors():
    w = wl.config(1, scale=[4], n_samples=10)
    ok = dict(integrand_id=1, bounds=w.bounds, lists=w.lists, n_samples=10)

    def st(**kw):
        a = dict(ok)
        a.update(kw)
        extra = {k: a.pop(k) for k in list(a) if k not in ("integrand_id", "bounds", "lists", "n_samples")}
        return zb.zmc_validate(a["integrand_id"], a["bounds"], a["lists"], a["n_samples"], **extra)[0]

    assert st() == zb.ZMC_OK
    assert st(n_samples=1) == zb.ZMC_ERR_INVALID_ARG
    assert st(n_samples=1 << 32) == zb.ZMC_ERR_INVALID_ARG
    assert st(bounds=[0.0, 0.0]) == zb.ZMC_ERR_INVALID_ARG
    assert st(bounds=[0.0, float("inf")]) == zb.ZMC_ERR_INVALID_ARG
    assert st(lists=[np.array([1.0, float("nan")])]) == zb.ZMC_ERR_INVALID_ARG
    assert st(integrand_id=42) == zb.ZMC_ERR_UNKNOWN_INTEGRAND
    assert st(integrand_id=2) == zb.ZMC_ERR_SHAPE_MISMATCH
    assert st(integrand_id=3, lists=[w.lists[0]] * 3) == zb.ZMC_ERR_SHAPE_MISMATCH      # c3 needs consts={u}
    assert st(integrand_id=3, lists=[w.lists[0]] * 3, consts=[0.25]) == zb.ZMC_OK
    assert st(integrand_id=101, consts=[1.0]) == zb.ZMC_ERR_SHAPE_MISMATCH                # echo index >= M
    assert st(first_index=5) == zb.ZMC_ERR_INVALID_ARG
    assert st(first_index=2, count=3) == zb.ZMC_ERR_INVALID_ARG
    assert st(first_index=2, count=2) == zb.ZMC_OK
    assert st(precision=7) == zb.ZMC_ERR_INVALID_ARG
    assert st(schedule=9) == zb.ZMC_ERR_INVALID_ARG
    big = [np.zeros(1 << 17)] * 3                                                         # 2^51 points
    assert st(integrand_id=6, lists=big) == zb.ZMC_ERR_GRID_TOO_LARGE
    assert st(integrand_id=6, bounds=[0.0, 1.0] * 16, n_samples=(1 << 30) + 1) == zb.ZMC_ERR_INVALID_ARG
    assert "invalid" in zb.zmc_status_string(zb.ZMC_ERR_INVALID_ARG)


def test_schedule_choice_follows_design_table():
    # cfg1 CTA, cfg2-5 THREAD (cfg 2 = 8.8 rounds of the 148 x 768 resident fp64 threads;
    # measured 2.8 % faster than WARP).  No GPU here: the chooser falls back to 148 SMs.
    expect = {1: zb.ZMC_SCHED_CTA, 2: zb.ZMC_SCHED_THREAD, 3: zb.ZMC_SCHED_THREAD, 4: zb.ZMC_SCHED_THREAD}
    for k, s in expect.items():
        w = wl.config(k)
        assert zb.zmc_pick_schedule(w.G, w.n_samples, w.N, w.precision) == s
    w = wl.config(5)
    assert zb.zmc_pick_schedule(1 << 28, w.n_samples, w.N, w.precision) == zb.ZMC_SCHED_THREAD
    assert zb.zmc_pick_schedule(10, 8, 1) == zb.ZMC_SCHED_THREAD          # too few samples to split
    # between the two: a 10^5-point grid with many samples goes warp-per-point; the fp32-evaluate kernels keep 1024
    # threads per SM resident instead of 768, so their THREAD threshold is higher
    assert zb.zmc_pick_schedule(10 ** 5, 10 ** 4, 2) == zb.ZMC_SCHED_WARP
    assert zb.zmc_pick_schedule(10 ** 6, 10 ** 4, 2, zb.ZMC_PREC_F64) == zb.ZMC_SCHED_THREAD
    assert zb.zmc_pick_schedule(10 ** 6, 10 ** 4, 2, zb.ZMC_PREC_F32E) == zb.ZMC_SCHED_WARP
    # WARP from two rounds of resident warps (148 SMs x 24 fp64 / 32 fp32-evaluate warps), one CTA per point below that
    assert zb.zmc_pick_schedule(7000, 10 ** 4, 2) == zb.ZMC_SCHED_CTA and zb.zmc_pick_schedule(7200, 10 ** 4, 2) == zb.ZMC_SCHED_WARP
    assert zb.zmc_pick_schedule(9400, 10 ** 4, 4, zb.ZMC_PREC_F32E) == zb.ZMC_SCHED_CTA
    assert zb.zmc_pick_schedule(9500, 10 ** 4, 4, zb.ZMC_PREC_F32E) == zb.ZMC_SCHED_WARP


def test_explicit_count_makes_an_empty_range_expressible():
    # count == 0 used to mean only "to the end of the grid"; a caller whose shard is empty at first < G
    # had no way to say so.  ZMC_OPT_EXPLICIT_COUNT takes count literally.
    w = wl.config(1, scale=[4], n_samples=10)
    import ctypes
    m = zb._Marshalled(w.bounds, w.lists, None)
    for flags, first, count, want in [(0, 2, 0, zb.ZMC_OK), (zb.ZMC_OPT_EXPLICIT_COUNT, 2, 0, zb.ZMC_OK),
                                      (zb.ZMC_OPT_EXPLICIT_COUNT, 4, 0, zb.ZMC_OK), (zb.ZMC_OPT_EXPLICIT_COUNT, 2, 3, zb.ZMC_ERR_INVALID_ARG),
                                      (64, 0, 0, zb.ZMC_ERR_INVALID_ARG)]:
        o = zb._make_options(m, zb.ZMC_PREC_F64, zb.ZMC_OUT_F64, zb.ZMC_LOC_DEVICE, 0, -1, 0, first, count, flags)
        g = ctypes.c_uint64(0)
        st = zb.load().zmc_validate(1, m.N, m.bounds_ptr(), m.M, m.c_lists, 10, ctypes.byref(o), ctypes.byref(g))
        assert st == want, (flags, first, count)
    # an explicitly empty range is a no-op that needs no GPU: nothing is enqueued, outputs stay untouched
    mean, err = np.full(1, 7.0), np.full(1, 7.0)
    zb.zmc_scan_ex(1, w.bounds, w.lists, 10, 1, mean, err, stream=0, first_index=2, count=0, flags=zb.ZMC_OPT_EXPLICIT_COUNT)
    assert mean[0] == 7.0 and err[0] == 7.0


@pytest.mark.parametrize("first,count,bp", [(0, 10 ** 10, 1 << 28), (5, 1000, 97), (0, 7, 0), (3, 7, 100), (0, 8, 4)])
def test_batch_cutting_covers_range_exactly(first, count, bp):
    nb, _, _ = zb.zmc_batch_range(first, count, bp, 0)
    pos = first
    for b in range(nb):
        n2, f, c = zb.zmc_batch_range(first, count, bp, b)
        assert n2 == nb and f == pos and c >= 1
        assert c == (bp if bp and b < nb - 1 else c)
        pos += c
    assert pos == first + count
    if (first, count, bp) == (0, 10 ** 10, 1 << 28):
        assert nb == 38 and zb.zmc_batch_range(first, count, bp, 37)[2] == 67_888_128


def test_compute_call_fails_loudly_without_gpu():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    w = wl.config(1, scale=[4], n_samples=10)
    mean, err = np.zeros(4), np.zeros(4)
    with pytest.raises(zb.ZmcError) as ei:
        zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, stream=0)
    assert ei.value.status == zb.ZMC_ERR_CUDA
    assert np.all(mean == 0) and np.all(err == 0)
