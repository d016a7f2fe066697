"""-m gpu: edge cases of the CUDA path against the CPU oracle -- empty and ragged inputs, smallest and largest
shapes the boundary accepts, degenerate grids, lists too long for shared-memory staging."""
import os

import numpy as np
import pytest

from oracle import zmc_oracle as orc
from paper_1910_01965_b200 import workloads as wl
from test_gpu_parity import assert_parity, run_gpu

pytestmark = pytest.mark.gpu
NT = min(16, os.cpu_count() or 1)


def _check(w, **kw):
    first, count = kw.get("first_index", 0), kw.get("count", 0)
    rc, mean_o, err_o = orc.scan_workload(w, first, count or None, n_threads=NT)
    assert rc == 0
    for sched in (1, 2, 3):
        mean, err = run_gpu(w, schedule=sched, **kw)
        assert_parity(w, mean, err, mean_o, err_o)


@pytest.mark.parametrize("n", [2, 3, 4, 5, 7, 8, 9, 31, 33, 255, 257])
@pytest.mark.parametrize("cfg", [1, 2, 3, 4, 5])
def test_smallest_and_ragged_sample_counts(cfg, n):
    """n = 2 is the smallest count the estimator accepts; the others straddle the sample-group sizes (1, 2, 4, 8) and
    the lane counts, so groups are clipped and most lanes of the WARP / CTA schedules stay idle."""
    scale = {1: [7], 2: [3, 5], 3: [2, 3, 2], 4: [2, 2, 3, 2], 5: [2, 2, 2, 3, 2]}[cfg]
    _check(wl.config(cfg, scale=scale, n_samples=n))


def test_single_point_grid_and_length_one_lists():
    w = wl.config(5, scale=[1, 1, 1, 1, 1], n_samples=300)
    assert w.G == 1
    _check(w)
    _check(wl.config(4, scale=[1, 6, 1, 5], n_samples=100))


def test_maximum_dimensions_N16_M8():
    """N = 16 (runtime-N kernels, 16 Philox blocks per 4-sample group) and M = 8 lists."""
    lists = [wl.linspace(0.0, 0.3, c) for c in (2, 1, 3, 2, 1, 2, 2, 3)]
    w = wl.Workload("p6_max", wl.P6_SIN_SUM, np.array([0.0, 1.0] * 16), lists, 203, 11, wl.PREC_F64, np.zeros(0))
    _check(w)
    w32 = wl.Workload("p6_max32", wl.P6_SIN_SUM, np.array([0.0, 0.5] * 16), lists, 203, 11, wl.PREC_F32E, np.zeros(0))
    _check(w32)
    w3 = wl.config(3, scale=[3, 2, 3], n_samples=130)
    w3.bounds = np.array([0.0, 1.0] * 16)
    _check(w3)


def test_empty_ranges_enqueue_nothing():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(2, scale=[4, 5], n_samples=10)
    mean = torch.full((4,), -3.0, dtype=torch.float64, device="cuda")
    err = torch.full((4,), -3.0, dtype=torch.float64, device="cuda")
    # first_index == G with count 0 (= "to the end of the grid"): nothing to do, status OK, outputs untouched
    tm = zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, first_index=w.G, count=0,
                        timing=True)
    torch.cuda.synchronize()
    assert torch.all(mean == -3.0) and torch.all(err == -3.0)
    assert tm["gpu_launches"] == 0 and tm["n_batches"] == 0
    with pytest.raises(zb.ZmcError):       # a range reaching past the grid is an argument error
        zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, first_index=w.G - 1, count=2)


def test_ragged_subranges_and_batches_fp32_host_output():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(5, scale=[3, 4, 5, 3, 7], n_samples=70)        # G = 1260
    first, count = 13, 1009                                      # prime count, 7 batches of 150 + one of 109... ragged
    rc, mean_o, err_o = orc.scan_workload(w, first, count, n_threads=NT)
    for sched in (1, 2, 3):
        m, e, tm = zb.scan_workload(w, schedule=sched, first_index=first, count=count, batch_points=150, host_out=True,
                                    timing=True)
        torch.cuda.synchronize()
        assert tm["n_batches"] == 7 and tm["d2h_bytes"] == 8 * count
        assert_parity(w, m.numpy(), e.numpy(), mean_o, err_o)


def test_lists_too_long_for_shared_memory_staging():
    """2 x 40 000 doubles = 640 KB of lists: the THREAD schedule falls back to reading them through L1/L2."""
    lists = [wl.linspace(0.5, 5.0, 40_000), wl.linspace(0.5, 5.0, 40_000)]
    w = wl.Workload("long_lists", wl.C2_SIN_XY2, np.array([0.0, wl.PI, 0.0, wl.PI]), lists, 64, 3, wl.PREC_F64, np.zeros(0))
    first = 40_000 * 12_345 + 39_990                             # straddles a row of the grid
    _check(w, first_index=first, count=700)


def test_seed_uses_all_64_bits():
    w = wl.config(1, scale=[5], n_samples=50)
    w.seed = 0x0123456789ABCDEF
    _check(w)
    a, _ = run_gpu(w, schedule=1)
    w.seed = 0x0123456789ABCDEF ^ (1 << 40)
    b, _ = run_gpu(w, schedule=1)
    assert not np.array_equal(a, b)


def test_back_to_back_host_output_scans_on_two_streams_and_after_shutdown():
    """The D2H staging buffers alternate across batches and across calls; several host-output scans in flight at once
    (different user streams, no synchronisation in between) must not overwrite each other's staged results, and the
    library must come back after zmc_shutdown()."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    ws = [wl.config(5, scale=[5, 4, 3, 6, 7], n_samples=64 + 8 * i) for i in range(4)]
    refs = []
    for w in ws:
        w.host_out, w.batch_points = False, 0
        refs.append(run_gpu(w, schedule=1))
    streams = [torch.cuda.Stream(), torch.cuda.Stream()]
    outs = []
    for i, w in enumerate(ws):                    # four scans enqueued without waiting, 3-5 batches each
        m = torch.full((w.G,), float("nan"), dtype=torch.float32).pin_memory()
        e = torch.full((w.G,), float("nan"), dtype=torch.float32).pin_memory()
        zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, streams[i & 1], precision=w.precision,
                       schedule=1, batch_points=600 + 100 * i, consts=w.consts)
        outs.append((m, e))
    torch.cuda.synchronize()
    for (m, e), (rm, re) in zip(outs, refs):
        assert np.array_equal(m.numpy(), rm) and np.array_equal(e.numpy(), re)
    zb.zmc_shutdown()
    m2, e2 = run_gpu(ws[0], schedule=1)
    assert np.array_equal(m2, refs[0][0]) and np.array_equal(e2, refs[0][1])


def test_measure_pipes_reports_the_dispatch_costs_the_roofline_uses():
    """bench_probe.py (bench.py's micro-benchmark, its own libzmc_probe.so): the rows bench.py prints as `pipe_rates`.  Sanity bands only -- the numbers are
    measurements -- around what DESIGN.md section 6 builds the ALU roofline from: integer 2 cycles per warp-instruction,
    FP32 1, FP64 2, XU 8, and a `serial >= parallel` pair of bounds on every mixed row."""
    import torch
    import bench_probe
    rep = bench_probe.measure_pipes(torch.cuda.current_stream().cuda_stream)
    rows = {r["name"]: r for r in rep["rows"]}
    assert rep["sm_count"] >= 1 and 500.0 < rep["sm_mhz"] < 3000.0 and len(rows) >= 40
    for name, lo, hi in [("LOP3", 1.8, 2.6), ("SHF", 1.8, 2.6), ("IMAD.WIDE+LOP3", 3.6, 5.0), ("FFMA", 0.9, 1.5),
                         ("DFMA", 1.8, 2.6), ("DADD", 1.8, 2.6), ("MUFU.EX2", 7.0, 9.5), ("F2F.F64.F32", 7.0, 9.5)]:
        assert lo < rows[name]["cycles"] < hi, (name, rows[name])
    for r in rep["rows"]:
        assert r["serial"] >= r["parallel"] > 0 and 0.8 * r["parallel"] < r["cycles"] < 1.25 * r["serial"], r
    both = rows["cfg2 block: both, same warp (ptxas order)"]
    assert both["parallel"] < both["cycles"] < both["serial"]
    # the Philox-block rows: a 32-bit product overlaps with the XORs, the high half of the product is what
    # costs; inside the Philox stream an FP32 instruction adds about 1 cycle and an integer one about 2 -- nothing hides
    assert 1.8 < rows["IMAD.LO"]["cycles"] < 2.6 and 3.6 < rows["IMAD.HI"]["cycles"] < 5.0
    assert rows["1xIMAD.LO + 1xLOP3, same warp"]["cycles"] < 0.85 * rows["1xIMAD.LO + 1xLOP3, same warp"]["serial"]
    base = rows["Philox block: 16 IMAD.WIDE + 18 LOP3 per thread + uniform rounds 1-2"]["cycles"]
    assert 64.0 < base < 90.0
    assert 0.5 < (rows["  + 8 independent FFMA per block"]["cycles"] - base) / 8 < 1.6
    assert 1.4 < (rows["  + 8 independent LOP3 per block"]["cycles"] - base) / 8 < 2.6
    assert rows["  control: low halves only (16 IMAD.LO + 18 LOP3; NOT Philox)"]["cycles"] < 0.85 * base
    assert rows["  high halves by DFMA.RZ (FP64 pipe) + IMAD.LO: same output"]["cycles"] > 0.9 * base


def test_scan_plan_is_the_same_call_and_an_explicitly_empty_shard_is_a_no_op():
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(3, scale=[5, 4, 6], n_samples=300)
    m, e, _ = zb.scan_workload(w)
    pm, pe = torch.full_like(m, -3.0), torch.full_like(e, -3.0)
    plan = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, pm, pe, precision=w.precision, consts=w.consts)
    tm = plan(None, timing=True)
    torch.cuda.synchronize()
    assert torch.equal(pm, m) and torch.equal(pe, e) and tm["gpu_launches"] == 1
    pm.fill_(-3.0)
    empty = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, pm, pe, precision=w.precision, consts=w.consts,
                        first_index=7, count=0, flags=zb.ZMC_OPT_EXPLICIT_COUNT)
    tm = empty(None, timing=True)
    torch.cuda.synchronize()
    assert tm["gpu_launches"] == 0 and bool((pm == -3.0).all())


def test_pinned_empty_is_page_locked_host_memory_the_library_streams_into():
    """binding.pinned_empty (memory plumbing for HOST outputs): parallel first touch + cudaHostRegister.  The library must
    see the buffer as pinned (zmc_timing.host_out_pinned == 1) and the scan through it must equal the device-output scan."""
    import gc
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(5, scale=[8] * 5, n_samples=64)
    count = 1 << 25                                     # 128 MiB per fp32 array: above the helper's small-size fallback
    big = zb.pinned_empty(count, torch.float32, fill=float("nan"))
    err = zb.pinned_empty(count, torch.float32, fill=float("nan"))
    assert big.is_pinned() and err.is_pinned() and bool(torch.isnan(big[::4099]).all())
    m, e, tm = zb.scan_workload(w, out_mean=big[:w.G], out_stderr=err[:w.G], host_out=True, batch_points=10_000, timing=True)
    torch.cuda.synchronize()
    assert tm["host_out_pinned"] == 1 and tm["n_batches"] == 4
    dm, de, _ = zb.scan_workload(w, host_out=False)
    torch.cuda.synchronize()
    assert torch.equal(m, dm.cpu()) and torch.equal(e, de.cpu())
    assert bool(torch.isnan(big[w.G:w.G + 1000]).all())           # nothing written past the range
    small = zb.pinned_empty(1000, torch.float64)                  # small sizes: torch's own pinned allocator
    assert small.is_pinned() and small.numel() == 1000
    del big, err, m, e
    gc.collect()                                                   # the registration is undone with the tensor


def test_small_one_batch_host_scans_are_written_by_the_kernel_itself():
    """H8, small results: one batch, <= 1 MiB, page-locked host buffers -> the kernel stores straight into host memory
    (zmc_timing.host_out_pinned == 2, no copy); bit-identical to the device-output scan.  Larger, batched or pageable
    outputs take the staged path."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(2, scale=[37, 29], n_samples=300)                       # 1073 points x 16 B
    dm, de, _ = zb.scan_workload(w, host_out=False)
    hm = torch.full((w.G + 64,), float("nan"), dtype=torch.float64).pin_memory()
    he = torch.full((w.G + 64,), float("nan"), dtype=torch.float64).pin_memory()
    _, _, tm = zb.scan_workload(w, out_mean=hm[32:32 + w.G], out_stderr=he[32:32 + w.G], host_out=True, batch_points=0, timing=True)
    torch.cuda.synchronize()
    assert tm["host_out_pinned"] == 2 and tm["d2h_bytes"] == 16 * w.G and tm["d2h_ms"] == 0 and tm["n_batches"] == 1
    assert torch.equal(hm[32:32 + w.G], dm.cpu()) and torch.equal(he[32:32 + w.G], de.cpu())
    assert bool(torch.isnan(hm[:32]).all()) and bool(torch.isnan(hm[32 + w.G:]).all())
    # batched -> staged copies; pageable -> reported as such
    _, _, tm = zb.scan_workload(w, out_mean=hm[32:32 + w.G], out_stderr=he[32:32 + w.G], host_out=True, batch_points=500, timing=True)
    torch.cuda.synchronize()
    assert tm["host_out_pinned"] == 1 and tm["n_batches"] == 3 and torch.equal(hm[32:32 + w.G], dm.cpu())
    pm, pe = np.empty(w.G), np.empty(w.G)
    import warnings
    with warnings.catch_warnings():
        warnings.simplefilter("ignore")
        _, _, tm = zb.scan_workload(w, out_mean=pm, out_stderr=pe, host_out=True, batch_points=0, timing=True)
    torch.cuda.synchronize()
    assert tm["host_out_pinned"] == 0 and np.array_equal(pm, dm.cpu().numpy())
    # the adaptive scan, out_n included
    n_d = torch.zeros(w.G, dtype=torch.int32, device="cuda")
    am, ae = torch.empty_like(dm), torch.empty_like(de)
    zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, 256, 2048, 0.2, w.seed, am, ae, n_d)
    n_h = torch.zeros(w.G, dtype=torch.int32).pin_memory()
    tm = zb.zmc_scan_adaptive(w.integrand_id, w.bounds, w.lists, 256, 2048, 0.2, w.seed, hm[32:32 + w.G], he[32:32 + w.G], n_h, timing=True)
    torch.cuda.synchronize()
    assert tm["host_out_pinned"] == 2 and tm["d2h_bytes"] == 20 * w.G
    assert torch.equal(n_h, n_d.cpu()) and torch.equal(hm[32:32 + w.G], am.cpu()) and torch.equal(he[32:32 + w.G], ae.cpu())


def test_host_buffers_that_only_start_in_page_locked_memory_do_not_take_the_direct_path():
    """A result buffer whose first bytes lie in a cudaHostRegister'ed region but whose end runs past it (a slice near the end
    of a registered range, pageable memory behind it) must not be written by the kernel through the mapped alias: the part
    that is not mapped would fault the kernel and poison the context.  It goes through the staged copies instead; whatever
    the runtime makes of a copy into such a range (it may also refuse it), the library stays usable."""
    import mmap
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(2, scale=[37, 29], n_samples=300)                       # 1073 points x 8 B per array
    dm, de, _ = zb.scan_workload(w, host_out=False)
    page = mmap.PAGESIZE
    bufs, arrays = [], []
    rt = torch.cuda.cudart()
    for _ in range(2):
        mm = mmap.mmap(-1, 8 * page)
        arr = np.frombuffer(mm, dtype=np.float64)
        arr[:] = -7.0
        assert int(rt.cudaHostRegister(arr.ctypes.data, 2 * page, 1)) == 0          # only the first two pages are page-locked
        bufs.append(mm)
        arrays.append(arr)
    start = (2 * page - 1024) // 8                                         # the last KiB of the registered part ...
    hm, he = (torch.from_numpy(a)[start:start + w.G] for a in arrays)      # ... and 7.5 KiB of pageable memory behind it
    try:
        import warnings
        with warnings.catch_warnings():
            warnings.simplefilter("ignore")
            try:
                _, _, tm = zb.scan_workload(w, out_mean=hm, out_stderr=he, host_out=True, batch_points=0, timing=True)
                torch.cuda.synchronize()
                assert tm["host_out_pinned"] != 2                          # not the direct path
                assert torch.equal(hm, dm.cpu()) and torch.equal(he, de.cpu())
            except zb.ZmcError as exc:                                     # a clean refusal of the copy is acceptable too
                assert exc.status == zb.ZMC_ERR_CUDA
        torch.cuda.synchronize()                                           # no sticky error: the context still works
        dm2, de2, _ = zb.scan_workload(w, host_out=False)
        torch.cuda.synchronize()
        assert torch.equal(dm2, dm) and torch.equal(de2, de)
    finally:
        for a in arrays:
            rt.cudaHostUnregister(a.ctypes.data)


def test_a_scan_with_device_outputs_can_be_captured_into_a_cuda_graph():
    """A scan into device memory whose value lists are already cached on the device enqueues one kernel and one event record
    on the caller's stream (include/zmc.h, zmc_scan_ex): it can be captured into a CUDA graph and replayed, and ordinary
    calls keep working afterwards (list uploads and evictions included)."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(2, scale=[41, 23], n_samples=500)
    m = torch.zeros(w.G, dtype=torch.float64, device="cuda")
    e = torch.zeros_like(m)
    plan = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, precision=w.precision, consts=w.consts)
    s = torch.cuda.Stream()
    plan(s)                                           # uploads the lists: the captured call must find them cached
    s.synchronize()
    ref_m, ref_e = m.clone(), e.clone()
    m.zero_(); e.zero_()
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s):
        plan(torch.cuda.current_stream())
    torch.cuda.synchronize()
    assert not bool(m.any())                          # capture enqueued nothing
    for _ in range(3):
        m.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(m, ref_m) and torch.equal(e, ref_e)
    for k in range(10):                               # more lists than cache slots: uploads and evictions after the capture
        w2 = wl.config(2, scale=[41, 23], n_samples=500)
        w2.lists[0] = wl.linspace(0.5, 5.0 + k, 41)
        m2, e2, _ = zb.scan_workload(w2)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(m2).all())
    # The graph's kernel node holds the address of the library's cached copy of the lists.  That copy must have survived the
    # ten other list sets above (every ordinary slot was recycled) -- and a much longer set, which makes slots reallocate.
    big = wl.config(2, scale=[3000, 7], n_samples=16)
    zb.scan_workload(big, count=64)
    for k in range(9):
        w3 = wl.config(2, scale=[3000 + k, 5], n_samples=16)
        zb.scan_workload(w3, count=64)
    torch.cuda.synchronize()
    for _ in range(2):
        m.zero_(); e.zero_()
        g.replay()
        torch.cuda.synchronize()
        assert torch.equal(m, ref_m) and torch.equal(e, ref_e)


def test_calls_that_cannot_be_captured_are_refused_during_capture():
    """During stream capture a scan whose lists are not cached yet (it would have to upload), or one that asks for timing
    (it would synchronise), returns ZMC_ERR_CUDA / cudaErrorStreamCaptureUnsupported and leaves the capture intact."""
    import torch
    from paper_1910_01965_b200 import binding as zb
    w = wl.config(1, scale=[19], n_samples=64)
    w.lists[0] = wl.linspace(0.25, 7.75, 19)          # lists no other test uses: not in the cache
    m = torch.zeros(w.G, dtype=torch.float64, device="cuda")
    e = torch.zeros_like(m)
    plan = zb.ScanPlan(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, m, e, precision=w.precision, consts=w.consts)
    other = wl.config(1, scale=[23], n_samples=64)
    m2 = torch.zeros(other.G, dtype=torch.float64, device="cuda")
    e2 = torch.zeros_like(m2)
    plan2 = zb.ScanPlan(other.integrand_id, other.bounds, other.lists, other.n_samples, other.seed, m2, e2)
    s = torch.cuda.Stream()
    plan2(s)                                          # `other` is cached, `w` is not
    s.synchronize()
    ref2 = m2.clone()
    g = torch.cuda.CUDAGraph()
    statuses = []
    with torch.cuda.graph(g, stream=s):
        for call, kw in ((plan, {}), (plan2, {"timing": True})):
            with pytest.raises(zb.ZmcError) as exc:
                call(torch.cuda.current_stream(), **kw)
            statuses.append((exc.value.status, zb.load().zmc_last_cuda_error()))
        plan2(torch.cuda.current_stream())            # the capture is still usable
    assert statuses == [(zb.ZMC_ERR_CUDA, 900), (zb.ZMC_ERR_CUDA, 900)]
    m2.zero_()
    g.replay()
    torch.cuda.synchronize()
    assert torch.equal(m2, ref2) and not bool(m.any())


def test_decode_of_a_full_2_pow_30_point_launch_with_awkward_list_lengths():
    """H3: the per-point digits come from host-computed reciprocals that are exact for local indices below 2^30 -- the most a
    launch holds.  param_echo over a 1021 x 1031 x 1033 grid (1.09e9 points, prime lengths), first 2^30 points in ONE launch,
    every digit of every point checked against integer arithmetic on the device; then a range that starts in the middle
    (non-zero base digits, carries) and one with lists of length 1, 2, 3 and 65537."""
    import torch
    from paper_1910_01965_b200 import binding as zb

    def check(lengths, first, count):
        lists = [np.arange(L, dtype=np.float64) for L in lengths]
        strides = [int(np.prod(lengths[i + 1:])) for i in range(len(lengths))]
        mean = torch.empty(count, dtype=torch.float32, device="cuda")
        err = torch.empty(count, dtype=torch.float32, device="cuda")
        for i, L in enumerate(lengths):
            w = wl.Workload("echo", wl.D_PARAM_ECHO, np.array([0.0, 1.0]), lists, 2, 1, wl.PREC_F32E, np.array([float(i)]))
            w.out_f32 = True
            tm = zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, 2, 1, mean, err, None, precision=w.precision, schedule=1,
                                first_index=first, count=count, consts=w.consts, timing=True)
            assert tm["gpu_launches"] == (1 if count <= (1 << 30) else 2)
            step = 1 << 26
            for a in range(0, count, step):
                t = torch.arange(first + a, first + min(count, a + step), dtype=torch.int64, device="cuda")
                want = ((t // strides[i]) % L).to(torch.float32)
                got = mean[a:a + len(t)]
                assert torch.equal(got, want), (lengths, i, int((got != want).nonzero()[0]) + a + first)
            assert not bool(err.any())
        del mean, err
        torch.cuda.empty_cache()

    big = [1021, 1031, 1033]
    check(big, 0, 1 << 30)
    check(big, int(np.prod(big)) - (1 << 29) - 12345, (1 << 29) + 12345)          # up to the last point of the grid
    check([3, 1, 65537, 2, 1], 0, 3 * 65537 * 2)
