"""-m gpu: zmc_scan_noalloc, the scan for callers that must not allocate GPU memory, against the ordinary zmc_scan_ex.

Why the entry point exists: a process that gave all device memory to its own pool (an inference server, a framework's
caching allocator), a latency-critical loop, or a deployment with a fixed buffer plan cannot have a library call
cudaMalloc / cudaFree behind its back -- those calls take a driver lock, may synchronise the whole device, and change
the free memory the owner counts on.  zmc_scan_noalloc therefore keeps the library's device copy of the value lists in
a fixed 32 KiB array inside libzmc.so (at most ZMC_NOALLOC_MAX_LIST_VALUES list entries per call) where zmc_scan_ex
uses memory it allocates on demand.  Both run the same kernels on the same parameter block, so the results must be
bit-identical -- the standard this suite applies wherever only the plumbing differs (test_gpu_parity.py,
test_batch_and_subrange_invariance_bit_exact).

The array is shared by all calls and keeps the previous call's contents, so every comparison here is made on two calls
IN A ROW with different lists (longer, then shorter, then the first again): a call that read entries the previous one
left behind, or failed to overwrite its own, would differ from the reference.

This file is named to be collected last (pytest -x stops at the first failure; a failure here must not hide the other
tests), and each test passes both in a fresh process -- where its first call performs the per-device set-up -- and after
the rest of the suite.
"""
import numpy as np
import pytest

from paper_1910_01965_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _zb():
    from paper_1910_01965_b200 import binding
    return binding


def _outputs(w, n_out):
    import torch
    dtype = torch.float32 if w.out_f32 else torch.float64
    return (torch.full((n_out,), float("nan"), dtype=dtype, device="cuda"),
            torch.full((n_out,), float("nan"), dtype=dtype, device="cuda"))


def _reference(w, schedule, first_index=0, count=0):
    """The existing path: zmc_scan_ex into device memory."""
    import torch
    zb = _zb()
    mean, err = _outputs(w, count or w.G - first_index)
    zb.zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, precision=w.precision,
                   schedule=schedule, first_index=first_index, count=count, consts=w.consts)
    torch.cuda.synchronize()
    return mean.cpu().numpy(), err.cpu().numpy()


def _noalloc(w, schedule, first_index=0, count=0, stream=None):
    import torch
    zb = _zb()
    mean, err = _outputs(w, count or w.G - first_index)
    zb.zmc_scan_noalloc(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, stream,
                        precision=w.precision, schedule=schedule, first_index=first_index, count=count, consts=w.consts)
    torch.cuda.synchronize()
    return mean.cpu().numpy(), err.cpu().numpy()


def _same(a, b):
    return np.array_equal(a[0], b[0]) and np.array_equal(a[1], b[1]) and np.isfinite(a[0]).all() and np.isfinite(a[1]).all()


@pytest.mark.parametrize("schedule", [1, 2, 3], ids=["thread", "warp", "cta"])
@pytest.mark.parametrize("prec", ["f64", "f32e"])
def test_two_calls_in_a_row_match_the_allocating_path_bit_for_bit(prec, schedule):
    if prec == "f64":
        first = wl.config(2, scale=[37, 41], n_samples=301)            # 78 list entries
        second = wl.config(1, scale=[29], n_samples=257)               # 29: shorter, other family, other shape
    else:
        first = wl.config(5, scale=[3, 4, 5, 3, 7], n_samples=130)     # fp32 results
        second = wl.config(3, scale=[5, 2, 3], n_samples=97)
        first.host_out = False
    ref_first, ref_second = _reference(first, schedule), _reference(second, schedule)
    got_first = _noalloc(first, schedule)
    got_second = _noalloc(second, schedule)            # finds the first call's lists in the array
    got_again = _noalloc(first, schedule)              # finds the second call's
    assert _same(got_first, ref_first)
    assert _same(got_second, ref_second)
    assert _same(got_again, ref_first)


def test_back_to_back_on_one_stream_without_a_sync_in_between():
    """Two calls enqueued on the same (non-default) stream with no host synchronisation between them: the stream
    orders the second call's list upload after the first call's kernels."""
    import torch
    zb = _zb()
    a = wl.config(2, scale=[64, 50], n_samples=2000)
    b = wl.config(2, scale=[50, 64], n_samples=2000)
    ref_a, ref_b = _reference(a, 1), _reference(b, 1)
    stream = torch.cuda.Stream()
    outs = [_outputs(a, a.G), _outputs(b, b.G)]
    with torch.cuda.stream(stream):
        for w, (mean, err) in zip((a, b), outs):
            zb.zmc_scan_noalloc(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err, stream,
                                precision=w.precision, schedule=1, consts=w.consts)
    stream.synchronize()
    assert _same((outs[0][0].cpu().numpy(), outs[0][1].cpu().numpy()), ref_a)
    assert _same((outs[1][0].cpu().numpy(), outs[1][1].cpu().numpy()), ref_b)


def test_sub_range_and_auto_schedule():
    w = wl.config(4, scale=[3, 4, 5, 6], n_samples=100)
    assert _same(_noalloc(w, 0, first_index=77, count=201), _reference(w, 0, first_index=77, count=201))
    assert _same(_noalloc(w, 0), _reference(w, 0))


def test_the_limit_is_enforced_and_the_largest_accepted_size_works():
    import torch
    zb = _zb()
    cap = zb.ZMC_NOALLOC_MAX_LIST_VALUES
    bounds = np.array([0.0, 1.0, 0.0, 2.0])
    full = wl.Workload("full", wl.P6_SIN_SUM, bounds, [wl.linspace(0.5, 5.0, cap - 96), wl.linspace(0.1, 0.9, 96)],
                       64, 3, wl.PREC_F64, np.zeros(0))
    # exactly the maximum (10 list-staging launches, too long for shared-memory staging): a slice around the middle and the
    # last points of the grid, so the far end of the array is read
    for first_index, count in ((full.G // 2 - 100, 300), (full.G - 300, 300)):
        for schedule in (1, 2):
            assert _same(_noalloc(full, schedule, first_index, count), _reference(full, schedule, first_index, count))
    # one entry more: refused with the status of its own, nothing enqueued, outputs untouched
    over = wl.Workload("over", wl.P6_SIN_SUM, bounds, [wl.linspace(0.5, 5.0, cap - 95), wl.linspace(0.1, 0.9, 96)],
                       64, 3, wl.PREC_F64, np.zeros(0))
    mean, err = _outputs(over, 8)
    with pytest.raises(zb.ZmcError) as exc:
        zb.zmc_scan_noalloc(over.integrand_id, over.bounds, over.lists, over.n_samples, over.seed, mean, err, count=8)
    assert exc.value.status == zb.ZMC_ERR_NOALLOC_LIMIT
    assert "ZMC_NOALLOC_MAX_LIST_VALUES" in str(exc.value)
    torch.cuda.synchronize()
    assert torch.isnan(mean).all() and torch.isnan(err).all()


def test_what_it_cannot_do_is_refused_up_front():
    import torch
    zb = _zb()
    w = wl.config(1, scale=[5], n_samples=16)
    host = torch.full((5,), -1.0, dtype=torch.float64).pin_memory()
    with pytest.raises(zb.ZmcError) as exc:        # host outputs would need the library's staging buffers
        zb.zmc_scan_noalloc(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, host, host.clone().pin_memory())
    assert exc.value.status == zb.ZMC_ERR_INVALID_ARG
    mean, err = _outputs(w, 5)
    with pytest.raises(zb.ZmcError) as exc:        # run-time compiled integrands load code
        zb.zmc_scan_noalloc(1000, w.bounds, w.lists, w.n_samples, w.seed, mean, err)
    assert exc.value.status == zb.ZMC_ERR_UNKNOWN_INTEGRAND
    with pytest.raises(zb.ZmcError) as exc:        # the ordinary argument checks still apply
        zb.zmc_scan_noalloc(w.integrand_id, w.bounds, w.lists, 1, w.seed, mean, err)
    assert exc.value.status == zb.ZMC_ERR_INVALID_ARG
    torch.cuda.synchronize()
    assert (host == -1.0).all() and torch.isnan(mean).all()


def test_a_repeated_call_leaves_the_free_device_memory_where_it_was():
    """The point of the entry point, observed from outside: once the first call has done its set-up (array address,
    kernel code loaded), further calls change nothing in the device's memory accounting."""
    import torch
    zb = _zb()
    w = wl.config(2, scale=[40, 30], n_samples=500)
    mean, err = _outputs(w, w.G)

    def call():
        zb.zmc_scan_noalloc(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, mean, err,
                            precision=w.precision, schedule=2, consts=w.consts)
        torch.cuda.synchronize()

    call()                                             # set-up, kernel loading
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        call()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    assert _same((mean.cpu().numpy(), err.cpu().numpy()), _reference(w, 2))
