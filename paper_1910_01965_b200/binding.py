"""Thin ctypes binding of the C ABI in include/zmc.h -- argument marshalling only.

Every step of the hot path (decode, Philox, integrand, reduction, finalise, result streaming)
runs inside libzmc.so; this module converts Python/numpy/torch arguments to plain pointers and
sizes.  torch is used for device / pinned memory and streams only.  There is NO fallback: if
libzmc.so cannot be built or loaded, importing callers get a RuntimeError.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libzmc.so")

# --- mirrors of include/zmc.h ----------------------------------------------------------------
ZMC_OK, ZMC_ERR_INVALID_ARG, ZMC_ERR_UNKNOWN_INTEGRAND, ZMC_ERR_SHAPE_MISMATCH = 0, 1, 2, 3
ZMC_ERR_GRID_TOO_LARGE, ZMC_ERR_OUT_OF_MEMORY, ZMC_ERR_CUDA = 4, 5, 6
ZMC_ERR_COMPILE = 7
ZMC_ERR_NOALLOC_LIMIT = 8
ZMC_NOALLOC_MAX_LIST_VALUES = 4096
ZMC_PREC_F64, ZMC_PREC_F32E = 0, 1
ZMC_OUT_F64, ZMC_OUT_F32 = 0, 1
ZMC_LOC_DEVICE, ZMC_LOC_HOST = 0, 1
ZMC_SCHED_AUTO, ZMC_SCHED_THREAD, ZMC_SCHED_WARP, ZMC_SCHED_CTA = 0, 1, 2, 3
ZMC_FAST_MATH_DEFAULT, ZMC_FAST_MATH_OFF, ZMC_FAST_MATH_ON = -1, 0, 1
ZMC_OPT_EXPLICIT_COUNT, ZMC_OPT_FRESH_LISTS = 1, 2
ZMC_USER_FAST_MATH = 1

EXPORTS = ["zmc_scan", "zmc_scan_ex", "zmc_integrand_count", "zmc_integrand_info_at",
           "zmc_integrand_info_by_id", "zmc_status_string", "zmc_last_cuda_error", "zmc_version",
           "zmc_validate", "zmc_pick_schedule", "zmc_batch_range", "zmc_shutdown",
           "zmc_register_integrand", "zmc_last_compile_log", "zmc_scan_farm", "zmc_scan_adaptive",
           "zmc_pick_schedule_ex", "zmc_register_integrand_ex", "zmc_unregister_integrand", "zmc_scan_farm_adaptive",
           "zmc_scan_noalloc"]


class zmc_param_list(ctypes.Structure):
    _fields_ = [("values", ctypes.POINTER(ctypes.c_double)), ("count", ctypes.c_int64)]


class zmc_options(ctypes.Structure):
    _fields_ = [("struct_size", ctypes.c_uint32), ("precision", ctypes.c_int32), ("out_dtype", ctypes.c_int32),
                ("out_location", ctypes.c_int32), ("schedule", ctypes.c_int32), ("fast_math", ctypes.c_int32),
                ("batch_points", ctypes.c_uint64), ("first_index", ctypes.c_uint64), ("count", ctypes.c_uint64),
                ("consts", ctypes.POINTER(ctypes.c_double)), ("n_consts", ctypes.c_int32),
                ("flags", ctypes.c_int32)]


class zmc_timing(ctypes.Structure):
    _fields_ = [("h2d_ms", ctypes.c_double), ("kernel_ms", ctypes.c_double), ("d2h_ms", ctypes.c_double),
                ("exposed_d2h_ms", ctypes.c_double), ("wall_ms", ctypes.c_double), ("n_batches", ctypes.c_int64),
                ("gpu_launches", ctypes.c_int64), ("d2h_bytes", ctypes.c_uint64), ("h2d_bytes", ctypes.c_uint64),
                ("schedule", ctypes.c_int32), ("host_out_pinned", ctypes.c_int32)]

    def as_dict(self):
        return {f: getattr(self, f) for f, _ in self._fields_}


ZMC_MAX_FARM_DEVICES = 16


class zmc_farm_timing(ctypes.Structure):
    _fields_ = [("wall_ms", ctypes.c_double), ("n_batches", ctypes.c_int64), ("batch_points", ctypes.c_uint64),
                ("n_devices", ctypes.c_int32), ("reserved", ctypes.c_int32),
                ("batches_done", ctypes.c_int64 * ZMC_MAX_FARM_DEVICES), ("busy_ms", ctypes.c_double * ZMC_MAX_FARM_DEVICES)]


class zmc_integrand_info(ctypes.Structure):
    _fields_ = [("id", ctypes.c_int32), ("name", ctypes.c_char_p), ("N_min", ctypes.c_int32),
                ("N_max", ctypes.c_int32), ("M_min", ctypes.c_int32), ("M_max", ctypes.c_int32),
                ("n_consts", ctypes.c_int32), ("has_closed_form", ctypes.c_int32)]


class ZmcError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"zmc status {status}: {message}")
        self.status = status


_lib = None


def load():
    """Load libzmc.so.  The mtime-checked build runs first, so a library that is older than its sources is never loaded
    silently (the .so travels to GPU boxes although git ignores it).  Raises if there is no usable library."""
    global _lib
    if _lib is not None:
        return _lib
    default_path = os.path.join(_HERE, "libzmc.so")
    if LIB_PATH == default_path:
        try:
            from . import build as _build
            _build.build()
        except Exception as exc:  # noqa: BLE001
            if not os.path.exists(LIB_PATH):
                raise RuntimeError(f"libzmc.so is missing and could not be built ({exc}); "
                                   "run `python -m paper_1910_01965_b200.build` -- there is no CPU fallback") from exc
            import warnings
            warnings.warn(f"libzmc.so could not be rebuilt ({exc}); loading the existing one, which may be stale")
    lib = ctypes.CDLL(LIB_PATH)
    P = ctypes.POINTER
    scan_args = [ctypes.c_int, ctypes.c_int, P(ctypes.c_double), ctypes.c_int, P(zmc_param_list),
                 ctypes.c_uint64, ctypes.c_uint64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
    lib.zmc_scan.argtypes = scan_args
    lib.zmc_scan.restype = ctypes.c_int
    lib.zmc_scan_ex.argtypes = scan_args + [P(zmc_options), P(zmc_timing)]
    lib.zmc_scan_ex.restype = ctypes.c_int
    lib.zmc_scan_noalloc.argtypes = scan_args + [P(zmc_options)]
    lib.zmc_scan_noalloc.restype = ctypes.c_int
    lib.zmc_integrand_count.restype = ctypes.c_int
    lib.zmc_integrand_info_at.argtypes = [ctypes.c_int, P(zmc_integrand_info)]
    lib.zmc_integrand_info_by_id.argtypes = [ctypes.c_int, P(zmc_integrand_info)]
    lib.zmc_status_string.argtypes = [ctypes.c_int]
    lib.zmc_status_string.restype = ctypes.c_char_p
    lib.zmc_last_cuda_error.restype = ctypes.c_int
    lib.zmc_version.restype = ctypes.c_char_p
    lib.zmc_validate.argtypes = [ctypes.c_int, ctypes.c_int, P(ctypes.c_double), ctypes.c_int, P(zmc_param_list),
                                 ctypes.c_uint64, P(zmc_options), P(ctypes.c_uint64)]
    lib.zmc_validate.restype = ctypes.c_int
    lib.zmc_pick_schedule.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int]
    lib.zmc_pick_schedule.restype = ctypes.c_int
    lib.zmc_pick_schedule_ex.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int, ctypes.c_int]
    lib.zmc_pick_schedule_ex.restype = ctypes.c_int
    lib.zmc_batch_range.argtypes = [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_uint64, ctypes.c_int64,
                                    P(ctypes.c_uint64), P(ctypes.c_uint64)]
    lib.zmc_batch_range.restype = ctypes.c_int64
    lib.zmc_shutdown.restype = None
    lib.zmc_register_integrand.argtypes = [ctypes.c_char_p, ctypes.c_char_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                           P(ctypes.c_int)]
    lib.zmc_register_integrand.restype = ctypes.c_int
    lib.zmc_last_compile_log.restype = ctypes.c_char_p
    lib.zmc_register_integrand_ex.argtypes = [ctypes.c_char_p, ctypes.c_char_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_int, P(ctypes.c_int)]
    lib.zmc_register_integrand_ex.restype = ctypes.c_int
    lib.zmc_unregister_integrand.argtypes = [ctypes.c_int]
    lib.zmc_unregister_integrand.restype = ctypes.c_int
    lib.zmc_scan_farm.argtypes = scan_args[:9] + [P(ctypes.c_int), ctypes.c_int, P(zmc_options), P(zmc_farm_timing)]
    lib.zmc_scan_farm.restype = ctypes.c_int
    lib.zmc_scan_adaptive.argtypes = scan_args[:5] + [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_double, ctypes.c_uint64,
                                                      ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
                                                      P(zmc_options), P(zmc_timing)]
    lib.zmc_scan_adaptive.restype = ctypes.c_int
    lib.zmc_scan_farm_adaptive.argtypes = scan_args[:5] + [ctypes.c_uint64, ctypes.c_uint64, ctypes.c_double, ctypes.c_uint64,
                                                           ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, P(ctypes.c_int),
                                                           ctypes.c_int, P(zmc_options), P(zmc_farm_timing)]
    lib.zmc_scan_farm_adaptive.restype = ctypes.c_int
    _lib = lib
    return lib


def _check(status: int):
    if status != ZMC_OK:
        lib = load()
        msg = lib.zmc_status_string(status).decode()
        if status == ZMC_ERR_CUDA:
            msg += f" (cudaError {lib.zmc_last_cuda_error()})"
        raise ZmcError(status, msg)


class _Marshalled:
    """Keeps the numpy buffers alive while the C call reads them."""

    def __init__(self, bounds, lists, consts):
        self.bounds = np.ascontiguousarray(bounds, dtype=np.float64)
        self.lists = [np.ascontiguousarray(l, dtype=np.float64) for l in lists]
        self.c_lists = (zmc_param_list * max(len(self.lists), 1))()
        for i, l in enumerate(self.lists):
            self.c_lists[i].values = l.ctypes.data_as(ctypes.POINTER(ctypes.c_double))
            self.c_lists[i].count = len(l)
        self.consts = np.ascontiguousarray(consts if consts is not None else [], dtype=np.float64)

    @property
    def N(self):
        return len(self.bounds) // 2

    @property
    def M(self):
        return len(self.lists)

    def bounds_ptr(self):
        return self.bounds.ctypes.data_as(ctypes.POINTER(ctypes.c_double))

    def consts_ptr(self):
        return self.consts.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if len(self.consts) else None


def _make_options(m: _Marshalled, precision, out_dtype, out_location, schedule, fast_math, batch_points,
                  first_index, count, flags: int = 0) -> zmc_options:
    o = zmc_options()
    o.struct_size = ctypes.sizeof(zmc_options)
    o.precision, o.out_dtype, o.out_location = precision, out_dtype, out_location
    o.schedule, o.fast_math = schedule, fast_math
    o.batch_points, o.first_index, o.count = batch_points, first_index, count
    o.consts = m.consts_ptr()
    o.n_consts = len(m.consts)
    o.flags = flags
    return o


_warned_pageable = False


def _warn_pageable():
    """HOST outputs in pageable memory: cudaMemcpyAsync then runs synchronously on the host, so the copy of batch b
    does not overlap the kernel of batch b+1 (zmc_timing.host_out_pinned reports 0).  Said once."""
    global _warned_pageable
    if not _warned_pageable:
        import warnings
        warnings.warn("zmc: host output buffers are pageable; result copies will not overlap compute -- pass pinned "
                      "memory (binding.pinned_empty or torch.empty(..., pin_memory=True)) for streaming scans", stacklevel=3)
        _warned_pageable = True


def pinned_empty(count: int, dtype, fill=None):
    """A 1-D torch CPU tensor in page-locked host memory, for HOST outputs of streaming scans (memory plumbing only).
    torch's own `pin_memory=True` page-faults the buffer on one thread (80 GB for cfg 5: ~50 s); here an anonymous
    mapping is first touched by all cores and then page-locked with cudaHostRegister (~10 s for 80 GB, measured on the
    B200 box).  The registration is undone when the tensor is garbage-collected.  Falls back to torch for tiny sizes."""
    import mmap
    import threading
    import weakref
    import torch
    np_dtype = {torch.float32: np.float32, torch.float64: np.float64, torch.int32: np.int32, torch.uint8: np.uint8}[dtype]
    nbytes = int(count) * np.dtype(np_dtype).itemsize
    if nbytes < (64 << 20):
        t = torch.empty(int(count), dtype=dtype, pin_memory=True)
        if fill is not None:
            t.fill_(fill)
        return t
    mm = mmap.mmap(-1, nbytes, flags=mmap.MAP_PRIVATE | mmap.MAP_ANONYMOUS)
    arr = np.frombuffer(mm, dtype=np_dtype)
    n_thr = max(1, min(os.cpu_count() or 1, 32))
    chunk = (int(count) + n_thr - 1) // n_thr
    value = 0 if fill is None else fill

    def touch(i):                       # first touch = page fault + zero fill, in parallel (numpy releases the GIL)
        arr[i * chunk:min(int(count), (i + 1) * chunk)] = value

    threads = [threading.Thread(target=touch, args=(i,)) for i in range(n_thr)]
    for th in threads:
        th.start()
    for th in threads:
        th.join()
    rt = torch.cuda.cudart()
    rc = rt.cudaHostRegister(arr.ctypes.data, nbytes, 1)          # cudaHostRegisterPortable: pinned for every device (farm)
    if int(rc) != 0:
        raise RuntimeError(f"cudaHostRegister of {nbytes} bytes failed: {rc}")
    t = torch.from_numpy(arr)
    weakref.finalize(t, rt.cudaHostUnregister, arr.ctypes.data)
    return t


def _tensor_ptr(t):
    """(pointer, out_dtype, out_location) of a torch tensor (cuda or pinned/pageable cpu) or numpy array."""
    if isinstance(t, np.ndarray):
        dt = {np.dtype(np.float64): ZMC_OUT_F64, np.dtype(np.float32): ZMC_OUT_F32}[t.dtype]
        assert t.flags["C_CONTIGUOUS"]
        _warn_pageable()
        return t.ctypes.data, dt, ZMC_LOC_HOST
    import torch
    assert t.is_contiguous()
    dt = {torch.float64: ZMC_OUT_F64, torch.float32: ZMC_OUT_F32}[t.dtype]
    if not t.is_cuda and not t.is_pinned():
        _warn_pageable()
    return t.data_ptr(), dt, (ZMC_LOC_DEVICE if t.is_cuda else ZMC_LOC_HOST)


def _stream_handle(stream):
    if stream is None:
        import torch
        return torch.cuda.current_stream().cuda_stream if torch.cuda.is_available() else 0
    if isinstance(stream, int):
        return stream
    return stream.cuda_stream


def zmc_scan(integrand_id: int, bounds, lists, n_samples: int, seed: int, out_mean, out_stderr, stream=None):
    """include/zmc.h zmc_scan: fp64 path, double device outputs, one batch, AUTO schedule."""
    m = _Marshalled(bounds, lists, None)
    pm, dm, lm = _tensor_ptr(out_mean)
    pe, de, le = _tensor_ptr(out_stderr)
    if (dm, lm, de, le) != (ZMC_OUT_F64, ZMC_LOC_DEVICE, ZMC_OUT_F64, ZMC_LOC_DEVICE):
        raise ZmcError(ZMC_ERR_INVALID_ARG, "zmc_scan writes float64 CUDA tensors; use zmc_scan_ex otherwise")
    _check(load().zmc_scan(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_samples, seed,
                           ctypes.c_void_p(pm), ctypes.c_void_p(pe), ctypes.c_void_p(_stream_handle(stream))))


def zmc_scan_ex(integrand_id: int, bounds, lists, n_samples: int, seed: int, out_mean, out_stderr, stream=None, *,
                precision: int = ZMC_PREC_F64, schedule: int = ZMC_SCHED_AUTO,
                fast_math: int = ZMC_FAST_MATH_DEFAULT, batch_points: int = 0, first_index: int = 0,
                count: int = 0, consts=None, timing: bool = False, flags: int = 0) -> Optional[dict]:
    """include/zmc.h zmc_scan_ex.  Output dtype/location are taken from the output tensors
    (torch CUDA tensor = DEVICE; torch CPU tensor or numpy array = HOST).  Returns the timing
    dict when timing=True (the call then synchronises), else None."""
    m = _Marshalled(bounds, lists, consts)
    pm, dm, lm = _tensor_ptr(out_mean)
    pe, de, le = _tensor_ptr(out_stderr)
    if (dm, lm) != (de, le):
        raise ZmcError(ZMC_ERR_INVALID_ARG, "out_mean and out_stderr must share dtype and location")
    o = _make_options(m, precision, dm, lm, schedule, fast_math, batch_points, first_index, count, flags)
    tm = zmc_timing() if timing else None
    _check(load().zmc_scan_ex(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_samples, seed,
                              ctypes.c_void_p(pm), ctypes.c_void_p(pe), ctypes.c_void_p(_stream_handle(stream)),
                              ctypes.byref(o), ctypes.byref(tm) if timing else None))
    return tm.as_dict() if timing else None


def zmc_scan_noalloc(integrand_id: int, bounds, lists, n_samples: int, seed: int, out_mean, out_stderr, stream=None, *,
                     precision: int = ZMC_PREC_F64, schedule: int = ZMC_SCHED_AUTO,
                     fast_math: int = ZMC_FAST_MATH_DEFAULT, first_index: int = 0, count: int = 0, consts=None,
                     flags: int = 0) -> None:
    """include/zmc.h zmc_scan_noalloc: the scan for callers that must not allocate GPU memory (a process whose device
    memory all belongs to its own pool, a latency-critical loop, a fixed buffer plan).  The library's copy of the value
    lists lives in a fixed 32 KiB array inside libzmc.so instead of cudaMalloc'ed memory, so at most
    ZMC_NOALLOC_MAX_LIST_VALUES list entries in total (else ZmcError with status ZMC_ERR_NOALLOC_LIMIT).  Outputs are
    CUDA tensors the caller allocated; built-in families only.  Overlapping calls on one device race on that array --
    issue them on one stream.  Same results, bit for bit, as zmc_scan_ex."""
    m = _Marshalled(bounds, lists, consts)
    pm, dm, lm = _tensor_ptr(out_mean)
    pe, de, le = _tensor_ptr(out_stderr)
    if (dm, lm) != (de, le):
        raise ZmcError(ZMC_ERR_INVALID_ARG, "out_mean and out_stderr must share dtype and location")
    o = _make_options(m, precision, dm, lm, schedule, fast_math, 0, first_index, count, flags)
    _check(load().zmc_scan_noalloc(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_samples, seed,
                                   ctypes.c_void_p(pm), ctypes.c_void_p(pe), ctypes.c_void_p(_stream_handle(stream)),
                                   ctypes.byref(o)))


def zmc_validate(integrand_id: int, bounds, lists, n_samples: int, *, precision: int = ZMC_PREC_F64,
                 first_index: int = 0, count: int = 0, consts=None, schedule: int = ZMC_SCHED_AUTO,
                 out_dtype: int = ZMC_OUT_F64, out_location: int = ZMC_LOC_DEVICE,
                 fast_math: int = ZMC_FAST_MATH_DEFAULT, batch_points: int = 0):
    """Returns (status, grid_points) without raising and without touching a GPU."""
    m = _Marshalled(bounds, lists, consts)
    o = _make_options(m, precision, out_dtype, out_location, schedule, fast_math, batch_points, first_index, count)
    g = ctypes.c_uint64(0)
    st = load().zmc_validate(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_samples, ctypes.byref(o),
                             ctypes.byref(g))
    return int(st), int(g.value)


def zmc_pick_schedule(count: int, n_samples: int, N: int, precision: Optional[int] = None) -> int:
    if precision is None:
        return int(load().zmc_pick_schedule(count, n_samples, N))
    return int(load().zmc_pick_schedule_ex(count, n_samples, N, precision))


class ScanPlan:
    """The arguments of one zmc_scan_ex call, marshalled once.  Calling the plan is a single ctypes call, so a loop over a
    small grid (cfg 1: the kernel runs 25 us) does not pay the numpy conversions again.  Marshalling only: the plan holds
    pointers and sizes, nothing is computed here."""

    def __init__(self, integrand_id: int, bounds, lists, n_samples: int, seed: int, out_mean, out_stderr, *,
                 precision: int = ZMC_PREC_F64, schedule: int = ZMC_SCHED_AUTO, fast_math: int = ZMC_FAST_MATH_DEFAULT,
                 batch_points: int = 0, first_index: int = 0, count: int = 0, consts=None, flags: int = 0):
        self._m = _Marshalled(bounds, lists, consts)
        pm, dm, lm = _tensor_ptr(out_mean)
        pe, de, le = _tensor_ptr(out_stderr)
        if (dm, lm) != (de, le):
            raise ZmcError(ZMC_ERR_INVALID_ARG, "out_mean and out_stderr must share dtype and location")
        self._keep = (out_mean, out_stderr)
        self._o = _make_options(self._m, precision, dm, lm, schedule, fast_math, batch_points, first_index, count, flags)
        self._tm = zmc_timing()
        self._fn = load().zmc_scan_ex
        self._args = (integrand_id, self._m.N, self._m.bounds_ptr(), self._m.M, self._m.c_lists, n_samples, seed,
                      ctypes.c_void_p(pm), ctypes.c_void_p(pe))

    def __call__(self, stream=None, timing: bool = False) -> Optional[dict]:
        st = self._fn(*self._args, ctypes.c_void_p(_stream_handle(stream)), ctypes.byref(self._o),
                      ctypes.byref(self._tm) if timing else None)
        if st != ZMC_OK:
            _check(st)
        return self._tm.as_dict() if timing else None


def zmc_batch_range(first_index: int, count: int, batch_points: int, b: int):
    """Returns (n_batches, batch_first, batch_count) of batch b."""
    f, c = ctypes.c_uint64(0), ctypes.c_uint64(0)
    nb = load().zmc_batch_range(first_index, count, batch_points, b, ctypes.byref(f), ctypes.byref(c))
    return int(nb), int(f.value), int(c.value)


def zmc_integrands():
    lib = load()
    out = []
    for i in range(lib.zmc_integrand_count()):
        info = zmc_integrand_info()
        _check(lib.zmc_integrand_info_at(i, ctypes.byref(info)))
        out.append({"id": info.id, "name": info.name.decode(), "N": (info.N_min, info.N_max),
                    "M": (info.M_min, info.M_max), "n_consts": info.n_consts,
                    "has_closed_form": bool(info.has_closed_form)})
    return out


def zmc_scan_adaptive(integrand_id: int, bounds, lists, n_first: int, n_max: int, target_stderr: float, seed: int,
                      out_mean, out_stderr, out_n, stream=None, *, precision: int = ZMC_PREC_F64,
                      fast_math: int = ZMC_FAST_MATH_DEFAULT, batch_points: int = 0, first_index: int = 0,
                      count: int = 0, consts=None, timing: bool = False) -> Optional[dict]:
    """include/zmc.h zmc_scan_adaptive.  out_n: int32/uint32 torch CUDA tensor (samples used per point)."""
    m = _Marshalled(bounds, lists, consts)
    pm, dm, lm = _tensor_ptr(out_mean)
    pe, de, le = _tensor_ptr(out_stderr)
    if (dm, lm) != (de, le) or out_n.element_size() != 4 or out_n.is_cuda != (lm == ZMC_LOC_DEVICE):
        raise ZmcError(ZMC_ERR_INVALID_ARG, "outputs must share dtype/location; out_n must be a 4-byte tensor in the same memory")
    o = _make_options(m, precision, dm, lm, ZMC_SCHED_AUTO, fast_math, batch_points, first_index, count)
    tm = zmc_timing() if timing else None
    _check(load().zmc_scan_adaptive(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_first, n_max, target_stderr, seed,
                                    ctypes.c_void_p(pm), ctypes.c_void_p(pe), ctypes.c_void_p(out_n.data_ptr()),
                                    ctypes.c_void_p(_stream_handle(stream)), ctypes.byref(o),
                                    ctypes.byref(tm) if timing else None))
    return tm.as_dict() if timing else None


def zmc_scan_farm(integrand_id: int, bounds, lists, n_samples: int, seed: int, out_mean, out_stderr, devices, *,
                  precision: int = ZMC_PREC_F64, schedule: int = ZMC_SCHED_AUTO, fast_math: int = ZMC_FAST_MATH_DEFAULT,
                  batch_points: int = 0, first_index: int = 0, count: int = 0, consts=None) -> dict:
    """zmc_scan over several GPUs of one node (host outputs, synchronous).  Returns the farm timing as a dict."""
    lib = load()
    m = _Marshalled(bounds, lists, consts)
    pm, dt_m, loc_m = _tensor_ptr(out_mean)
    pe, dt_e, loc_e = _tensor_ptr(out_stderr)
    if dt_m != dt_e or loc_m != ZMC_LOC_HOST or loc_e != ZMC_LOC_HOST:
        raise ValueError("zmc_scan_farm needs two host arrays of the same dtype")
    o = _make_options(m, precision, dt_m, ZMC_LOC_HOST, schedule, fast_math, batch_points, first_index, count)
    devs = (ctypes.c_int * len(devices))(*devices)
    tm = zmc_farm_timing()
    _check(lib.zmc_scan_farm(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_samples, seed, ctypes.c_void_p(pm),
                             ctypes.c_void_p(pe), devs, len(devices), ctypes.byref(o), ctypes.byref(tm)))
    n = tm.n_devices
    return {"wall_ms": tm.wall_ms, "n_batches": tm.n_batches, "batch_points": tm.batch_points, "n_devices": n,
            "batches_done": list(tm.batches_done[:n]), "busy_ms": list(tm.busy_ms[:n])}


def zmc_scan_farm_adaptive(integrand_id: int, bounds, lists, n_first: int, n_max: int, target_stderr: float, seed: int,
                           out_mean, out_stderr, out_n, devices, *, precision: int = ZMC_PREC_F64,
                           fast_math: int = ZMC_FAST_MATH_DEFAULT, batch_points: int = 0, first_index: int = 0,
                           count: int = 0, consts=None) -> dict:
    """zmc_scan_adaptive farmed over several GPUs (host outputs incl. out_n, synchronous)."""
    lib = load()
    m = _Marshalled(bounds, lists, consts)
    pm, dt_m, loc_m = _tensor_ptr(out_mean)
    pe, dt_e, loc_e = _tensor_ptr(out_stderr)
    if dt_m != dt_e or loc_m != ZMC_LOC_HOST or loc_e != ZMC_LOC_HOST or out_n.is_cuda or out_n.element_size() != 4:
        raise ValueError("zmc_scan_farm_adaptive needs host arrays (mean/stderr of one dtype, out_n 4-byte)")
    o = _make_options(m, precision, dt_m, ZMC_LOC_HOST, ZMC_SCHED_AUTO, fast_math, batch_points, first_index, count)
    devs = (ctypes.c_int * len(devices))(*devices)
    tm = zmc_farm_timing()
    _check(lib.zmc_scan_farm_adaptive(integrand_id, m.N, m.bounds_ptr(), m.M, m.c_lists, n_first, n_max, target_stderr, seed,
                                      ctypes.c_void_p(pm), ctypes.c_void_p(pe), ctypes.c_void_p(out_n.data_ptr()), devs,
                                      len(devices), ctypes.byref(o), ctypes.byref(tm)))
    n = tm.n_devices
    return {"wall_ms": tm.wall_ms, "n_batches": tm.n_batches, "batch_points": tm.batch_points, "n_devices": n,
            "batches_done": list(tm.batches_done[:n]), "busy_ms": list(tm.busy_ms[:n])}


def zmc_unregister_integrand(integrand_id: int):
    _check(load().zmc_unregister_integrand(integrand_id))


def zmc_register_integrand(name: str, body: str, N: int, M: int, n_consts: int = 0, flags: int = 0) -> int:
    """Compile a user integrand (body of `template <typename R> __device__ R g(const R* y, const R* x, const R* c)`)
    with NVRTC; returns its integrand id (the cached one if this integrand was registered before).  Raises ZmcError
    (status ZMC_ERR_COMPILE carries the NVRTC log)."""
    lib = load()
    out = ctypes.c_int(0)
    st = lib.zmc_register_integrand_ex(name.encode(), body.encode(), N, M, n_consts, flags, ctypes.byref(out))
    if st != ZMC_OK:
        log = (lib.zmc_last_compile_log() or b"").decode(errors="replace")
        raise ZmcError(st, lib.zmc_status_string(st).decode() + (": " + log[-2000:] if log else ""))
    return int(out.value)


def zmc_last_compile_log() -> str:
    return (load().zmc_last_compile_log() or b"").decode(errors="replace")


def zmc_version() -> str:
    return load().zmc_version().decode()


def zmc_status_string(status: int) -> str:
    return load().zmc_status_string(status).decode()


def zmc_shutdown():
    load().zmc_shutdown()


def scan_workload(w, *, schedule: int = ZMC_SCHED_AUTO, fast_math: int = ZMC_FAST_MATH_DEFAULT,
                  first_index: int = 0, count: int = 0, batch_points: Optional[int] = None,
                  host_out: Optional[bool] = None, out_mean=None, out_stderr=None, timing: bool = False,
                  stream=None, flags: int = 0):
    """Convenience for tests/bench: run a workloads.Workload; allocates the outputs (torch) unless given.
    Returns (out_mean, out_stderr, timing_dict_or_None); outputs are valid after the stream is synchronised."""
    import torch
    n_out = count if count else w.G - first_index
    dtype = torch.float32 if w.out_f32 else torch.float64
    host = w.host_out if host_out is None else host_out
    if out_mean is None:
        if host:
            out_mean = pinned_empty(n_out, dtype)
            out_stderr = pinned_empty(n_out, dtype)
        else:
            out_mean = torch.empty(n_out, dtype=dtype, device="cuda")
            out_stderr = torch.empty(n_out, dtype=dtype, device="cuda")
    tm = zmc_scan_ex(w.integrand_id, w.bounds, w.lists, w.n_samples, w.seed, out_mean, out_stderr, stream,
                     precision=w.precision, schedule=schedule, fast_math=fast_math,
                     batch_points=w.batch_points if batch_points is None else batch_points,
                     first_index=first_index, count=count, consts=w.consts, timing=timing, flags=flags)
    return out_mean, out_stderr, tm
