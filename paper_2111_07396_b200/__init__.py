"""paper_2111_07396_b200 -- B200-native batched SuperSmoother periodogram (arXiv 2111.07396).

Thin ctypes binding over the C ABI declared in include/ss_periodogram.h.  Argument marshalling
only: every step of the hot path runs in the CUDA kernels of libss_b200.so.  PyTorch supplies device
memory and streams.  There is no CPU fallback: if the library is missing or no CUDA device is
present, calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import numpy as np

CROSS_VALIDATION = 0
GENERALIZED_VALIDATION = 1
PATH_AUTO, PATH_WARP, PATH_BLOCK, PATH_STAGE, PATH_GROUP, PATH_CLUSTER = 0, 1, 2, 3, 4, 5
PRECISION_F64, PRECISION_MIXED = 0, 1
SS_OK, SS_ERR_INVALID_ARG, SS_ERR_OUT_OF_MEMORY, SS_ERR_CUDA, SS_ERR_UNSUPPORTED = range(5)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libss_b200.so")

EXPORTS = ["ss_default_options", "ss_periodogram", "ss_periodogram_ex", "ss_periodogram_host",
           "ss_plan", "ss_workspace_bytes", "ss_paper_footprint_bytes", "ss_paper_batches",
           "ss_path_for_n", "ss_debug_eval", "ss_microbench", "ss_last_launch_count", "ss_last_kernel_ms", "ss_last_kernel_count",
           "ss_last_error", "ss_version", "ss_release_workspace", "ss_periodogram_peaks", "ss_periodogram_peaks_host", "ss_synchronize",
           "ss_periodogram_static"]


class SSError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"ss status {status}: {msg}")
        self.status = status


class Options(C.Structure):
    _fields_ = [("alpha", C.c_double), ("span", C.c_double), ("iper", C.c_int),
                ("force_path", C.c_int), ("stream", C.c_void_p), ("workspace_cap", C.c_size_t),
                ("freq_tile", C.c_int64), ("skip_validation", C.c_int), ("profile", C.c_int),
                ("k_begin", C.c_int64), ("k_count", C.c_int64), ("precision", C.c_int), ("shared_times", C.c_int), ("workspace", C.c_void_p), ("workspace_bytes", C.c_size_t),
                ("offsets_host", C.c_void_p), ("async_mode", C.c_int), ("defer_capacity", C.c_uint)]


class Plan(C.Structure):
    _fields_ = [("n_freq_tiles", C.c_int64), ("freq_per_tile", C.c_int64),
                ("n_object_tiles", C.c_int64), ("objects_per_tile", C.c_int64),
                ("tile_bytes", C.c_size_t), ("fixed_bytes", C.c_size_t),
                ("stage_bytes", C.c_size_t), ("total_bytes", C.c_size_t)]


_lib = None


def load():
    """dlopen libss_b200.so and set signatures.  The library is rebuilt with nvcc first when it is missing or
    when the hash of the sources it was built from (stored beside it) no longer matches csrc/ and include/: an
    edited kernel can never be exercised through a stale binary."""
    global _lib
    if _lib is not None:
        return _lib
    from . import _build
    if os.environ.get("SS_REBUILD") or not _build.is_fresh():
        _build.build(force=True)
    if not os.path.exists(LIB_PATH):
        raise SSError(SS_ERR_CUDA, f"{LIB_PATH} is missing and could not be built")
    L = C.CDLL(LIB_PATH)
    vp, d, i64 = C.c_void_p, C.c_double, C.c_int64
    L.ss_default_options.argtypes = [C.POINTER(Options)]
    L.ss_default_options.restype = None
    common = [vp, vp, vp, vp, i64, d, d, i64, C.c_int, vp, vp, vp]
    L.ss_periodogram.argtypes = common
    L.ss_periodogram_ex.argtypes = common + [C.POINTER(Options)]
    L.ss_periodogram_host.argtypes = common + [C.POINTER(Options)]
    L.ss_periodogram_static.argtypes = [vp, vp, vp, vp, vp, i64, d, d, i64, C.c_int, vp, vp, vp, vp]
    L.ss_plan.argtypes = [i64, i64, i64, i64, C.c_int, C.c_size_t, C.c_int, C.c_int, C.POINTER(Plan)]
    L.ss_workspace_bytes.argtypes = [i64, i64, i64, i64, C.c_int]
    L.ss_workspace_bytes.restype = C.c_size_t
    L.ss_paper_footprint_bytes.argtypes = [i64, i64]
    L.ss_paper_footprint_bytes.restype = d
    L.ss_paper_batches.argtypes = [i64, i64, C.c_int, d, d]
    L.ss_paper_batches.restype = i64
    L.ss_path_for_n.argtypes = [i64, C.c_int]
    L.ss_debug_eval.argtypes = [vp, vp, vp, i64, d, C.c_int, C.POINTER(Options), vp, vp, vp]
    L.ss_microbench.argtypes = [C.POINTER(d), C.POINTER(d), vp]
    L.ss_last_launch_count.restype = i64
    L.ss_last_kernel_ms.restype = d
    L.ss_last_kernel_count.restype = i64
    L.ss_last_error.restype = C.c_char_p
    L.ss_version.restype = C.c_int
    L.ss_release_workspace.restype = None
    peaks = [vp, i64, i64, i64, d, d, C.c_int, vp, vp, vp]
    L.ss_periodogram_peaks.argtypes = peaks + [vp]
    L.ss_periodogram_peaks_host.argtypes = peaks
    _lib = L
    return L


def _check(st):
    if st != SS_OK:
        raise SSError(st, load().ss_last_error().decode())


def default_options(**kw) -> Options:
    o = Options()
    load().ss_default_options(C.byref(o))
    for k, v in kw.items():
        if not hasattr(o, k):
            raise TypeError(f"unknown option {k}")
        setattr(o, k, v)
    return o


def synchronize() -> None:
    """Complete this thread's pending asynchronous call (ss_synchronize)."""
    _check(load().ss_synchronize())


def release_workspace() -> None:
    """Free the device buffers the library caches between calls of this thread (ss_release_workspace)."""
    load().ss_release_workspace()


def version() -> int:
    return load().ss_version()


def last_launch_count() -> int:
    return int(load().ss_last_launch_count())


def last_kernel_ms():
    """(total ms, launches) of the eval kernels of the last call made with options.profile = 1."""
    L = load()
    return float(L.ss_last_kernel_ms()), int(L.ss_last_kernel_count())


def path_for_n(n: int, mode: int = CROSS_VALIDATION) -> int:
    return load().ss_path_for_n(int(n), int(mode))


def plan(n_points_total, max_n, n_objects, n_freq, mode=CROSS_VALIDATION, cap_bytes=2 ** 62,
         host_tiles=False, want_pgram=True) -> Plan:
    p = Plan()
    _check(load().ss_plan(int(n_points_total), int(max_n), int(n_objects), int(n_freq), int(mode),
                          int(cap_bytes), int(bool(host_tiles)), int(bool(want_pgram)), C.byref(p)))
    return p


def workspace_bytes(n_points_total, max_n, n_objects, n_freq, mode=CROSS_VALIDATION) -> int:
    return int(load().ss_workspace_bytes(int(n_points_total), int(max_n), int(n_objects), int(n_freq), int(mode)))


def paper_footprint_bytes(n_t, n_f) -> float:
    return load().ss_paper_footprint_bytes(int(n_t), int(n_f))


def paper_batches(n_t, n_f, mode, device_gib, beta=0.75) -> int:
    return int(load().ss_paper_batches(int(n_t), int(n_f), int(mode), float(device_gib), float(beta)))


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise SSError(SS_ERR_CUDA, "no CUDA device: the SuperSmoother periodogram has no CPU path")
    return torch


def _dev_ptr(t, dtype, name):
    torch = _torch()
    if t is None:
        return None
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError(f"{name} must be a contiguous CUDA tensor of dtype {dtype}")
    return C.c_void_p(t.data_ptr())


def ss_periodogram(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode=CROSS_VALIDATION,
                   pgram_out=None, best_freq_out=None, best_index_out=None, options: Options | None = None):
    """Device-tensor call (include/ss_periodogram.h: ss_periodogram_ex).  Output tensors are written
    in place; work is enqueued on torch's current stream unless options.stream is set."""
    torch = _torch()
    L = load()
    o = options if options is not None else default_options()
    if not o.stream:
        o.stream = torch.cuda.current_stream().cuda_stream
    st = L.ss_periodogram_ex(_dev_ptr(times, torch.float64, "times"), _dev_ptr(mags, torch.float64, "mags"),
                             _dev_ptr(errs, torch.float64, "errs"), _dev_ptr(offsets, torch.int64, "offsets"),
                             int(n_objects), float(f_min), float(f_max), int(n_freq), int(mode),
                             _dev_ptr(pgram_out, torch.float64, "pgram_out"),
                             _dev_ptr(best_freq_out, torch.float64, "best_freq_out"),
                             _dev_ptr(best_index_out, torch.int64, "best_index_out"), C.byref(o))
    _check(st)


STATIC_SCRATCH_BYTES = 32 << 20      # SS_STATIC_SCRATCH_BYTES


def ss_periodogram_static(times, mags, errs, offsets, offsets_host, n_objects, f_min, f_max, n_freq,
                          mode=CROSS_VALIDATION, pgram_out=None, best_freq_out=None, best_index_out=None, stream=None):
    """Device-tensor call that allocates nothing on the device (include/ss_periodogram.h: ss_periodogram_static):
    the workspace is the library's built-in scratch array of STATIC_SCRATCH_BYTES.  offsets_host is a C-contiguous
    int64 numpy copy of offsets.  Calls that overlap on one GPU race on that array."""
    torch = _torch()
    L = load()
    if not (isinstance(offsets_host, np.ndarray) and offsets_host.dtype == np.int64 and offsets_host.flags["C_CONTIGUOUS"]
            and offsets_host.size == int(n_objects) + 1):
        raise TypeError("offsets_host must be a C-contiguous int64 numpy array of n_objects + 1 values")
    if stream is None:
        stream = torch.cuda.current_stream().cuda_stream
    st = L.ss_periodogram_static(_dev_ptr(times, torch.float64, "times"), _dev_ptr(mags, torch.float64, "mags"),
                                 _dev_ptr(errs, torch.float64, "errs"), _dev_ptr(offsets, torch.int64, "offsets"),
                                 C.c_void_p(offsets_host.ctypes.data), int(n_objects), float(f_min), float(f_max),
                                 int(n_freq), int(mode), _dev_ptr(pgram_out, torch.float64, "pgram_out"),
                                 _dev_ptr(best_freq_out, torch.float64, "best_freq_out"),
                                 _dev_ptr(best_index_out, torch.int64, "best_index_out"), C.c_void_p(stream))
    _check(st)


def _host_ptr(a, dtype, name):
    if a is None:
        return None
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or not a.is_contiguous():
                raise TypeError(f"{name} must be a contiguous host tensor")
            return C.c_void_p(a.data_ptr())
    except ImportError:
        pass
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]):
        raise TypeError(f"{name} must be a C-contiguous numpy array of dtype {dtype}")
    return C.c_void_p(a.ctypes.data)


def ss_periodogram_host(times, mags, errs, offsets, n_objects, f_min, f_max, n_freq, mode=CROSS_VALIDATION,
                        pgram_out=None, best_freq_out=None, best_index_out=None, options: Options | None = None):
    """Host-array call (numpy arrays or pinned/pageable CPU tensors); copies and tiling happen inside
    the library (ss_periodogram_host)."""
    torch = _torch()
    L = load()
    o = options if options is not None else default_options()
    if not o.stream:
        o.stream = torch.cuda.current_stream().cuda_stream
    st = L.ss_periodogram_host(_host_ptr(times, np.float64, "times"), _host_ptr(mags, np.float64, "mags"),
                               _host_ptr(errs, np.float64, "errs"), _host_ptr(offsets, np.int64, "offsets"),
                               int(n_objects), float(f_min), float(f_max), int(n_freq), int(mode),
                               _host_ptr(pgram_out, np.float64, "pgram_out"),
                               _host_ptr(best_freq_out, np.float64, "best_freq_out"),
                               _host_ptr(best_index_out, np.int64, "best_index_out"), C.byref(o))
    _check(st)


@dataclass
class Result:
    pgram: np.ndarray | None
    best_freq: np.ndarray
    best_index: np.ndarray


def periodogram(times, mags, errs, offsets, f_min, f_max, n_freq, mode=CROSS_VALIDATION,
                want_pgram=True, **opts) -> Result:
    """Convenience wrapper: numpy in, numpy out, through ss_periodogram_host."""
    times = np.ascontiguousarray(times, dtype=np.float64)
    mags = np.ascontiguousarray(mags, dtype=np.float64)
    errs = np.ascontiguousarray(errs, dtype=np.float64)
    offsets = np.ascontiguousarray(offsets, dtype=np.int64)
    n_obj = len(offsets) - 1
    k_begin = int(opts.get("k_begin", 0))
    n_cols = int(opts.get("k_count", 0)) or int(n_freq) - k_begin
    pg = np.empty((n_obj, n_cols)) if want_pgram else None
    bf = np.empty(n_obj)
    bi = np.empty(n_obj, dtype=np.int64)
    ss_periodogram_host(times, mags, errs, offsets, n_obj, f_min, f_max, n_freq, mode, pg, bf, bi,
                        default_options(**opts))
    return Result(pg, bf, bi)


def ss_periodogram_peaks(pgram, n_objects, n_freq, row_stride, f_min, f_max, n_peaks, peak_index_out,
                         peak_power_out=None, peak_freq_out=None):
    """Device-tensor call (include/ss_periodogram.h: ss_periodogram_peaks); enqueued on torch's current stream."""
    torch = _torch()
    _check(load().ss_periodogram_peaks(_dev_ptr(pgram, torch.float64, "pgram"), int(n_objects), int(n_freq), int(row_stride),
                                       float(f_min), float(f_max), int(n_peaks),
                                       _dev_ptr(peak_index_out, torch.int64, "peak_index_out"),
                                       _dev_ptr(peak_power_out, torch.float64, "peak_power_out"),
                                       _dev_ptr(peak_freq_out, torch.float64, "peak_freq_out"),
                                       C.c_void_p(torch.cuda.current_stream().cuda_stream)))


def peaks(pgram, f_min, f_max, n_peaks):
    """Convenience wrapper: numpy periodogram [n_objects, n_freq] in, (index, power, freq) [n_objects, n_peaks] out,
    through ss_periodogram_peaks_host."""
    _torch()
    pgram = np.ascontiguousarray(pgram, dtype=np.float64)
    n_obj, n_freq = pgram.shape
    pi = np.empty((n_obj, n_peaks), dtype=np.int64)
    pv = np.empty((n_obj, n_peaks))
    pf = np.empty((n_obj, n_peaks))
    _check(load().ss_periodogram_peaks_host(_host_ptr(pgram, np.float64, "pgram"), n_obj, n_freq, n_freq, float(f_min),
                                            float(f_max), int(n_peaks), _host_ptr(pi, np.int64, "pi"),
                                            _host_ptr(pv, np.float64, "pv"), _host_ptr(pf, np.float64, "pf")))
    return pi, pv, pf


def debug_eval(times, mags, errs, freq, mode=CROSS_VALIDATION, **opts):
    """One (object, frequency) eval: returns (P, smooth in phase order, permutation).  Test hook."""
    torch = _torch()
    L = load()
    dev = torch.device("cuda")
    t = torch.as_tensor(np.ascontiguousarray(times, dtype=np.float64), device=dev)
    y = torch.as_tensor(np.ascontiguousarray(mags, dtype=np.float64), device=dev)
    e = torch.as_tensor(np.ascontiguousarray(errs, dtype=np.float64), device=dev)
    n = t.numel()
    smo = torch.empty(n, dtype=torch.float64, device=dev)
    perm = torch.empty(n, dtype=torch.int32, device=dev)
    p = torch.empty(1, dtype=torch.float64, device=dev)
    o = default_options(**opts)
    o.stream = torch.cuda.current_stream().cuda_stream
    _check(L.ss_debug_eval(C.c_void_p(t.data_ptr()), C.c_void_p(y.data_ptr()), C.c_void_p(e.data_ptr()), n,
                           float(freq), int(mode), C.byref(o), C.c_void_p(smo.data_ptr()),
                           C.c_void_p(perm.data_ptr()), C.c_void_p(p.data_ptr())))
    return float(p.item()), smo.cpu().numpy(), perm.cpu().numpy()


def microbench():
    """(fp64 FLOP/s, shared-memory B/s) measured on the current device (roofline denominators)."""
    torch = _torch()
    a, b = C.c_double(), C.c_double()
    _check(load().ss_microbench(C.byref(a), C.byref(b), C.c_void_p(torch.cuda.current_stream().cuda_stream)))
    return a.value, b.value
