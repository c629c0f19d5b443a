"""paper_2412_13755_b200 — B200-native TPC cluster finder (binding of include/tpcclus.h).

Thin ctypes binding with the SAME names as the C-ABI: argument marshalling only, every step
of the path runs in the CUDA kernels of ``csrc/``.  PyTorch is used by callers for device
memory and streams (``tensor.data_ptr()``, ``torch.cuda.current_stream().cuda_stream``);
nothing here touches torch.  There is no CPU fallback: if the extension cannot be built or
loaded, or there is no sm_100 device, the calls raise.
"""
from __future__ import annotations

import ctypes
import threading

import numpy as np

from . import build as _build

TPCCLUS_OK = 0
TPCCLUS_ERR_INVALID = -1
TPCCLUS_ERR_GEOMETRY = -2
TPCCLUS_ERR_CAPACITY = -3
TPCCLUS_ERR_DIGIT = -4
TPCCLUS_ERR_CUDA = -5
TPCCLUS_ERR_NOMEM = -6
TPCCLUS_ERR_OCCUPANCY = -7
TPCCLUS_ERR_TOO_LARGE = -8
TPCCLUS_SELECT_STATIC_MAX_RECORDS = 1 << 24

TPCCLUS_FLAG_EDGE_PAD, TPCCLUS_FLAG_EDGE_TIME, TPCCLUS_FLAG_SATURATED, TPCCLUS_FLAG_SPLIT = 1, 2, 4, 8
TPCCLUS_OPT_STRICT_DIGITS, TPCCLUS_OPT_HOST_STAGING, TPCCLUS_OPT_BIN_DIRECT = 1, 2, 4

# record layouts of include/tpcclus.h
DIGIT_DTYPE = np.dtype([("row", "u1"), ("pad", "u1"), ("time", "<u2"), ("charge", "<f4")])
CLUSTER_DTYPE = np.dtype([
    ("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"), ("time", "<u4"),
    ("qmax_q16", "<u2"), ("ncells", "<u2"), ("qtot", "<f4"), ("dpad", "<f4"), ("dtime", "<f4"),
    ("sigma_pad", "<f4"), ("sigma_time", "<f4")])
assert DIGIT_DTYPE.itemsize == 8 and CLUSTER_DTYPE.itemsize == 32

EXPORTS = ("tpcclus_create", "tpcclus_run", "tpcclus_run_based", "tpcclus_result", "tpcclus_run_host", "tpcclus_run_tf_host",
           "tpcclus_select", "tpcclus_select_result", "tpcclus_select_static",
           "tpcclus_set_profiling", "tpcclus_get_profile", "tpcclus_launch_count", "tpcclus_device_bytes", "tpcclus_destroy", "tpcclus_strerror")


class tpcclus_geometry(ctypes.Structure):
    _fields_ = [("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
                ("npads", ctypes.POINTER(ctypes.c_uint16)),
                ("tf_time_bins", ctypes.c_uint32), ("max_core_bins", ctypes.c_uint32),
                ("halo_bins", ctypes.c_uint32),
                ("peak_min_q16", ctypes.c_uint16), ("options", ctypes.c_uint16),
                ("max_digits", ctypes.c_uint64), ("max_clusters", ctypes.c_uint64),
                ("bin_occupancy_pct", ctypes.c_uint32), ("reserved_", ctypes.c_uint32)]


class tpcclus_run_stats(ctypes.Structure):
    _fields_ = [("n_digits_in", ctypes.c_uint64), ("n_digits_dropped", ctypes.c_uint64),
                ("n_clusters", ctypes.c_uint64), ("status", ctypes.c_int32), ("cuda_error", ctypes.c_int32)]


class tpcclus_fragment(ctypes.Structure):
    _fields_ = [("h_digits", ctypes.c_void_p), ("n", ctypes.c_uint64),
                ("h_sector_offsets", ctypes.c_void_p),
                ("t_core_begin", ctypes.c_uint32), ("t_core_end", ctypes.c_uint32),
                ("t_time_base", ctypes.c_uint32), ("reserved_", ctypes.c_uint32)]


class tpcclus_cuts(ctypes.Structure):
    _fields_ = [("min_qtot", ctypes.c_float), ("min_qmax_q16", ctypes.c_uint16), ("min_ncells", ctypes.c_uint16),
                ("reject_flags", ctypes.c_uint8), ("reject_single_pad", ctypes.c_uint8),
                ("reject_single_time", ctypes.c_uint8), ("reserved_", ctypes.c_uint8)]


class TpcclusError(RuntimeError):
    def __init__(self, code, where, cuda_error=0):
        self.code, self.cuda_error = code, cuda_error
        msg = f"{where}: {tpcclus_strerror(code)} ({code})"
        if cuda_error:
            msg += f", cudaError {cuda_error}"
        super().__init__(msg)


_lock = threading.Lock()
_lib = None
_checked = False


def use_checked_build() -> None:
    """Select csrc/libtpcclus_checked.so (same sources with -DTPCCLUS_CHECKED: device asserts on every shared-memory
    and list index).  Must be called before the first use of the library; for tests/sanitizer_cases.py."""
    global _checked
    assert _lib is None, "the library is already loaded"
    _checked = True


def lib():
    """Load (building if needed) csrc/libtpcclus.so.  Raises if that is impossible."""
    global _lib
    with _lock:
        if _lib is None:
            L = ctypes.CDLL(_build.build(checked=_checked))
            vp, u64, u32 = ctypes.c_void_p, ctypes.c_uint64, ctypes.c_uint32
            L.tpcclus_create.restype = ctypes.c_int
            L.tpcclus_create.argtypes = [ctypes.POINTER(tpcclus_geometry), ctypes.c_int, ctypes.POINTER(vp)]
            L.tpcclus_run.restype = ctypes.c_int
            L.tpcclus_run.argtypes = [vp, vp, u64, vp, u32, u32, vp, u64, vp]
            L.tpcclus_run_based.restype = ctypes.c_int
            L.tpcclus_run_based.argtypes = [vp, vp, u64, vp, u32, u32, u32, vp, u64, vp]
            L.tpcclus_result.restype = ctypes.c_int
            L.tpcclus_result.argtypes = [vp, ctypes.POINTER(tpcclus_run_stats)]
            L.tpcclus_run_host.restype = ctypes.c_int
            L.tpcclus_run_host.argtypes = [vp, vp, u64, vp, u32, u32, vp, u64, ctypes.POINTER(tpcclus_run_stats)]
            L.tpcclus_run_tf_host.restype = ctypes.c_int
            L.tpcclus_run_tf_host.argtypes = [vp, ctypes.POINTER(tpcclus_fragment), u32, vp, u64,
                                              ctypes.POINTER(tpcclus_run_stats)]
            L.tpcclus_select.restype = ctypes.c_int
            L.tpcclus_select.argtypes = [vp, vp, u64, ctypes.POINTER(tpcclus_cuts), vp, u64, vp]
            L.tpcclus_select_static.restype = ctypes.c_int
            L.tpcclus_select_static.argtypes = [vp, u64, ctypes.POINTER(tpcclus_cuts), vp, u64, vp, vp]
            L.tpcclus_select_result.restype = ctypes.c_int
            L.tpcclus_select_result.argtypes = [vp, ctypes.POINTER(u64)]
            L.tpcclus_set_profiling.restype = ctypes.c_int
            L.tpcclus_set_profiling.argtypes = [vp, ctypes.c_int]
            L.tpcclus_get_profile.restype = ctypes.c_int
            L.tpcclus_get_profile.argtypes = [vp, ctypes.POINTER(ctypes.c_double), ctypes.POINTER(u64)]
            L.tpcclus_launch_count.restype = u64
            L.tpcclus_launch_count.argtypes = [vp]
            L.tpcclus_device_bytes.restype = u64
            L.tpcclus_device_bytes.argtypes = [vp]
            L.tpcclus_destroy.restype = None
            L.tpcclus_destroy.argtypes = [vp]
            L.tpcclus_strerror.restype = ctypes.c_char_p
            L.tpcclus_strerror.argtypes = [ctypes.c_int]
            _lib = L
    return _lib


def tpcclus_strerror(code: int) -> str:
    return lib().tpcclus_strerror(int(code)).decode()


def tpcclus_create(npads, *, n_sectors, tf_time_bins, max_core_bins=None, halo_bins=0, peak_min_q16=64,
                   options=0, max_digits, max_clusters=0, bin_occupancy_pct=0, cuda_device=0):
    """tpcclus_create(geometry, device) -> opaque context handle (int)."""
    npads = np.ascontiguousarray(npads, dtype=np.uint16)
    g = tpcclus_geometry()
    g.n_sectors, g.n_rows = int(n_sectors), int(npads.shape[0])
    g.npads = npads.ctypes.data_as(ctypes.POINTER(ctypes.c_uint16))
    g.tf_time_bins = int(tf_time_bins)
    g.max_core_bins = int(tf_time_bins if max_core_bins is None else max_core_bins)
    g.halo_bins, g.peak_min_q16, g.options = int(halo_bins), int(peak_min_q16), int(options)
    g.max_digits, g.max_clusters = int(max_digits), int(max_clusters)
    g.bin_occupancy_pct, g.reserved_ = int(bin_occupancy_pct), 0
    h = ctypes.c_void_p()
    rc = lib().tpcclus_create(ctypes.byref(g), int(cuda_device), ctypes.byref(h))
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_create")
    return h.value


def _offsets(sector_offsets):
    return np.ascontiguousarray(sector_offsets, dtype=np.uint64)


def tpcclus_run(ctx, d_digits_ptr, n, sector_offsets, t_core_begin, t_core_end, d_out_ptr, out_capacity,
                cuda_stream=0):
    """Asynchronous enqueue; pointers are DEVICE addresses (ints), sector_offsets a host array."""
    offs = _offsets(sector_offsets)
    rc = lib().tpcclus_run(ctx, d_digits_ptr, int(n), offs.ctypes.data, int(t_core_begin), int(t_core_end),
                           d_out_ptr, int(out_capacity), cuda_stream)
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_run")


def tpcclus_run_based(ctx, d_digits_ptr, n, sector_offsets, t_time_base, t_core_begin, t_core_end, d_out_ptr,
                      out_capacity, cuda_stream=0):
    """tpcclus_run for digits whose u16 time counts from t_time_base (time frames longer than 65536 bins)."""
    offs = _offsets(sector_offsets)
    rc = lib().tpcclus_run_based(ctx, d_digits_ptr, int(n), offs.ctypes.data, int(t_time_base), int(t_core_begin),
                                 int(t_core_end), d_out_ptr, int(out_capacity), cuda_stream)
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_run_based")


def tpcclus_result(ctx, check=True):
    """Synchronise the run and return its stats dict; raises on error unless check=False."""
    st = tpcclus_run_stats()
    rc = lib().tpcclus_result(ctx, ctypes.byref(st))
    out = dict(n_digits_in=st.n_digits_in, n_digits_dropped=st.n_digits_dropped, n_clusters=st.n_clusters,
               status=st.status, cuda_error=st.cuda_error)
    if check and rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_result", st.cuda_error)
    return out


def tpcclus_run_host(ctx, h_digits, sector_offsets, t_core_begin, t_core_end, h_out, check=True):
    """HOST numpy buffers in, HOST numpy records out (h_out: CLUSTER_DTYPE array, its length is the capacity)."""
    offs = _offsets(sector_offsets)
    st = tpcclus_run_stats()
    rc = lib().tpcclus_run_host(ctx, h_digits.ctypes.data, int(h_digits.shape[0]), offs.ctypes.data,
                                int(t_core_begin), int(t_core_end), h_out.ctypes.data, int(h_out.shape[0]),
                                ctypes.byref(st))
    out = dict(n_digits_in=st.n_digits_in, n_digits_dropped=st.n_digits_dropped, n_clusters=st.n_clusters,
               status=st.status, cuda_error=st.cuda_error)
    if check and rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_run_host", st.cuda_error)
    return out


def tpcclus_run_tf_host(ctx, fragments, h_out_ptr, out_capacity, check=True):
    """fragments: list of (h_digits_ptr, n, offsets ndarray(uint64), b, e[, t_time_base]); pointers are HOST addresses."""
    nf = len(fragments)
    arr = (tpcclus_fragment * nf)()
    keep = []
    for i, fr in enumerate(fragments):
        ptr, n, offs, b, e = fr[:5]
        o = _offsets(offs)
        keep.append(o)
        arr[i].h_digits, arr[i].n, arr[i].h_sector_offsets = ptr, int(n), o.ctypes.data
        arr[i].t_core_begin, arr[i].t_core_end = int(b), int(e)
        arr[i].t_time_base, arr[i].reserved_ = (int(fr[5]) if len(fr) > 5 else 0), 0
    stats = (tpcclus_run_stats * nf)()
    rc = lib().tpcclus_run_tf_host(ctx, arr, nf, h_out_ptr, int(out_capacity), stats)
    out = [dict(n_digits_in=s.n_digits_in, n_digits_dropped=s.n_digits_dropped, n_clusters=s.n_clusters,
                status=s.status, cuda_error=s.cuda_error) for s in stats]
    if check and rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_run_tf_host")
    return out


def tpcclus_select(ctx, d_in_ptr, n, d_out_ptr, out_capacity, cuda_stream=0, *, min_qtot=0.0, min_qmax_q16=0,
                   min_ncells=0, reject_flags=0, reject_single_pad=False, reject_single_time=False):
    """Asynchronous D13 selection over n DEVICE records; collect the count with tpcclus_select_result."""
    cuts = tpcclus_cuts(float(min_qtot), int(min_qmax_q16), int(min_ncells), int(reject_flags),
                        1 if reject_single_pad else 0, 1 if reject_single_time else 0, 0)
    rc = lib().tpcclus_select(ctx, d_in_ptr, int(n), ctypes.byref(cuts), d_out_ptr, int(out_capacity), cuda_stream)
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_select")


def tpcclus_select_static(d_in_ptr, n, d_out_ptr, out_capacity, d_n_kept_ptr, cuda_stream=0, *, min_qtot=0.0, min_qmax_q16=0,
                          min_ncells=0, reject_flags=0, reject_single_pad=False, reject_single_time=False):
    """The D13 selection without a context and without any allocation (scratch in a fixed device array inside the
    library): n <= TPCCLUS_SELECT_STATIC_MAX_RECORDS DEVICE records on the current device; the kept count goes to the
    8-byte DEVICE word d_n_kept_ptr in stream order.  Calls that overlap on the GPU race (include/tpcclus.h)."""
    cuts = tpcclus_cuts(float(min_qtot), int(min_qmax_q16), int(min_ncells), int(reject_flags),
                        1 if reject_single_pad else 0, 1 if reject_single_time else 0, 0)
    rc = lib().tpcclus_select_static(d_in_ptr, int(n), ctypes.byref(cuts), d_out_ptr, int(out_capacity), d_n_kept_ptr, cuda_stream)
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_select_static")


def tpcclus_select_result(ctx, check=True) -> int:
    """Waits for the selection; returns the number of records kept (the number required)."""
    k = ctypes.c_uint64()
    rc = lib().tpcclus_select_result(ctx, ctypes.byref(k))
    if rc != TPCCLUS_OK and (check or rc != TPCCLUS_ERR_CAPACITY):
        raise TpcclusError(rc, "tpcclus_select_result")
    return int(k.value)


def tpcclus_set_profiling(ctx, on: bool) -> None:
    rc = lib().tpcclus_set_profiling(ctx, 1 if on else 0)
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_set_profiling")


def tpcclus_get_profile(ctx):
    """-> ({"k_init": ms, "k_bin": ms, "k_tile": ms} summed over runs, n_runs)."""
    ms = (ctypes.c_double * 3)()
    n = ctypes.c_uint64()
    rc = lib().tpcclus_get_profile(ctx, ms, ctypes.byref(n))
    if rc != TPCCLUS_OK:
        raise TpcclusError(rc, "tpcclus_get_profile")
    return dict(k_init=ms[0], k_bin=ms[1], k_tile=ms[2]), int(n.value)


def tpcclus_launch_count(ctx) -> int:
    return int(lib().tpcclus_launch_count(ctx))


def tpcclus_device_bytes(ctx) -> int:
    return int(lib().tpcclus_device_bytes(ctx))


def tpcclus_destroy(ctx) -> None:
    if ctx:
        lib().tpcclus_destroy(ctx)
