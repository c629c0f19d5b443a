"""ORACLE binding — test infrastructure, not product.

Loads ``oracle/libtpc_oracle.so`` (plain single-threaded C++, ``tpc_oracle.cpp``) through
ctypes.  Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` leg may import this module.  It imports nothing from
``paper_2412_13755_b200`` and the product imports nothing from here.

The record dtypes below restate BASELINE.json:configs[0] (8-byte digit) and SURVEY.md §8(b)
(32-byte cluster) on their own.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "tpc_oracle.cpp")
# TPC_ORACLE_SANITIZE=1: the checker itself built with -fsanitize=address,undefined, for
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) TPC_ORACLE_SANITIZE=1 python -m pytest tests -m "not gpu"
_SANITIZE = os.environ.get("TPC_ORACLE_SANITIZE") == "1"
_LIB = os.path.join(_HERE, "libtpc_oracle_san.so" if _SANITIZE else "libtpc_oracle.so")

DIGIT_DTYPE = np.dtype(
    [("row", "u1"), ("pad", "u1"), ("time", "<u2"), ("charge", "<f4")], align=False
)
CLUSTER_DTYPE = np.dtype(
    [
        ("sector", "u1"), ("row", "u1"), ("pad", "u1"), ("flags", "u1"),
        ("time", "<u4"),
        ("qmax_q16", "<u2"), ("ncells", "<u2"),
        ("qtot", "<f4"), ("dpad", "<f4"), ("dtime", "<f4"),
        ("sigma_pad", "<f4"), ("sigma_time", "<f4"),
    ],
    align=False,
)
assert DIGIT_DTYPE.itemsize == 8 and CLUSTER_DTYPE.itemsize == 32

FLAG_EDGE_PAD, FLAG_EDGE_TIME, FLAG_SATURATED, FLAG_SPLIT = 1, 2, 4, 8


class _Params(ctypes.Structure):
    _fields_ = [
        ("n_sectors", ctypes.c_uint32), ("n_rows", ctypes.c_uint32),
        ("npads", ctypes.POINTER(ctypes.c_uint16)),
        ("tf_time_bins", ctypes.c_uint32), ("halo_bins", ctypes.c_uint32),
        ("peak_min_q16", ctypes.c_uint16), ("reserved", ctypes.c_uint16),
        ("t_time_base", ctypes.c_uint32),
    ]


class _Stats(ctypes.Structure):
    _fields_ = [
        ("n_digits_in", ctypes.c_uint64), ("n_digits_dropped", ctypes.c_uint64),
        ("n_duplicates", ctypes.c_uint64), ("n_clusters", ctypes.c_uint64),
        ("sum_q16_loaded", ctypes.c_uint64), ("sum_W", ctypes.c_uint64),
    ]


class _Cuts(ctypes.Structure):
    _fields_ = [
        ("min_qtot", ctypes.c_float), ("min_qmax_q16", ctypes.c_uint16), ("min_ncells", ctypes.c_uint16),
        ("reject_flags", ctypes.c_uint8), ("reject_single_pad", ctypes.c_uint8),
        ("reject_single_time", ctypes.c_uint8), ("reserved", ctypes.c_uint8),
    ]


_lock = threading.Lock()
_lib = None


def build(force: bool = False) -> str:
    """Compile the oracle with g++ (no CUDA, no other dependency)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + ".tmp%d" % os.getpid()
        subprocess.check_call(
            ["g++", "-O2", "-std=c++17", "-shared", "-fPIC", "-Wall", "-Wextra",
             *(["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
               if _SANITIZE else []), _SRC, "-o", tmp]
        )
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    with _lock:
        if _lib is None:
            lib = ctypes.CDLL(build())
            lib.tpc_oracle_run.restype = ctypes.c_int
            lib.tpc_oracle_run.argtypes = [
                ctypes.POINTER(_Params), ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p,
                ctypes.c_uint32, ctypes.c_uint32, ctypes.c_void_p, ctypes.c_uint64,
                ctypes.POINTER(_Stats),
            ]
            lib.tpc_oracle_quantise.restype = ctypes.c_uint16
            lib.tpc_oracle_quantise.argtypes = [ctypes.c_float]
            lib.tpc_oracle_peak_flags.restype = ctypes.c_int64
            lib.tpc_oracle_peak_flags.argtypes = [
                ctypes.POINTER(_Params), ctypes.c_void_p, ctypes.c_uint64, ctypes.c_void_p,
                ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32, ctypes.c_uint32,
                ctypes.c_void_p, ctypes.c_void_p,
            ]
            lib.tpc_oracle_select.restype = ctypes.c_uint64
            lib.tpc_oracle_select.argtypes = [ctypes.c_void_p, ctypes.c_uint64, ctypes.POINTER(_Cuts),
                                              ctypes.c_void_p, ctypes.c_uint64]
            _lib = lib
    return _lib


def _params(npads, n_sectors, tf_time_bins, halo_bins, peak_min_q16, t_time_base=0):
    npads = np.ascontiguousarray(npads, dtype=np.uint16)
    p = _Params()
    p.n_sectors = int(n_sectors)
    p.n_rows = int(npads.shape[0])
    p.npads = npads.ctypes.data_as(ctypes.POINTER(ctypes.c_uint16))
    p.tf_time_bins = int(tf_time_bins)
    p.halo_bins = int(halo_bins)
    p.peak_min_q16 = int(peak_min_q16)
    p.t_time_base = int(t_time_base)
    return p, npads


def quantise(charge: float) -> int:
    """D1 for one value."""
    return int(_load().tpc_oracle_quantise(ctypes.c_float(charge)))


def run(digits, sector_offsets, npads, *, n_sectors, tf_time_bins, t_core_begin=0,
        t_core_end=None, halo_bins=0, peak_min_q16=64, capacity=None, t_time_base=0):
    """Cluster one fragment.  Returns (clusters[CLUSTER_DTYPE], stats dict).

    digits: array of DIGIT_DTYPE grouped per sector by sector_offsets[n_sectors+1]; a digit's global time
    bin is t_time_base + digit.time (reading A19: time frames longer than 65536 bins).
    """
    lib = _load()
    digits = np.ascontiguousarray(digits, dtype=DIGIT_DTYPE)
    offs = np.ascontiguousarray(sector_offsets, dtype=np.uint64)
    assert offs.shape[0] == n_sectors + 1
    if t_core_end is None:
        t_core_end = tf_time_bins
    prm, keep = _params(npads, n_sectors, tf_time_bins, halo_bins, peak_min_q16, t_time_base)
    st = _Stats()
    if capacity is None:
        # count first, then allocate exactly
        rc = lib.tpc_oracle_run(ctypes.byref(prm), digits.ctypes.data, digits.shape[0],
                                offs.ctypes.data, t_core_begin, t_core_end, None, 0,
                                ctypes.byref(st))
        if rc != 0:
            raise ValueError("tpc_oracle_run: bad arguments")
        capacity = int(st.n_clusters)
    out = np.zeros(int(capacity), dtype=CLUSTER_DTYPE)
    rc = lib.tpc_oracle_run(ctypes.byref(prm), digits.ctypes.data, digits.shape[0],
                            offs.ctypes.data, t_core_begin, t_core_end,
                            out.ctypes.data if capacity else None, capacity, ctypes.byref(st))
    if rc != 0:
        raise ValueError("tpc_oracle_run: bad arguments")
    del keep
    stats = {k: int(getattr(st, k)) for k, _ in _Stats._fields_}
    return out[: min(int(st.n_clusters), int(capacity))], stats


def peak_flags(digits, sector_offsets, npads, *, n_sectors, tf_time_bins, sector, row,
               t_core_begin=0, t_core_end=None, halo_bins=0, peak_min_q16=64, t_time_base=0):
    """D4 flags and the q16 map of one (sector,row): two arrays [ntime_loaded, npads[row]]."""
    lib = _load()
    digits = np.ascontiguousarray(digits, dtype=DIGIT_DTYPE)
    offs = np.ascontiguousarray(sector_offsets, dtype=np.uint64)
    if t_core_end is None:
        t_core_end = tf_time_bins
    prm, keep = _params(npads, n_sectors, tf_time_bins, halo_bins, peak_min_q16, t_time_base)
    lo = max(0, t_core_begin - halo_bins)
    hi = min(tf_time_bins, t_core_end + halo_bins)
    w = int(keep[row])
    flags = np.zeros((hi - lo, w), dtype=np.uint8)
    q = np.zeros((hi - lo, w), dtype=np.uint16)
    n = lib.tpc_oracle_peak_flags(ctypes.byref(prm), digits.ctypes.data, digits.shape[0],
                                  offs.ctypes.data, t_core_begin, t_core_end, sector, row,
                                  flags.ctypes.data, q.ctypes.data)
    assert n == hi - lo
    return flags, q


def select(clusters, *, min_qtot=0.0, min_qmax_q16=0, min_ncells=0, reject_flags=0, reject_single_pad=False,
           reject_single_time=False, capacity=None):
    """D13: order-preserving quality selection over a cluster list.  Returns (kept records, number kept)."""
    lib = _load()
    clusters = np.ascontiguousarray(clusters, dtype=CLUSTER_DTYPE)
    cuts = _Cuts(float(min_qtot), int(min_qmax_q16), int(min_ncells), int(reject_flags),
                 1 if reject_single_pad else 0, 1 if reject_single_time else 0, 0)
    cap = len(clusters) if capacity is None else int(capacity)
    out = np.zeros(cap, dtype=CLUSTER_DTYPE)
    kept = int(lib.tpc_oracle_select(clusters.ctypes.data, len(clusters), ctypes.byref(cuts),
                                     out.ctypes.data if cap else None, cap))
    return out[: min(kept, cap)], kept
