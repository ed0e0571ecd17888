"""CPU ORACLE for the RFIm sigma cuts -- TEST INFRASTRUCTURE ONLY.

ctypes front end of ``oracle/rfim_oracle.c`` (see ``rfim_oracle.h`` for the
contract and the passages of PAPER.md each function follows).  Only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from
``paper_2001_03389_b200`` and the product imports nothing from here.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rfim_oracle.c")
_LIB = os.path.join(_HERE, "librfim_oracle.so")

U8, F32 = 0, 1
MEAN, MEDIAN = 0, 1


class _Opts(ctypes.Structure):
    _fields_ = [
        ("sample_stride", ctypes.c_int64),
        ("window", ctypes.c_int32),
        ("bin_size", ctypes.c_int32),
        ("out", ctypes.c_void_p),
        ("flags", ctypes.c_void_p),
        ("counts", ctypes.c_void_p),
        ("reserved", ctypes.c_void_p),
    ]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no CUDA, no headers from the product)."""
    stale = (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < max(
        os.path.getmtime(_SRC), os.path.getmtime(os.path.join(_HERE, "rfim_oracle.h")))
    if force or stale:
        subprocess.check_call(
            ["gcc", "-O2", "-std=c11", "-Wall", "-Wextra", "-shared", "-fPIC", "-o", _LIB, _SRC, "-lm"])
    return _LIB


_lib = None


def lib() -> ctypes.CDLL:
    global _lib
    if _lib is None:
        _lib = ctypes.CDLL(build())
        sig = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
               ctypes.POINTER(ctypes.c_double), ctypes.c_int, ctypes.c_int, ctypes.POINTER(_Opts)]
        for name in ("rfim_oracle_time_sigma_cut", "rfim_oracle_freq_sigma_cut"):
            fn = getattr(_lib, name)
            fn.argtypes = sig
            fn.restype = ctypes.c_int
        _lib.rfim_oracle_quantise_threshold.argtypes = [ctypes.c_double]
        _lib.rfim_oracle_quantise_threshold.restype = ctypes.c_uint64
        _lib.rfim_oracle_stats_u8.argtypes = [ctypes.c_void_p, ctypes.c_int64,
                                              ctypes.POINTER(ctypes.c_uint64), ctypes.POINTER(ctypes.c_uint64)]
        _lib.rfim_oracle_stats_u8.restype = None
        _lib.rfim_oracle_stats_f32.argtypes = [ctypes.c_void_p, ctypes.c_int64,
                                               ctypes.POINTER(ctypes.c_double), ctypes.POINTER(ctypes.c_double)]
        _lib.rfim_oracle_stats_f32.restype = None
    return _lib


def _dtype_code(a: np.ndarray) -> int:
    if a.dtype == np.uint8:
        return U8
    if a.dtype == np.float32:
        return F32
    raise TypeError("oracle: dtype must be uint8 or float32")


def _run(fn_name, data, thresholds, policy, window, bin_size, want_flags, want_counts):
    """data: C-contiguous [beams][channels][samples] ndarray (not modified).
    Returns (cleaned, flags or None, counts or None)."""
    a = np.ascontiguousarray(data)
    if a.ndim != 3:
        raise ValueError("oracle: data must be [beams][channels][samples]")
    out = a.copy()
    b, c, s = out.shape
    th = np.asarray(thresholds, dtype=np.float64)
    n = int(th.size)
    flags = np.zeros(out.shape, dtype=np.uint8) if want_flags else None
    counts = np.zeros(max(n, 1), dtype=np.uint64) if want_counts else None
    o = _Opts(0, int(window), int(bin_size), None,
              flags.ctypes.data if flags is not None else None,
              counts.ctypes.data if counts is not None else None, None)
    st = getattr(lib(), fn_name)(
        out.ctypes.data, b, c, s, _dtype_code(out),
        th.ctypes.data_as(ctypes.POINTER(ctypes.c_double)), n, int(policy), ctypes.byref(o))
    if st != 0:
        raise ValueError(f"oracle: {fn_name} returned status {st}")
    return out, flags, (counts[:n] if counts is not None else None)


def time_sigma_cut(data, thresholds, policy=MEAN, window=0, want_flags=True, want_counts=True):
    """TDSC on [beams][channels][samples]; returns (cleaned, flags, counts)."""
    return _run("rfim_oracle_time_sigma_cut", data, thresholds, policy, window, 0, want_flags, want_counts)


def freq_sigma_cut(data, thresholds, policy=MEAN, bin_size=0, want_flags=True, want_counts=True):
    """FDSC on [beams][channels][samples]; returns (cleaned, flags, counts)."""
    return _run("rfim_oracle_freq_sigma_cut", data, thresholds, policy, 0, bin_size, want_flags, want_counts)


def raw_call(fn_name, data_ptr, beams, channels, samples, dtype, thresholds, policy, opts=None):
    """Direct call for argument-validation tests; returns the status code."""
    th = None
    n = 0
    if thresholds is not None:
        th = np.asarray(thresholds, dtype=np.float64)
        n = int(th.size)
    o = ctypes.byref(opts) if opts is not None else None
    return getattr(lib(), fn_name)(
        data_ptr, beams, channels, samples, dtype,
        th.ctypes.data_as(ctypes.POINTER(ctypes.c_double)) if th is not None else None, n, policy, o)


def quantise_threshold(k: float) -> int:
    return int(lib().rfim_oracle_quantise_threshold(float(k)))


def stats_u8(x: np.ndarray):
    x = np.ascontiguousarray(x, dtype=np.uint8)
    s, q = ctypes.c_uint64(), ctypes.c_uint64()
    lib().rfim_oracle_stats_u8(x.ctypes.data, x.size, ctypes.byref(s), ctypes.byref(q))
    return int(s.value), int(q.value)


def stats_f32(x: np.ndarray):
    x = np.ascontiguousarray(x, dtype=np.float32)
    m, sg = ctypes.c_double(), ctypes.c_double()
    lib().rfim_oracle_stats_f32(x.ctypes.data, x.size, ctypes.byref(m), ctypes.byref(sg))
    return float(m.value), float(sg.value)


Opts = _Opts
