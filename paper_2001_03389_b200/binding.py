"""Thin ctypes binding of librfim (include/rfim.h): argument marshalling only.

Every step of the path runs in the CUDA kernels behind the C ABI; PyTorch supplies device memory
and streams.  There is no CPU fallback: if the library is missing or a call fails, this raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional, Sequence

import torch

from . import build as _build

U8, F32 = 0, 1
MEAN, MEDIAN = 0, 1
OK, ERR_INVALID, ERR_UNSUPPORTED, ERR_CUDA, ERR_TOO_LARGE = 0, -1, -2, -3, -4
NOALLOC_MAX_TILES = 1 << 24                  # include/rfim.h: RFIM_NOALLOC_MAX_TILES
VARIANT_AUTO, VARIANT_GENERIC, VARIANT_STAGED = 0, 1, 2
VARIANT_STAGED_1W, VARIANT_STAGED_2W = 3, 4
VARIANT_FD_STRIP_BULK, VARIANT_FD_STRIP_CLUSTER, VARIANT_FD_STRIP, VARIANT_FD_STREAM = 13, 14, 15, 16
VARIANT_FD_QUAD = 17
VARIANT_FD_QBIN = 18
OP_TIME, OP_FREQ, OP_TIME_FREQ, OP_HOST = 0, 1, 2, 3

EXPORTS = ("rfim_time_sigma_cut", "rfim_freq_sigma_cut", "rfim_freq_sigma_cut_noalloc", "rfim_time_freq_sigma_cut",
           "rfim_sigma_cut_host",
           "rfim_workspace_bytes",
           "rfim_launch_count", "rfim_last_variant", "rfim_status_string", "rfim_last_cuda_error",
           "rfim_version")


class RfimOpts(ctypes.Structure):
    _fields_ = [
        ("sample_stride", ctypes.c_int64),
        ("window", ctypes.c_int32),
        ("bin_size", ctypes.c_int32),
        ("out", ctypes.c_void_p),
        ("flags", ctypes.c_void_p),
        ("counts", ctypes.c_void_p),
        ("stream", ctypes.c_void_p),
        ("workspace", ctypes.c_void_p),
        ("variant", ctypes.c_int32),
        ("reserved", ctypes.c_int32),
    ]


class RfimError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"librfim status {status}: {message}")
        self.status = status


_lib = None


def lib() -> ctypes.CDLL:
    """Load librfim.so from the package directory (building it with nvcc if the sources are newer)."""
    global _lib
    if _lib is None:
        path = _build.LIB
        try:
            path = _build.build_librfim()
        except Exception as exc:  # no nvcc here: the prebuilt library must exist
            if not os.path.exists(path):
                raise RuntimeError(
                    f"librfim.so is missing and could not be built ({exc}); there is no CPU fallback") from exc
        _lib = ctypes.CDLL(path)
        dp = ctypes.POINTER(ctypes.c_double)
        sig = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, dp, ctypes.c_int,
               ctypes.c_int, ctypes.POINTER(RfimOpts)]
        for name in ("rfim_time_sigma_cut", "rfim_freq_sigma_cut", "rfim_freq_sigma_cut_noalloc"):
            getattr(_lib, name).argtypes = sig
            getattr(_lib, name).restype = ctypes.c_int
        _lib.rfim_time_freq_sigma_cut.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                                  ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int, ctypes.c_int,
                                                  ctypes.POINTER(RfimOpts)]
        _lib.rfim_time_freq_sigma_cut.restype = ctypes.c_int
        _lib.rfim_sigma_cut_host.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_int, ctypes.c_int, dp, ctypes.c_int, dp, ctypes.c_int,
                                             ctypes.c_int, ctypes.POINTER(RfimOpts)]
        _lib.rfim_sigma_cut_host.restype = ctypes.c_int
        _lib.rfim_workspace_bytes.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                              ctypes.c_int, ctypes.c_int, ctypes.POINTER(RfimOpts)]
        _lib.rfim_workspace_bytes.restype = ctypes.c_size_t
        _lib.rfim_launch_count.restype = ctypes.c_uint64
        _lib.rfim_last_variant.restype = ctypes.c_char_p
        _lib.rfim_status_string.argtypes = [ctypes.c_int]
        _lib.rfim_status_string.restype = ctypes.c_char_p
        _lib.rfim_last_cuda_error.restype = ctypes.c_char_p
        _lib.rfim_version.restype = ctypes.c_int
    return _lib


def _check(status: int) -> None:
    if status != OK:
        msg = lib().rfim_status_string(status).decode()
        if status == ERR_CUDA:
            msg += ": " + lib().rfim_last_cuda_error().decode()
        raise RfimError(status, msg)


def _doubles(values: Sequence[float]):
    arr = (ctypes.c_double * max(1, len(values)))(*[float(v) for v in values])
    return arr, len(values)


def _dtype_code(t: torch.Tensor) -> int:
    if t.dtype == torch.uint8:
        return U8
    if t.dtype == torch.float32:
        return F32
    raise TypeError("librfim: dtype must be torch.uint8 or torch.float32")


def _policy_code(policy) -> int:
    if policy in (MEAN, "mean"):
        return MEAN
    if policy in (MEDIAN, "median"):
        return MEDIAN
    raise ValueError(f"librfim: unknown replacement policy {policy!r}")


def _layout(t: torch.Tensor):
    """[beams][channels][samples] with unit sample stride and rows a constant pitch apart."""
    if t.dim() != 3:
        raise ValueError("librfim: data must be [beams][channels][samples]")
    b, c, s = t.shape
    sb, sc, ss = t.stride()
    if (s > 1 and ss != 1) or (c > 1 and sb != sc * c and b > 1):
        raise ValueError("librfim: rows must be a constant pitch apart with contiguous samples")
    pitch = sc if c > 1 else (sb if b > 1 else s)
    return b, c, s, pitch


def _call(fn_name: str, data: torch.Tensor, thresholds, policy, out, window, bin_size, flags, counts, stream,
          variant, workspace):
    if not data.is_cuda:
        raise ValueError("librfim: data must be a CUDA tensor (device pointer ABI; no CPU fallback)")
    b, c, s, pitch = _layout(data)
    if out is not None:
        if out.shape != data.shape or out.dtype != data.dtype or _layout(out)[3] != pitch or not out.is_cuda:
            raise ValueError("librfim: out must match data in shape, dtype and pitch")
    if flags is not None and (flags.dtype != torch.uint8 or not flags.is_contiguous() or flags.numel() != b * c * s):
        raise ValueError("librfim: flags must be a dense uint8 [B][C][S] tensor")
    th, n = _doubles(thresholds)
    if counts is not None and (counts.dtype != torch.int64 or counts.numel() < n):
        raise ValueError("librfim: counts must be int64 with n_thresholds entries")
    if stream is None:
        stream = torch.cuda.current_stream(data.device)
    o = RfimOpts(pitch if pitch != s else 0, int(window), int(bin_size),
                 out.data_ptr() if out is not None else None,
                 flags.data_ptr() if flags is not None else None,
                 counts.data_ptr() if counts is not None else None,
                 stream.cuda_stream, workspace.data_ptr() if workspace is not None else None, int(variant), 0)
    with torch.cuda.device(data.device):
        st = getattr(lib(), fn_name)(data.data_ptr(), b, c, s, _dtype_code(data), th, n, _policy_code(policy),
                                     ctypes.byref(o))
    _check(st)
    return out if out is not None else data


def rfim_time_sigma_cut(data: torch.Tensor, thresholds: Sequence[float], policy=MEAN, *,
                        out: Optional[torch.Tensor] = None, window: int = 0,
                        flags: Optional[torch.Tensor] = None, counts: Optional[torch.Tensor] = None,
                        stream=None, variant: int = VARIANT_AUTO, workspace=None) -> torch.Tensor:
    """TDSC.  Asynchronous on `stream` (default: torch's current stream); in place unless `out`."""
    return _call("rfim_time_sigma_cut", data, thresholds, policy, out, window, 0, flags, counts, stream, variant,
                 workspace)


def rfim_freq_sigma_cut(data: torch.Tensor, thresholds: Sequence[float], policy=MEAN, *,
                        out: Optional[torch.Tensor] = None, bin_size: int = 0,
                        flags: Optional[torch.Tensor] = None, counts: Optional[torch.Tensor] = None,
                        stream=None, variant: int = VARIANT_AUTO, workspace=None) -> torch.Tensor:
    """FDSC.  Asynchronous on `stream`; in place unless `out`."""
    return _call("rfim_freq_sigma_cut", data, thresholds, policy, out, 0, bin_size, flags, counts, stream, variant,
                 workspace)


def rfim_freq_sigma_cut_noalloc(data: torch.Tensor, thresholds: Sequence[float], *,
                                out: Optional[torch.Tensor] = None,
                                flags: Optional[torch.Tensor] = None, counts: Optional[torch.Tensor] = None,
                                stream=None) -> torch.Tensor:
    """FDSC (uint8, one bin, mean) through the entry point that allocates no device memory: its scratch is a static
    device array inside the library (include/rfim.h).  Calls that overlap on the GPU race on that array."""
    return _call("rfim_freq_sigma_cut_noalloc", data, thresholds, MEAN, out, 0, 0, flags, counts, stream, VARIANT_AUTO,
                 None)


def rfim_time_freq_sigma_cut(data: torch.Tensor, time_thresholds: Sequence[float], freq_thresholds: Sequence[float],
                             policy=MEAN, *, out: Optional[torch.Tensor] = None, window: int = 0, bin_size: int = 0,
                             flags: Optional[torch.Tensor] = None, counts: Optional[torch.Tensor] = None,
                             stream=None, variant: int = VARIANT_AUTO) -> torch.Tensor:
    """TDSC then FDSC on its result.  Asynchronous on `stream`; TDSC writes `out` (or works in
    place), FDSC cleans that result in place.  counts: int64 [len(time) + len(freq)]."""
    if not data.is_cuda:
        raise ValueError("librfim: data must be a CUDA tensor (device pointer ABI; no CPU fallback)")
    b, c, s, pitch = _layout(data)
    if out is not None:
        if out.shape != data.shape or out.dtype != data.dtype or _layout(out)[3] != pitch or not out.is_cuda:
            raise ValueError("librfim: out must match data in shape, dtype and pitch")
    if flags is not None and (flags.dtype != torch.uint8 or not flags.is_contiguous() or flags.numel() != b * c * s):
        raise ValueError("librfim: flags must be a dense uint8 [B][C][S] tensor")
    tt, nt = _doubles(time_thresholds)
    ft, nf = _doubles(freq_thresholds)
    if counts is not None and (counts.dtype != torch.int64 or counts.numel() < nt + nf):
        raise ValueError("librfim: counts must be int64 with n_time + n_freq entries")
    if stream is None:
        stream = torch.cuda.current_stream(data.device)
    o = RfimOpts(pitch if pitch != s else 0, int(window), int(bin_size),
                 out.data_ptr() if out is not None else None,
                 flags.data_ptr() if flags is not None else None,
                 counts.data_ptr() if counts is not None else None,
                 stream.cuda_stream, None, int(variant), 0)
    with torch.cuda.device(data.device):
        st = lib().rfim_time_freq_sigma_cut(data.data_ptr(), b, c, s, _dtype_code(data), tt, nt, ft, nf,
                                            _policy_code(policy), ctypes.byref(o))
    _check(st)
    return out if out is not None else data


def rfim_workspace_bytes(op: int, beams: int, channels: int, samples: int, dtype=U8, n_thresholds: int = 0,
                         policy=MEAN, sample_stride: int = 0) -> int:
    o = RfimOpts(int(sample_stride), 0, 0, None, None, None, None, None, 0, 0)
    return int(lib().rfim_workspace_bytes(int(op), beams, channels, samples, int(dtype), n_thresholds,
                                          _policy_code(policy), ctypes.byref(o)))


def rfim_sigma_cut_host(data: torch.Tensor, time_thresholds: Sequence[float], freq_thresholds: Sequence[float],
                        policy=MEAN, *, out: Optional[torch.Tensor] = None, window: int = 0,
                        bin_size: int = 0, workspace: Optional[torch.Tensor] = None) -> torch.Tensor:
    """End-to-end path on HOST tensors (pinned memory recommended): H2D, TDSC, FDSC, D2H, streamed by beam.
    `workspace`: device tensor of >= rfim_workspace_bytes(OP_HOST, ...) bytes for the staging buffers."""
    if data.is_cuda:
        raise ValueError("rfim_sigma_cut_host takes host tensors")
    b, c, s, pitch = _layout(data)
    if out is not None and (out.shape != data.shape or out.dtype != data.dtype or _layout(out)[3] != pitch):
        raise ValueError("librfim: out must match data in shape, dtype and pitch")
    tt, nt = _doubles(time_thresholds)
    ft, nf = _doubles(freq_thresholds)
    if workspace is not None:
        need = rfim_workspace_bytes(OP_HOST, b, c, s, _dtype_code(data), sample_stride=pitch if pitch != s else 0)
        if not workspace.is_cuda or workspace.numel() * workspace.element_size() < need:
            raise ValueError(f"librfim: workspace must be a CUDA tensor of at least {need} bytes")
    o = RfimOpts(pitch if pitch != s else 0, int(window), int(bin_size), None, None, None, None,
                 workspace.data_ptr() if workspace is not None else None, 0, 0)
    st = lib().rfim_sigma_cut_host(data.data_ptr(), out.data_ptr() if out is not None else None, b, c, s,
                                   _dtype_code(data), tt, nt, ft, nf, _policy_code(policy), ctypes.byref(o))
    _check(st)
    return out if out is not None else data


def rfim_launch_count() -> int:
    return int(lib().rfim_launch_count())


def rfim_last_variant() -> str:
    return lib().rfim_last_variant().decode()


def rfim_version() -> int:
    return int(lib().rfim_version())
