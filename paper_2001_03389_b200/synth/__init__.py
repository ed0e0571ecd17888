"""Seeded synthetic dynamic spectra with the shapes and structure of the paper's workloads.

INPUT GENERATOR ONLY -- none of the sigma-cut arithmetic lives in this module; it is the single
piece of code that feeds both the CUDA path (tests, bench) and the CPU oracle (tests).  The paper
measured on an Apertif observation of PSR B0531+21 and on simulated
ARTS-parameter data; neither is available, so these inputs stand in for both:
1536 channels of 0.1953125 MHz over 1220-1520 MHz, 81.92 us sampling (12,500 samples per 1.024 s
batch), 12 beams, Gaussian noise + narrow-band RFI + broadband impulses + one
faint dispersed pulse at DM = 500 pc/cm^3 placed with Eq. 2.  DESIGN.md, "Input
recipe", states every parameter.

Master seed 200103389; config n uses seed + n.  Everything is counter-based, so any beam range is
reproducible on its own (host or device) and uint8 host/device twins are bit-identical.
"""
from __future__ import annotations

import ctypes
import math
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_HOST_LIB = os.path.join(_HERE, "librfim_synth_host.so")
_CUDA_LIB = os.path.join(_HERE, "librfim_synth_cuda.so")

MASTER_SEED = 200103389
_M64 = (1 << 64) - 1
_GOLD = 0x9E3779B97F4A7C15

# BASELINE.json configs[0..4] -> ids 1..5
CONFIGS = {
    1: dict(name="tiny_td", beams=1, channels=64, samples=1024, dtype="u8", mu=100.0, sigma=10.0,
            kind="tiny", op="time", thresholds=[3.0], policy="mean"),
    2: dict(name="arts_td", beams=12, channels=1536, samples=12500, dtype="u8", mu=100.0, sigma=12.0,
            kind="arts", op="time", thresholds=[5.0, 4.0, 3.0], policy="mean"),
    3: dict(name="arts_fd", beams=12, channels=1536, samples=12500, dtype="u8", mu=100.0, sigma=12.0,
            kind="arts", op="freq", thresholds=[4.0, 3.0], policy="mean"),
    4: dict(name="arts_480_chain", beams=480, channels=1536, samples=12500, dtype="u8", mu=100.0, sigma=12.0,
            kind="arts", op="chain", thresholds=[5.0, 4.0, 3.0], freq_thresholds=[4.0, 3.0], policy="mean"),
    5: dict(name="arts_f32_windowed", beams=12, channels=1536, samples=12500, dtype="f32", mu=0.0, sigma=1.0,
            kind="arts", op="time", thresholds=[4.0, 3.0], policy="median", windows=[256, 1024, 12500],
            f32_scale=12.0),
}


def config(n: int, **override) -> dict:
    cfg = dict(CONFIGS[n])
    cfg["id"] = n
    # configs 2, 3 and 4 share one generator and seed rule: seed + 2
    cfg["seed"] = MASTER_SEED + (2 if n in (2, 3, 4) else n)
    cfg.update(override)
    return cfg


# ------------------------------------------------------------------ small seeded RNG (descriptors)
def _mix64(z: int) -> int:
    z &= _M64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _M64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _M64
    z ^= z >> 31
    return z


class _Stream:
    """splitmix64 sequence keyed by (seed, ids...) -- used only for the few thousand draws that
    place the RFI; the per-sample noise is drawn inside the C / CUDA twins."""

    def __init__(self, seed: int, *ids: int):
        s = _mix64(seed)
        for i in ids:
            s = _mix64(s ^ ((i + 1) * 0xD1342543DE82EF95 & _M64))
        self.state = s

    def u64(self) -> int:
        self.state = (self.state + _GOLD) & _M64
        return _mix64(self.state)

    def randint(self, lo: int, hi: int) -> int:
        return lo + self.u64() % (hi - lo + 1)


# ------------------------------------------------------------------------------- descriptor
def noise_cdf(mu: float, sigma: float) -> np.ndarray:
    """[255] u32 table for the rounded-and-clipped Gaussian: P(X <= v) = Phi((v + 0.5 - mu)/sigma)."""
    t = np.empty(255, dtype=np.uint32)
    for v in range(255):
        p = 0.5 * (1.0 + math.erf((v + 0.5 - mu) / (sigma * math.sqrt(2.0))))
        t[v] = min((1 << 32) - 1, int(math.floor(p * 4294967296.0)))
    return t


def pulse_starts(channels: int, dm: float = 500.0, t0: int = 1000, f_lo: float = 1220.0,
                 bw: float = 300.0, tsamp: float = 81.92e-6) -> np.ndarray:
    """Arrival sample of the dispersed pulse per channel, Eq. 2:
    dt = 4.15e3 * DM * (nu^-2 - nu_top^-2) seconds, channel 0 = lowest frequency."""
    c = np.arange(channels, dtype=np.float64)
    nu = f_lo + (c + 0.5) * bw / channels
    dt = 4.15e3 * dm * (nu ** -2 - (f_lo + bw) ** -2)
    return (t0 + np.rint(dt / tsamp)).astype(np.int32)


class Descriptor:
    """Host-side arrays describing the structure of beams [beam0, beam0 + beams)."""

    def __init__(self, cfg: dict, beam0: int = 0, beams: int | None = None):
        self.cfg = cfg
        self.beam0 = beam0
        self.beams = cfg["beams"] - beam0 if beams is None else beams
        B, C, S = self.beams, cfg["channels"], cfg["samples"]
        self.cdf = noise_cdf(cfg["mu"], cfg["sigma"]) if cfg["dtype"] == "u8" else np.zeros(255, np.uint32)
        self.row_offset = np.zeros((B, C), dtype=np.uint8)
        self.imp_amp = np.zeros((B, S), dtype=np.uint8)
        self.pulse_start = np.zeros(C, dtype=np.int32)
        self.pulse_width = 0
        self.pulse_amp = 0
        ptr = [0]
        bstart, blen, bamp = [], [], []
        per_row = [[] for _ in range(B * C)]
        for b in range(B):
            rng = _Stream(cfg["seed"], 7, beam0 + b)
            if cfg["kind"] == "tiny":
                for ch in (7, 40):
                    if ch < C:
                        self.row_offset[b, ch] = 60
                picked = []
                while len(picked) < min(3, S):
                    s = rng.randint(0, S - 1)
                    if s not in picked:
                        picked.append(s)
                for s in picked:
                    self.imp_amp[b, s] = 80
            elif cfg["kind"] == "arts":
                n_rfi = max(1, int(round(0.05 * C))) if C >= 20 else 0
                chans = list(range(C))
                for i in range(n_rfi):                      # partial Fisher-Yates
                    j = rng.randint(i, C - 1)
                    chans[i], chans[j] = chans[j], chans[i]
                for ch in chans[:n_rfi]:
                    if rng.randint(0, 1) == 0:              # persistent
                        self.row_offset[b, ch] = rng.randint(40, 100)
                    else:                                    # intermittent bursts
                        for _ in range(rng.randint(1, 6)):
                            st = rng.randint(0, S - 1)
                            ln = min(rng.randint(10, 500), S - st)
                            per_row[b * C + ch].append((st, ln, rng.randint(40, 100)))
                for _ in range(20):                          # broadband impulses
                    st = rng.randint(0, S - 1)
                    wd = rng.randint(1, 5)
                    am = rng.randint(40, 100)
                    seg = self.imp_amp[b, st:st + wd].astype(np.int32) + am
                    self.imp_amp[b, st:st + wd] = np.minimum(seg, 255).astype(np.uint8)
            elif cfg["kind"] == "noise":
                pass
            else:
                raise ValueError(cfg["kind"])
        if cfg["kind"] == "arts":
            self.pulse_start = pulse_starts(C)
            self.pulse_width = 4
            self.pulse_amp = 15
        for lst in per_row:
            for (st, ln, am) in lst:
                bstart.append(st)
                blen.append(ln)
                bamp.append(am)
            ptr.append(len(bstart))
        self.burst_ptr = np.asarray(ptr, dtype=np.int32)
        self.burst_start = np.asarray(bstart + [0], dtype=np.int32)
        self.burst_len = np.asarray(blen + [0], dtype=np.int32)
        self.burst_amp = np.asarray(bamp + [0], dtype=np.uint8)

    ARRAYS = ("cdf", "row_offset", "imp_amp", "pulse_start", "burst_ptr", "burst_start", "burst_len", "burst_amp")


class _CDesc(ctypes.Structure):
    _fields_ = [
        ("seed", ctypes.c_uint64), ("beam0", ctypes.c_int32), ("beams", ctypes.c_int32),
        ("channels", ctypes.c_int32), ("samples", ctypes.c_int32), ("sample_stride", ctypes.c_int64),
        ("cdf", ctypes.c_void_p), ("row_offset", ctypes.c_void_p), ("imp_amp", ctypes.c_void_p),
        ("pulse_start", ctypes.c_void_p), ("pulse_width", ctypes.c_int32), ("pulse_amp", ctypes.c_int32),
        ("burst_ptr", ctypes.c_void_p), ("burst_start", ctypes.c_void_p), ("burst_len", ctypes.c_void_p),
        ("burst_amp", ctypes.c_void_p), ("f32_scale", ctypes.c_double),
    ]


def _cdesc(d: Descriptor, ptrs: dict, stride: int) -> _CDesc:
    cfg = d.cfg
    return _CDesc(cfg["seed"], d.beam0, d.beams, cfg["channels"], cfg["samples"], stride,
                  ptrs["cdf"], ptrs["row_offset"], ptrs["imp_amp"], ptrs["pulse_start"],
                  d.pulse_width, d.pulse_amp, ptrs["burst_ptr"], ptrs["burst_start"], ptrs["burst_len"],
                  ptrs["burst_amp"], float(cfg.get("f32_scale", 1.0)))


# ------------------------------------------------------------------------------------ build
def build_host(force: bool = False) -> str:
    src = os.path.join(_HERE, "synth_host.c")
    hdr = os.path.join(_HERE, "synth_core.h")
    if force or not os.path.exists(_HOST_LIB) or os.path.getmtime(_HOST_LIB) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-Wall", "-shared", "-fPIC", "-o", _HOST_LIB, src, "-lm"])
    return _HOST_LIB


def build_cuda(force: bool = False) -> str:
    src = os.path.join(_HERE, "synth_cuda.cu")
    hdr = os.path.join(_HERE, "synth_core.h")
    if force or not os.path.exists(_CUDA_LIB) or os.path.getmtime(_CUDA_LIB) < max(os.path.getmtime(src), os.path.getmtime(hdr)):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-shared",
                               "-Xcompiler", "-fPIC", "-o", _CUDA_LIB, src])
    return _CUDA_LIB


_host = None
_cuda = None


def _host_lib():
    global _host
    if _host is None:
        _host = ctypes.CDLL(build_host())
        for n in ("rfim_synth_fill_u8_host", "rfim_synth_fill_f32_host"):
            getattr(_host, n).argtypes = [ctypes.POINTER(_CDesc), ctypes.c_void_p]
            getattr(_host, n).restype = None
    return _host


def _cuda_lib():
    global _cuda
    if _cuda is None:
        if not os.path.exists(_CUDA_LIB):
            build_cuda()
        _cuda = ctypes.CDLL(_CUDA_LIB)
        _cuda.rfim_synth_fill_u8_cuda.argtypes = [ctypes.POINTER(_CDesc), ctypes.c_void_p, ctypes.c_void_p]
        _cuda.rfim_synth_fill_u8_cuda.restype = ctypes.c_int
    return _cuda


# ------------------------------------------------------------------------------------- fill
def fill_host(cfg: dict, beam0: int = 0, beams: int | None = None, sample_stride: int = 0) -> np.ndarray:
    """Generate beams [beam0, beam0+beams) of a config on the host.  Returns [beams][channels][stride]
    (uint8 or float32); columns >= samples (padding) are zero."""
    d = Descriptor(cfg, beam0, beams)
    C, S = cfg["channels"], cfg["samples"]
    stride = sample_stride or S
    dtype = np.uint8 if cfg["dtype"] == "u8" else np.float32
    out = np.zeros((d.beams, C, stride), dtype=dtype)
    ptrs = {k: getattr(d, k).ctypes.data for k in Descriptor.ARRAYS}
    cd = _cdesc(d, ptrs, stride)
    fn = _host_lib().rfim_synth_fill_u8_host if cfg["dtype"] == "u8" else _host_lib().rfim_synth_fill_f32_host
    fn(ctypes.byref(cd), out.ctypes.data)
    return out


def fill_device(cfg: dict, out, beam0: int = 0, beams: int | None = None, sample_stride: int = 0):
    """uint8 only: generate beams [beam0, beam0+beams) straight into the CUDA tensor `out`
    (torch.uint8, at least beams*channels*stride elements).  Bit-identical to fill_host."""
    import torch
    if cfg["dtype"] != "u8":
        raise ValueError("device generator is uint8-only; use fill_host for float32")
    d = Descriptor(cfg, beam0, beams)
    stride = sample_stride or cfg["samples"]
    assert out.is_cuda and out.dtype == torch.uint8 and out.numel() >= d.beams * cfg["channels"] * stride
    dev = {k: torch.from_numpy(getattr(d, k)).to(out.device) for k in Descriptor.ARRAYS}
    ptrs = {k: v.data_ptr() for k, v in dev.items()}
    cd = _cdesc(d, ptrs, stride)
    stream = torch.cuda.current_stream(out.device).cuda_stream
    err = _cuda_lib().rfim_synth_fill_u8_cuda(ctypes.byref(cd), out.data_ptr(), ctypes.c_void_p(stream))
    if err != 0:
        raise RuntimeError(f"synth_fill_u8_cuda: CUDA error {err}")
    torch.cuda.current_stream(out.device).synchronize()   # descriptors may be freed after this
    return out
