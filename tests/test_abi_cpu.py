"""CPU-only checks of the C-ABI boundary: librfim.so loads, exports every symbol include/rfim.h
declares, and rejects bad arguments before touching the device (no compute calls here)."""
import ctypes
import os
import re

import pytest

import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import binding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions():
    text = open(os.path.join(ROOT, "include", "rfim.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(rfim_[a-z_0-9]+)\s*\(", text)))


def test_header_symbols_are_exported():
    names = declared_functions()
    assert set(binding.EXPORTS) == set(names), (names, binding.EXPORTS)
    lib = binding.lib()
    for n in names:
        assert hasattr(lib, n), n


def test_version_and_strings():
    assert rfim.rfim_version() == 200
    lib = binding.lib()
    assert lib.rfim_status_string(0) == b"ok"
    assert b"invalid" in lib.rfim_status_string(-1)
    assert b"unsupported" in lib.rfim_status_string(-2)
    assert b"CUDA" in lib.rfim_status_string(-3)


def test_opts_struct_layout():
    # must mirror include/rfim.h: int64, 2 x int32, 5 pointers, 2 x int32
    assert ctypes.sizeof(binding.RfimOpts) == 8 + 4 + 4 + 5 * 8 + 4 + 4
    assert binding.RfimOpts.out.offset == 16 and binding.RfimOpts.variant.offset == 56


@pytest.mark.parametrize("fn", ["rfim_time_sigma_cut", "rfim_freq_sigma_cut", "rfim_time_freq_sigma_cut"])
def test_invalid_arguments_return_minus_one(fn):
    """Validation precedes every CUDA call, so these run without a GPU.  The pointer is never dereferenced."""
    lib = binding.lib()
    f = getattr(lib, fn)
    fake = ctypes.c_void_p(0x1000)
    th = (ctypes.c_double * 17)(*([3.0] * 17))

    def call(data=fake, b=2, c=4, s=8, dtype=0, thr=th, n=1, policy=0, opts=None):
        if fn == "rfim_time_freq_sigma_cut":      # the same list for both operations
            return f(data, b, c, s, dtype, thr, n, thr, n, policy, opts)
        return f(data, b, c, s, dtype, thr, n, policy, opts)

    assert call(data=None) == -1
    assert call(b=0) == -1 and call(c=-1) == -1 and call(s=0) == -1
    assert call(dtype=2) == -1 and call(policy=2) == -1
    assert call(n=-1) == -1 and call(n=17) == -1
    assert call(thr=None, n=1) == -1
    for bad in (0.0, -1.0, float("nan"), 256.0, float("inf")):
        t = (ctypes.c_double * 1)(bad)
        assert call(thr=t) == -1, bad
    o = binding.RfimOpts()
    o.sample_stride = 7
    assert call(opts=ctypes.byref(o)) == -1          # stride < samples
    o = binding.RfimOpts(); o.window = -1
    assert call(opts=ctypes.byref(o)) == -1
    o = binding.RfimOpts(); o.bin_size = -1
    assert call(opts=ctypes.byref(o)) == -1
    o = binding.RfimOpts(); o.reserved = 1
    assert call(opts=ctypes.byref(o)) == -1
    for v in (19, -1, 7):                                       # 5..12 were the removed cluster variants
        o = binding.RfimOpts(); o.variant = v
        assert call(opts=ctypes.byref(o)) == -1, v
    assert call(data=ctypes.c_void_p(0x1001), dtype=1) == -1   # float32 pointer not 4-byte aligned
    # out overlapping data without being data: 2 x 4 x 8 bytes = 64, out 16 bytes in
    o = binding.RfimOpts(); o.out = 0x1010
    assert call(opts=ctypes.byref(o)) == -1
    o = binding.RfimOpts(); o.out = 0x1000 - 63
    assert call(opts=ctypes.byref(o)) == -1
    if fn != "rfim_time_sigma_cut":
        o = binding.RfimOpts(); o.bin_size = 3                  # does not divide 4 channels
        assert call(opts=ctypes.byref(o)) == -1
        assert call(c=(1 << 24) + 1) == -1
    if fn != "rfim_freq_sigma_cut":
        assert call(s=(1 << 24) + 1) == -1
    # a variant of the other operation is a valid value that this operation cannot run: UNSUPPORTED, decided
    # before anything is enqueued
    if fn == "rfim_time_sigma_cut":
        for v in (13, 14, 15, 16, 17, 18):
            o = binding.RfimOpts(); o.variant = v
            assert call(opts=ctypes.byref(o)) == -2, v
    elif fn == "rfim_freq_sigma_cut":
        for v in (3, 4):
            o = binding.RfimOpts(); o.variant = v
            assert call(opts=ctypes.byref(o)) == -2, v
    else:
        for v in (3, 4, 13, 16, 17, 18):
            o = binding.RfimOpts(); o.variant = v
            assert call(opts=ctypes.byref(o)) == -2, v


def test_host_path_validates_only_what_runs():
    """rfim_sigma_cut_host: a bin_size that does not divide the channels is an error only if FDSC runs; opts->out,
    flags, counts, stream must be NULL.  Decided before any CUDA call."""
    lib = binding.lib()
    fake = ctypes.c_void_p(0x1000)
    th = (ctypes.c_double * 2)(3.0, 3.0)
    o = binding.RfimOpts(); o.bin_size = 3
    assert lib.rfim_sigma_cut_host(fake, None, 2, 4, 8, 0, th, 1, th, 1, 0, ctypes.byref(o)) == -1
    o = binding.RfimOpts(); o.window = -1
    assert lib.rfim_sigma_cut_host(fake, None, 2, 4, 8, 0, th, 1, th, 0, 0, ctypes.byref(o)) == -1
    for field in ("out", "flags", "counts", "stream"):
        o = binding.RfimOpts(); setattr(o, field, 0x2000)
        assert lib.rfim_sigma_cut_host(fake, None, 2, 4, 8, 0, th, 1, th, 1, 0, ctypes.byref(o)) == -1, field
    assert lib.rfim_sigma_cut_host(fake, None, 2, 4, 8, 0, th, 17, th, 1, 0, None) == -1
    assert lib.rfim_sigma_cut_host(None, None, 2, 4, 8, 0, th, 1, th, 1, 0, None) == -1


def test_workspace_bytes():
    """TDSC needs no scratch, FDSC 256 bytes (the tile dispenser of the streaming kernel); the host path needs its
    three staging buffers (chunks of whole beams of about 128 MiB, rounded up to 256 bytes), fewer when there are
    fewer chunks."""
    assert rfim.rfim_workspace_bytes(rfim.OP_TIME, 480, 1536, 12500) == 0
    assert rfim.rfim_workspace_bytes(rfim.OP_FREQ, 480, 1536, 12500) == 256
    assert rfim.rfim_workspace_bytes(rfim.OP_TIME_FREQ, 480, 1536, 12500) == 256
    beam = 1536 * 12500
    per_chunk = (128 << 20) // beam
    assert per_chunk == 6
    slot = (per_chunk * beam + 255) // 256 * 256
    assert rfim.rfim_workspace_bytes(rfim.OP_HOST, 480, 1536, 12500) == 3 * slot
    assert rfim.rfim_workspace_bytes(rfim.OP_HOST, 7, 1536, 12500) == 2 * slot
    assert rfim.rfim_workspace_bytes(rfim.OP_HOST, 2, 1536, 12500) == (2 * beam + 255) // 256 * 256
    assert rfim.rfim_workspace_bytes(rfim.OP_HOST, 1, 64, 1024, dtype=1) == 64 * 1024 * 4


def test_binding_rejects_host_tensors():
    import torch
    x = torch.zeros((1, 2, 8), dtype=torch.uint8)
    with pytest.raises(ValueError):
        rfim.rfim_time_sigma_cut(x, [3.0])
    with pytest.raises(TypeError):
        binding._dtype_code(torch.zeros(1, dtype=torch.int32))


def test_header_is_plain_c():
    """include/rfim.h is the boundary: it must compile as C99 on its own (no C++ or CUDA types in the signatures)."""
    import os
    import subprocess
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    subprocess.check_call(["gcc", "-std=c99", "-Wall", "-Werror", "-fsyntax-only", "-x", "c",
                           os.path.join(root, "include", "rfim.h")])
