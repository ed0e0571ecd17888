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
    assert rfim.rfim_version() == 100
    lib = binding.lib()
    assert lib.rfim_status_string(0) == b"ok"
    assert b"invalid" in lib.rfim_status_string(-1)
    assert b"unsupported" in lib.rfim_status_string(-2)
    assert b"CUDA" in lib.rfim_status_string(-3)


def test_opts_struct_layout():
    # must mirror include/rfim.h: int64, 2 x int32, 5 pointers, 2 x int32
    assert ctypes.sizeof(binding.RfimOpts) == 8 + 4 + 4 + 5 * 8 + 4 + 4
    assert binding.RfimOpts.out.offset == 16 and binding.RfimOpts.variant.offset == 56


@pytest.mark.parametrize("fn", ["rfim_time_sigma_cut", "rfim_freq_sigma_cut"])
def test_invalid_arguments_return_minus_one(fn):
    """Validation precedes every CUDA call, so these run without a GPU.  The pointer is never dereferenced."""
    lib = binding.lib()
    f = getattr(lib, fn)
    fake = ctypes.c_void_p(0x1000)
    th = (ctypes.c_double * 17)(*([3.0] * 17))

    def call(data=fake, b=2, c=4, s=8, dtype=0, thr=th, n=1, policy=0, opts=None):
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
    o = binding.RfimOpts(); o.variant = 15
    assert call(opts=ctypes.byref(o)) == -1
    assert call(data=ctypes.c_void_p(0x1001), dtype=1) == -1   # float32 pointer not 4-byte aligned
    if fn == "rfim_freq_sigma_cut":
        o = binding.RfimOpts(); o.bin_size = 3                  # does not divide 4 channels
        assert call(opts=ctypes.byref(o)) == -1
        assert call(c=(1 << 24) + 1) == -1
    else:
        assert call(s=(1 << 24) + 1) == -1


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
