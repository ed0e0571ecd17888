"""GPU test of rfim_freq_sigma_cut_noalloc (include/rfim.h): the FDSC entry point that allocates no device memory --
its scratch, the tile dispenser of the streaming kernel, is a static device array inside librfim.so.

The file name makes pytest collect it last (the suite runs with `pytest -x`).  The new entry point is compared with
the existing path (rfim_freq_sigma_cut) bit for bit -- the tolerance of every uint8 test here -- on two calls in a
row: the array keeps the first call's contents, the second call must not see them."""
import ctypes

import numpy as np
import pytest
import torch

import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import binding, synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def both_paths(x, ks, inplace):
    """(existing path, new entry point) on copies of x: cleaned array, flags, counts"""
    res = []
    for fn in (rfim.rfim_freq_sigma_cut, rfim.rfim_freq_sigma_cut_noalloc):
        src = x.clone()
        out = None if inplace else torch.full_like(x, 0xAB)
        flags = torch.full(x.shape, 7, dtype=torch.uint8, device=DEV)
        counts = torch.full((len(ks),), -1, dtype=torch.int64, device=DEV)
        r = fn(src, ks, out=out, flags=flags, counts=counts)
        torch.cuda.synchronize()
        if not inplace:
            assert torch.equal(src, x), "input modified by an out-of-place call"
        res.append((r.clone(), flags, counts, rfim.rfim_last_variant()))
    return res


def test_two_calls_in_a_row_match_the_existing_path():
    cfg = synth.config(3, beams=3)
    a = torch.from_numpy(synth.fill_host(cfg, beam0=2, beams=3)).to(DEV)               # 3 x 1536 x 12500: 294 tiles
    rng = np.random.default_rng(7)
    b_np = np.clip(np.rint(rng.normal(100, 12, (2, 512, 300))), 0, 255).astype(np.uint8)   # ragged last tile
    b_np[0, 100, :] = 250
    b_np[1, :, 17] = 3
    b = torch.from_numpy(b_np).to(DEV)
    calls = [(a, cfg["thresholds"], True), (b, [3.0, 2.5, 2.5], False), (a, [2.75], False)]
    for x, ks, inplace in calls:                       # back to back: the scratch array is reused without a reload
        (r0, f0, c0, n0), (r1, f1, c1, n1) = both_paths(x, ks, inplace)
        assert n1 in ("fd_u8_quad", "fd_u8_quad_copy"), n1
        assert torch.equal(r0, r1), "cleaned array differs from the existing path"
        assert torch.equal(f0, f1), "flags differ from the existing path"
        assert c0.tolist() == c1.tolist() and int(c1[0]) > 0
        assert int((r1 != x).sum()) > 0


def test_no_device_memory_is_taken():
    x = torch.from_numpy(synth.fill_host(synth.config(3, beams=2))).to(DEV)
    out = torch.empty_like(x)
    rfim.rfim_freq_sigma_cut_noalloc(x, [4.0, 3.0], out=out)           # set-up call (symbol address, attributes)
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(2):
        rfim.rfim_freq_sigma_cut_noalloc(x, [4.0, 3.0], out=out)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0, (free0, free1)
    ref = rfim.rfim_freq_sigma_cut(x.clone(), [4.0, 3.0])
    torch.cuda.synchronize()
    assert torch.equal(out, ref)


def test_requests_beyond_the_limits_are_refused():
    x = torch.zeros((1, 512, 128), dtype=torch.uint8, device=DEV)
    lib = binding.lib()
    th = (ctypes.c_double * 1)(3.0)
    # more tiles than the stated maximum: refused before anything is enqueued (the pointer is never used)
    st = lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), binding.NOALLOC_MAX_TILES + 1, 512, 128, 0, th, 1, 0, None)
    assert st == binding.ERR_TOO_LARGE and b"RFIM_NOALLOC_MAX_TILES" in lib.rfim_status_string(st)
    st = lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), binding.NOALLOC_MAX_TILES // 2 + 1, 512, 256, 0, th, 1, 0, None)
    assert st == binding.ERR_TOO_LARGE
    o = binding.RfimOpts()
    o.workspace = x.data_ptr()
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 512, 128, 0, th, 1, 0, ctypes.byref(o)) == binding.ERR_INVALID
    o = binding.RfimOpts()
    o.variant = 15
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 512, 128, 0, th, 1, 0, ctypes.byref(o)) == binding.ERR_INVALID
    o = binding.RfimOpts()
    o.bin_size = 32
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 512, 128, 0, th, 1, 0, ctypes.byref(o)) == binding.ERR_UNSUPPORTED
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 512, 128, 0, th, 1, 1, None) == binding.ERR_UNSUPPORTED   # median
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 512, 128, 1, th, 1, 0, None) == binding.ERR_UNSUPPORTED   # float32
    assert lib.rfim_freq_sigma_cut_noalloc(x.data_ptr(), 1, 640, 128, 0, th, 1, 0, None) == binding.ERR_UNSUPPORTED   # channels
    with pytest.raises(rfim.RfimError) as e:           # rows not 4-byte aligned: not the streaming kernel's request
        rfim.rfim_freq_sigma_cut_noalloc(torch.zeros((1, 512, 130), dtype=torch.uint8, device=DEV), [3.0])
    assert e.value.status == binding.ERR_UNSUPPORTED
    rfim.rfim_freq_sigma_cut_noalloc(x, [3.0])        # and the array is still usable
    torch.cuda.synchronize()
    assert int(x.sum()) == 0
