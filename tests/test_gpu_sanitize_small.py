"""One small call of every tuned kernel, bit-exact (uint8) / within tolerance (float32) against the oracle.

This module is the workload of the compute-sanitizer runs kept under profiles/ (memcheck, racecheck, initcheck,
synccheck: SURVEY.md section 4, tier T3): shapes of config 1 and of narrow slices of configs 2, 3 and 5 -- small
enough for the sanitizer's slowdown, large enough to span several tiles, ring wrap-arounds, a ragged tail and
every barrier / mbarrier / bulk-copy hand-off of the kernels.  It also runs in the normal `-m gpu` suite."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def u8_slice(cfg_no, channels, samples, beams=1):
    cfg = synth.config(cfg_no, beams=beams, channels=channels, samples=samples)
    return synth.fill_host(cfg), cfg


@pytest.mark.parametrize("policy", ["mean", "median"])
def test_td_u8_staged(policy):
    x, cfg = u8_slice(2, 96, 12500)
    pol = oracle.MEDIAN if policy == "median" else oracle.MEAN
    ref, rflags, rcounts = oracle.time_sigma_cut(x, cfg["thresholds"], policy=pol)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.empty_like(xd)
    flags = torch.zeros(x.shape, dtype=torch.uint8, device=DEV)
    counts = torch.zeros(3, dtype=torch.int64, device=DEV)
    rfim.rfim_time_sigma_cut(xd, cfg["thresholds"], policy, out=out, flags=flags, counts=counts,
                             variant=rfim.VARIANT_STAGED)
    torch.cuda.synchronize()
    assert rfim.rfim_last_variant().startswith("td_u8_staged")
    assert np.array_equal(out.cpu().numpy(), ref) and np.array_equal(flags.cpu().numpy(), rflags)
    assert counts.cpu().tolist() == [int(c) for c in rcounts]


def test_config1_smoke_shape():
    cfg = synth.config(1)
    x = synth.fill_host(cfg)
    ref, _, _ = oracle.time_sigma_cut(x, cfg["thresholds"])
    xd = torch.from_numpy(x).to(DEV)
    rfim.rfim_time_sigma_cut(xd, cfg["thresholds"])
    torch.cuda.synchronize()
    assert np.array_equal(xd.cpu().numpy(), ref)


@pytest.mark.parametrize("variant,inplace,bins", [
    (rfim.VARIANT_FD_STRIP, True, 0), (rfim.VARIANT_FD_STRIP, False, 0), (rfim.VARIANT_FD_STRIP_BULK, True, 0),
    (rfim.VARIANT_FD_STREAM, True, 0), (rfim.VARIANT_FD_STREAM, False, 0), (rfim.VARIANT_FD_STREAM, True, 32),
    (rfim.VARIANT_FD_STREAM, False, 32), (rfim.VARIANT_FD_QUAD, True, 0), (rfim.VARIANT_FD_QUAD, False, 0)])
def test_fd_u8_tuned(variant, inplace, bins):
    x, cfg = u8_slice(3, 1536, 1100)                     # 9 tiles of 128 samples, the last one ragged (76)
    ks = [2.75, 2.75] if bins else cfg["thresholds"]
    ref, rflags, rcounts = oracle.freq_sigma_cut(x, ks, bin_size=bins)
    xd = torch.from_numpy(x).to(DEV)
    out = None if inplace else torch.empty_like(xd)
    flags = torch.zeros(x.shape, dtype=torch.uint8, device=DEV)
    counts = torch.zeros(2, dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(xd, ks, out=out, bin_size=bins, flags=flags, counts=counts, variant=variant)
    torch.cuda.synchronize()
    assert np.array_equal(res.cpu().numpy(), ref), rfim.rfim_last_variant()
    assert np.array_equal(flags.cpu().numpy(), rflags)
    assert counts.cpu().tolist() == [int(c) for c in rcounts]


@pytest.mark.parametrize("policy", ["mean", "median"])
@pytest.mark.parametrize("window", [256, 1024, 0])
def test_td_f32(policy, window):
    cfg = synth.config(5, beams=1, channels=24)
    x = synth.fill_host(cfg)
    from test_gpu_td_f32 import check
    check(x, cfg["thresholds"], policy=policy, window=window)


def test_chain_and_host_path():
    x, cfg = u8_slice(4, 512, 2048, beams=2)
    tks, fks = cfg["thresholds"], cfg["freq_thresholds"]
    y, _, _ = oracle.time_sigma_cut(x, tks)
    ref, _, _ = oracle.freq_sigma_cut(y, fks)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.empty_like(xd)
    rfim.rfim_time_freq_sigma_cut(xd, tks, fks, out=out)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), ref)
    h_in = torch.from_numpy(x).pin_memory()
    h_out = torch.empty_like(h_in).pin_memory()
    rfim.rfim_sigma_cut_host(h_in, tks, fks, out=h_out)
    assert np.array_equal(h_out.numpy(), ref)
