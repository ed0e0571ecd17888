"""GPU parity: rfim_freq_sigma_cut with the per-bin mean correction (bin_size; SURVEY.md 8f
NEXT-1) vs the CPU oracle, bit-exact (cleaned array, flags, counts)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def check(x_np, ks, bin_size, inplace=False, pitch=None):
    B, C, S = x_np.shape
    ref, rflags, rcounts = oracle.freq_sigma_cut(x_np, ks, bin_size=bin_size)
    if pitch is None:
        x = torch.from_numpy(x_np).to(DEV)
        out = None if inplace else torch.full_like(x, 0xAB)
    else:
        buf = torch.full((B, C, pitch), 0x5A, dtype=torch.uint8, device=DEV)
        buf[:, :, :S] = torch.from_numpy(x_np).to(DEV)
        x = buf[:, :, :S]
        out = None if inplace else torch.full((B, C, pitch), 0xAB, dtype=torch.uint8, device=DEV)[:, :, :S]
    flags = torch.full((B, C, S), 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((len(ks),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(x, ks, out=out, bin_size=bin_size, flags=flags, counts=counts)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    assert np.array_equal(res.cpu().numpy(), ref), f"{name}: cleaned array differs"
    assert np.array_equal(flags.cpu().numpy(), rflags), f"{name}: flags differ"
    assert counts.cpu().tolist() == [int(c) for c in rcounts]
    if pitch is not None:
        assert torch.all(buf[:, :, S:] == 0x5A)
    return name, rcounts


def banded(shape, seed):
    """Gaussian noise on a bandpass that differs per 32-channel block (what the bin correction is for), plus
    narrow-band RFI, a broadband spike and a dropout."""
    rng = np.random.default_rng(seed)
    B, C, S = shape
    band = 60 + 80 * rng.random((B, (C + 31) // 32, 1)).repeat(32, axis=1)[:, :C]
    x = np.clip(np.rint(rng.normal(band, 8, shape)), 0, 255)
    x[0, C // 3, :] += 70
    x[:, :, S // 2] += 90
    x[B - 1, C - 1, ::5] = 0
    return np.clip(x, 0, 255).astype(np.uint8)


@pytest.mark.parametrize("C,S,nb", [(64, 257, 32), (64, 100, 4), (96, 64, 48), (128, 33, 1), (1536, 40, 32),
                                    (60, 50, 20), (32, 16, 32)])
def test_binned_matches_oracle(C, S, nb):
    x = banded((2, C, S), seed=C * 3 + nb)
    name, counts = check(x, [2.75, 2.75], nb)
    want = ("fd_u8_qbin_copy" if (C, nb) == (1536, 32) else "fd_u8_binned_generic" if nb != C
            else "fd_u8_strip1" if S % 4 == 0 else "fd_u8_generic")
    assert name == want
    check(x, [4.0, 3.0, 3.0], nb, inplace=True)
    check(x, [0.5], nb)


def test_binned_config3_shape_fig5_parameters():
    """BASELINE.json configs[2] generator (one beam, 1536 channels, 500 samples) with the paper's Fig. 5 FDSC
    parameters: bins of 32 channels, 2.75 sigma."""
    cfg = synth.config(3, beams=1, samples=500)
    x = synth.fill_host(cfg)
    name, counts = check(x, [2.75], 32)
    assert name == "fd_u8_qbin_copy" and int(counts[0]) > 0
    check(x, [2.75, 2.75, 2.75], 32, pitch=512)


def check_policy(x_np, ks, bin_size, policy):
    pol = oracle.MEDIAN if policy == "median" else oracle.MEAN
    ref, rflags, rcounts = oracle.freq_sigma_cut(x_np, ks, policy=pol, bin_size=bin_size)
    x = torch.from_numpy(x_np).to(DEV)
    flags = torch.zeros(x_np.shape, dtype=torch.uint8, device=DEV)
    counts = torch.zeros(len(ks), dtype=torch.int64, device=DEV)
    out = torch.empty_like(x)
    # float32: the definition kernel (variant 1), whose fp64 operations follow the oracle's order exactly; the tuned
    # float32 kernel has its own test module (test_gpu_fd_f32_tile.py)
    rfim.rfim_freq_sigma_cut(x, ks, policy, out=out, bin_size=bin_size, flags=flags, counts=counts,
                             variant=rfim.VARIANT_GENERIC if x_np.dtype == np.float32 else rfim.VARIANT_AUTO)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    if x_np.dtype == np.uint8:
        assert np.array_equal(got, ref)
    else:
        # same fp64 operations in the same order as the definition: identical flags, values within 1e-5 relative
        assert np.allclose(got, ref, rtol=1e-5, atol=0.0)
    assert np.array_equal(flags.cpu().numpy(), rflags)
    assert counts.cpu().tolist() == [int(c) for c in rcounts]
    return rfim.rfim_last_variant(), rcounts


@pytest.mark.parametrize("C,S,nb", [(64, 100, 0), (64, 37, 32), (96, 20, 8), (33, 50, 0), (20, 16, 1)])
def test_median_replacement_u8(C, S, nb):
    """FDSC with the median strategy: the test still uses mean and sigma, the
    replacement is the lower median of the bin."""
    x = banded((2, C, S), seed=C + S + nb)
    name, counts = check_policy(x, [3.0, 3.0], nb, "median")
    # one bin on 4-byte aligned rows: the strip kernel finds the median on its resident tile; bins: the definition
    assert name == ("fd_u8_strip1_bulk_median" if nb == 0 and S % 4 == 0 and C % 4 != 0 else
                    "fd_u8_strip1_median" if nb == 0 and S % 4 == 0 else "fd_u8_binned_generic"), name
    check_policy(x, [1.0], nb, "median")


@pytest.mark.parametrize("policy", ["mean", "median"])
@pytest.mark.parametrize("C,S,nb", [(64, 100, 0), (64, 37, 32), (96, 20, 8), (1536, 24, 32)])
def test_float32_fdsc(C, S, nb, policy):
    """float32 FDSC, one bin or bins, mean or median."""
    rng = np.random.default_rng(C * 5 + S + nb)
    band = 3.0 * rng.random((2, (C + 31) // 32, 1)).repeat(32, axis=1)[:, :C]
    x = rng.normal(band, 1.0, (2, C, S))
    x[0, C // 3, :] += 8.0
    x[:, :, S // 2] += 10.0
    x = x.astype(np.float32)
    name, counts = check_policy(x, [2.75, 2.75], nb, policy)
    assert name == "fd_f32_generic" and int(counts[0]) > 0
    check_policy(x, [4.0, 3.0, 2.0], nb, policy)
