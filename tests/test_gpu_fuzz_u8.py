"""Seeded random shapes, thresholds and contents through the auto-selected uint8 kernels vs the oracle (bit-exact)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def random_case(rng, max_c, max_s, s_mult):
    B = int(rng.integers(1, 4))
    C = int(rng.integers(1, max_c + 1))
    S = int(rng.integers(1, max_s // s_mult + 1)) * s_mult
    kind = int(rng.integers(0, 4))
    if kind == 0:
        x = np.clip(np.rint(rng.normal(rng.uniform(20, 230), rng.uniform(0.5, 40), (B, C, S))), 0, 255)
    elif kind == 1:
        x = rng.integers(0, 256, (B, C, S)).astype(np.float64)
    elif kind == 2:
        x = np.full((B, C, S), float(rng.integers(0, 256)))
        x[rng.random((B, C, S)) < 0.01] = float(rng.integers(0, 256))
    else:
        x = np.clip(np.rint(rng.normal(100, 12, (B, C, S))), 0, 255)
        for _ in range(int(rng.integers(0, 6))):
            x[rng.integers(0, B), rng.integers(0, C), :] += rng.integers(-90, 90)
            x[rng.integers(0, B), :, rng.integers(0, S)] += rng.integers(-90, 90)
        x = np.clip(x, 0, 255)
    ks = [float(rng.choice([0.5, 1.0, 1.5, 2.0, 2.75, 3.0, 3.25, 4.0, 5.0, 16.0])) for _ in range(int(rng.integers(1, 5)))]
    return x.astype(np.uint8), ks


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_time(seed):
    rng = np.random.default_rng(1000 + seed)
    x, ks = random_case(rng, 40, 20000, 1)
    ref, rflags, rcounts = oracle.time_sigma_cut(x, ks)
    xd = torch.from_numpy(x).to(DEV)
    flags = torch.zeros(x.shape, dtype=torch.uint8, device=DEV)
    counts = torch.zeros(len(ks), dtype=torch.int64, device=DEV)
    rfim.rfim_time_sigma_cut(xd, ks, flags=flags, counts=counts)
    torch.cuda.synchronize()
    assert np.array_equal(xd.cpu().numpy(), ref), (rfim.rfim_last_variant(), x.shape, ks)
    assert np.array_equal(flags.cpu().numpy(), rflags) and counts.cpu().tolist() == [int(c) for c in rcounts]


@pytest.mark.parametrize("seed", range(24))
def test_fuzz_freq(seed):
    rng = np.random.default_rng(2000 + seed)
    x, ks = random_case(rng, 1700 if seed % 3 == 0 else 300, 900, 4 if seed % 4 else 1)
    ref, rflags, rcounts = oracle.freq_sigma_cut(x, ks)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.empty_like(xd) if seed % 2 else None
    flags = torch.zeros(x.shape, dtype=torch.uint8, device=DEV)
    counts = torch.zeros(len(ks), dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(xd, ks, out=out, flags=flags, counts=counts)
    torch.cuda.synchronize()
    assert np.array_equal(res.cpu().numpy(), ref), (rfim.rfim_last_variant(), x.shape, ks)
    assert np.array_equal(flags.cpu().numpy(), rflags) and counts.cpu().tolist() == [int(c) for c in rcounts]
