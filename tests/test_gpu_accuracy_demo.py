"""Qualitative accuracy demo on the recipe of the paper's Figs. 4-6: a float32
N(0,1) canvas with a faint pulse dispersed at DM = 500 pc cm^-3 (Eq. 2), strong narrow-band bursts
and broadband zero-DM impulses; TDSC three times at 3.25 sigma, then FDSC with bins of 32 channels at 2.75 sigma
(the parameters of PAPER.md:126,178); brute-force dedispersion at the pulse's DM.  The pulse must cross the
detection line only after cleaning.  The paper's own SNR figures need the Crab observation and AMBER and stay
unpinned; this shows the same effect on synthetic data and checks the GPU path against the
oracle on it.  Untimed."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
DETECTION_SNR = 10.0


def make(seed=4, C=256, S=8192, amp=0.55, width=8):
    rng = np.random.default_rng(seed)
    x = rng.normal(0, 1, (1, C, S)).astype(np.float32)
    nu = 1220 + (np.arange(C) + 0.5) * 300 / C                      # channel centres, MHz
    delay = np.rint(4.15e3 * 500 * (nu ** -2 - 1520.0 ** -2) / 81.92e-6).astype(int)
    t0 = 600
    for c in range(C):
        x[0, c, t0 + delay[c]: t0 + delay[c] + width] += amp
    for c in rng.choice(C, C // 8, replace=False):                 # narrow-band channels with strong bursts
        for _ in range(6):
            s = rng.integers(0, S - 400)
            x[0, c, s:s + rng.integers(50, 400)] += rng.uniform(6, 15)
    for _ in range(40):                                            # broadband zero-DM impulses
        s = rng.integers(0, S - 3)
        x[0, :, s:s + 2] += rng.uniform(4, 9)
    return x, delay, t0, width


def pulse_snr(x, delay, t0, width):
    """Dedisperse at the pulse's DM, boxcar of the pulse width, robust noise estimate off pulse."""
    C, S = x.shape[1:]
    n = S - delay.max() - 1
    ts = np.zeros(n)
    for c in range(C):
        ts += x[0, c, delay[c]: delay[c] + n]
    box = np.convolve(ts, np.ones(width), mode="valid")
    off = np.r_[box[: t0 - 50], box[t0 + 50:]]
    med = np.median(off)
    sig = 1.4826 * np.median(np.abs(off - med))
    return (box[t0] - med) / sig


def test_pulse_crosses_the_detection_line_only_after_cleaning():
    x, delay, t0, width = make()
    raw = pulse_snr(x, delay, t0, width)
    xd = torch.from_numpy(x).to(DEV)
    rfim.rfim_time_sigma_cut(xd, [3.25, 3.25, 3.25])
    torch.cuda.synchronize()
    td = xd.cpu().numpy()
    rfim.rfim_freq_sigma_cut(xd, [2.75], bin_size=32)
    torch.cuda.synchronize()
    fd = xd.cpu().numpy()
    snr_td, snr_fd = pulse_snr(td, delay, t0, width), pulse_snr(fd, delay, t0, width)
    assert raw < DETECTION_SNR, raw                                # hidden by the interference
    assert snr_td > raw                                            # TDSC alone already helps ...
    assert snr_fd > DETECTION_SNR and snr_fd > 2.0 * raw, (raw, snr_td, snr_fd)   # ... both together recover it
    # and the GPU path did what the oracle does
    ref, _, _ = oracle.time_sigma_cut(x, [3.25, 3.25, 3.25])
    assert np.allclose(td, ref, rtol=1e-5, atol=0.0)
    ref2, _, _ = oracle.freq_sigma_cut(ref, [2.75], bin_size=32)
    assert np.allclose(fd, ref2, rtol=1e-5, atol=0.0)
