"""GPU parity: the pooled-repair FDSC kernel with the paper's per-bin mean correction (csrc/fd_u8_qbin.cuh;
PAPER.md:102 step 1, :108, :126) through the C ABI vs the CPU oracle, bit-exact: cleaned
array, flags, counts, in place (only replaced samples are written) and out of place (copy + repair)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

from test_gpu_fd_stream import banded, check, noisy

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
QBIN = rfim.VARIANT_FD_QBIN


@pytest.mark.parametrize("C,nb", [(1536, 32), (1536, 16), (1536, 48), (1536, 64), (1536, 96), (1536, 128), (1536, 192),
                                  (1536, 256), (512, 16), (512, 32), (512, 128), (512, 256), (1024, 64), (1024, 256),
                                  (2048, 32), (2048, 64), (2048, 256)])
def test_bin_sizes(C, nb):
    """Every channel count (256 x {2, 4, 6, 8}) and bin sizes that are a multiple of 16, at most 256 and divide half
    the channels -- also the ones the 16-warp streaming kernel refuses (48, 192 and 256 of 1536): two iterations at
    2.75 sigma, a three-step list in place, and a cut that replaces a large part of the data."""
    x = banded((2, C, 260), seed=C + nb, block=nb)
    check(x, [2.75, 2.75], nb, want="fd_u8_qbin_copy", variant=QBIN)
    check(x, [4.0, 3.0, 3.0], nb, inplace=True, want="fd_u8_qbin", variant=QBIN)
    check(x, [0.5], nb, variant=QBIN)


def test_auto_mode_takes_it():
    x = banded((2, 1536, 200), seed=7)
    check(x, [2.75, 2.75], 32, want="fd_u8_qbin_copy", variant=rfim.VARIANT_AUTO)
    check(x, [2.75, 2.75], 32, inplace=True, want="fd_u8_qbin", variant=rfim.VARIANT_AUTO)


@pytest.mark.parametrize("S", [128, 300, 257 * 4 + 2, 44, 3])
def test_sample_counts(S):
    """Whole tiles, a ragged last tile, a last word with 2 or 3 valid bytes (the byte-granular path: rows made
    4-byte aligned by a padded pitch) and a single ragged tile."""
    x = banded((2, 512, S), seed=S)
    pitch = None if S % 4 == 0 else ((S + 3) // 4) * 4 + 4
    check(x, [2.75, 2.75], 32, pitch=pitch, want="fd_u8_qbin_copy", variant=QBIN)
    check(x, [3.0, 2.0, 2.0], 64, pitch=pitch, inplace=True, want="fd_u8_qbin", variant=QBIN)


@pytest.mark.parametrize("pitch,shift", [(1008, 0), (1004, 4), (1012, 8), (1024, 12), (1000, 4)])
def test_pitch_and_base_alignment(pitch, shift):
    x = banded((2, 512, 1000), seed=pitch + shift)
    check(x, [2.75, 2.75], 32, pitch=pitch, base_shift=shift, variant=QBIN)
    check(x, [2.75, 2.75], 32, pitch=pitch, base_shift=shift, inplace=True, variant=QBIN)


def test_many_tiles_config3_data():
    """More tiles than resident CTAs (7 beams x 98 tiles > 2 x 148): ring phases across tiles, both bin-sum buffers,
    the accumulator double-buffering, the tickets; BASELINE.json configs[2] data with the Fig. 5 parameters."""
    cfg = synth.config(3, beams=7)
    x = synth.fill_host(cfg, beam0=17, beams=7)
    check(x, [2.75, 2.75], 32, inplace=True, want="fd_u8_qbin", variant=QBIN)
    check(x[:2], [2.75, 2.75, 2.75], 32, want="fd_u8_qbin_copy", variant=QBIN)


def test_refused_requests():
    x = banded((1, 1536, 64), seed=3, block=24)
    xd = torch.from_numpy(x).to(DEV)
    for kw in ({"bin_size": 24}, {"bin_size": 8}, {"bin_size": 512}, {"bin_size": 0}, {"bin_size": 32, "policy": "median"}):
        with pytest.raises(rfim.RfimError) as e:
            rfim.rfim_freq_sigma_cut(xd.clone(), [2.75], variant=QBIN, **kw)
        assert e.value.status == -2, kw
    with pytest.raises(rfim.RfimError) as e:                     # 1280 channels: not a multiple of 256
        rfim.rfim_freq_sigma_cut(torch.zeros((1, 1280, 64), dtype=torch.uint8, device=DEV), [2.75], bin_size=32, variant=QBIN)
    assert e.value.status == -2


def test_degenerate_columns():
    C = 512
    x = np.zeros((1, C, 12), dtype=np.uint8)
    x[0, :, 1] = 255
    x[0, :, 2] = np.repeat(np.array([10, 200] * (C // 64), dtype=np.uint8), 32)     # bin-wise constant: nothing cut
    x[0, :, 3] = x[0, :, 2]; x[0, 40, 3] = 90                                        # one outlier inside a bin
    x[0, :, 4] = noisy((C,), 5)
    x[0, ::2, 5] = 100; x[0, 1::2, 5] = 101        # sigma = 0.5: tiny thresholds cut everything (empty kept interval)
    x[0, :, 6] = (np.arange(C) % 256).astype(np.uint8)
    x[0, :, 7] = noisy((C,), 6, 250, 20)
    x[0, :, 8] = 0; x[0, -1, 8] = 255
    x[0, :, 9] = 255; x[0, 0, 9] = 0
    x[0, : C // 2, 10] = 10; x[0, C // 2:, 10] = 240
    x[0, :, 11] = np.where(np.arange(C) % 50 < 3, 250, noisy((C,), 4))
    for ks in ([2.75], [0.4, 0.4], [0.4, 0.4, 3.0], [1.0, 2.0, 3.0], [200.0], [2.0 ** -16], [2.75] * 16):
        for nb in (32, 16, 256):
            check(x, ks, nb, variant=QBIN)
            check(x, ks, nb, inplace=True, variant=QBIN)


def test_heavy_rfi_overflows_the_candidate_list():
    """A third of the band raised and every seventh channel saturated: far more than 256 candidate blocks per warp
    and iteration (the repair list is worked off in chunks), many iterations with column and bin deltas."""
    x = noisy((2, 1536, 300), seed=21)
    x[0, 100:600, :] = np.minimum(x[0, 100:600, :].astype(int) + 90, 255).astype(np.uint8)
    x[1, ::7, :] = 255
    x[1, :, 100:110] = 3
    for ks in ([3.0], [2.75, 2.75], [1.5, 2.5, 3.5, 4.5], [1.0] * 6):
        check(x, ks, 32, variant=QBIN)
        check(x, ks, 64, inplace=True, variant=QBIN)


def test_other_stream_no_flags_no_counts():
    x = banded((2, 1024, 700), seed=81)
    xd = torch.from_numpy(x).to(DEV)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rfim.rfim_freq_sigma_cut(xd, [2.75, 2.75], bin_size=32, stream=s, variant=QBIN)
    s.synchronize()
    assert rfim.rfim_last_variant() == "fd_u8_qbin"
    assert np.array_equal(xd.cpu().numpy(), oracle.freq_sigma_cut(x, [2.75, 2.75], bin_size=32)[0])
