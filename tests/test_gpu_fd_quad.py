"""GPU parity: the class-per-warp streaming FDSC kernel (csrc/fd_u8_quad.cuh; one bin)
through the C ABI vs the CPU oracle, bit-exact: cleaned array, flag mask, per-iteration counts; in place (only
replaced samples are written) and out of place (copy + repair)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth
from test_gpu_fd_stream import check as check_variant, noisy

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
QUAD = rfim.VARIANT_FD_QUAD


def check(*a, **kw):
    return check_variant(*a, variant=QUAD, **kw)


@pytest.mark.parametrize("C", [512, 1024, 1536, 2048])
@pytest.mark.parametrize("S", [128, 300, 257 * 4 + 2, 44])
def test_one_bin_shapes(C, S):
    """Every supported channel count; whole tiles, a ragged last tile, a last word with 2 valid bytes (S = 1030 on a
    padded pitch: the byte-granular path) and a single ragged tile."""
    if S % 4 != 0:
        x = noisy((2, C, S), seed=C + S)
        x[0, C // 2, :] = 250
        with pytest.raises(rfim.RfimError) as e:            # dense rows not 4-byte aligned: not this kernel
            rfim.rfim_freq_sigma_cut(torch.from_numpy(x).to(DEV), [3.0], variant=QUAD)
        assert e.value.status == -2
        check(x, [4.0, 3.0], pitch=S + 6, want="fd_u8_quad_copy")
        check(x, [4.0, 3.0], pitch=S + 6, inplace=True, want="fd_u8_quad")
        return
    x = noisy((3, C, S), seed=C * 3 + S)
    x[0, C // 2, :] = np.minimum(x[0, C // 2, :].astype(int) + 90, 255).astype(np.uint8)   # narrow-band RFI
    x[1, 1, S // 2] = 255
    x[2, C - 1, S - 1] = 0
    x[0, :, 0] = 77                                                                          # constant column
    x[2, ::97, :] = 240
    check(x, [4.0, 3.0], want="fd_u8_quad_copy")
    check(x, [3.25, 3.25, 3.25], inplace=True, want="fd_u8_quad")
    check(x, [3.0], inplace=True, want="fd_u8_quad")


def test_config3_slice_and_many_tiles():
    """More tiles than resident CTAs (8 beams x 98 tiles > 4 x 148): ring phases across tiles, accumulator
    double-buffering, the prefetch of the next tile's boxes, tickets."""
    cfg = synth.config(3, beams=8)
    x = synth.fill_host(cfg, beam0=31, beams=8)
    check(x, cfg["thresholds"], inplace=True, want="fd_u8_quad")
    check(x[:2], cfg["thresholds"], want="fd_u8_quad_copy")


def test_many_candidates_overflow_the_list():
    """Heavy contamination: far more than 256 candidate blocks per warp and iteration (a third of all samples are
    outliers of the column statistics), so the candidate list is worked off in several chunks; and an iteration
    that cuts (almost) everything: a column with a tiny variance."""
    rng = np.random.default_rng(9)
    x = noisy((2, 1536, 256), seed=3)
    hot = rng.random(x.shape) < 0.04
    x[hot] = rng.integers(180, 256, size=int(hot.sum()), dtype=np.uint8)
    x[1, ::3, 64:192] = 15
    check(x, [2.0, 1.5, 1.5, 1.0], inplace=True, want="fd_u8_quad")
    check(x, [1.0, 1.0], want="fd_u8_quad_copy")


@pytest.mark.parametrize("pitch,shift", [(1008, 0), (1004, 4), (1012, 8), (1024, 12), (1000, 4)])
def test_pitch_and_base_alignment(pitch, shift):
    x = noisy((2, 512, 1000), seed=pitch + shift)
    x[:, 9, :] = 200
    x[1, :, 500] = 250
    check(x, [4.0, 3.0], pitch=pitch, base_shift=shift)
    check(x, [4.0, 3.0], pitch=pitch, base_shift=shift, inplace=True)


def test_degenerate_columns_and_unsupported_requests():
    C = 512
    x = np.zeros((1, C, 12), dtype=np.uint8)
    x[0, :, 1] = 255
    x[0, :, 2] = 7
    x[0, 5, 2] = 9                       # one spike in a constant column: N > k^2 + 1 -> cut
    x[0, ::2, 3] = 10
    x[0, 1::2, 3] = 20                   # every sample exactly 1 sigma away: k = 1 cuts nothing
    check(x, [1.0, 3.0], inplace=True, want="fd_u8_quad")
    xd = torch.from_numpy(noisy((1, 1536, 256), seed=1)).to(DEV)
    for kw in (dict(bin_size=32), dict(policy="median")):
        with pytest.raises(rfim.RfimError) as e:
            rfim.rfim_freq_sigma_cut(xd.clone(), [3.0], variant=QUAD, **kw)
        assert e.value.status == -2
    with pytest.raises(rfim.RfimError) as e:                # 640 channels: not 128 * {4, 8, 12, 16}
        rfim.rfim_freq_sigma_cut(torch.from_numpy(noisy((1, 640, 256), seed=2)).to(DEV), [3.0], variant=QUAD)
    assert e.value.status == -2


def test_non_default_stream_and_caller_workspace():
    x = noisy((2, 1024, 512), seed=12)
    x[0, 100, :] = 230
    ref, _, _ = oracle.freq_sigma_cut(x, [4.0, 3.0])
    xd = torch.from_numpy(x).to(DEV)
    ws = torch.zeros(256, dtype=torch.uint8, device=DEV)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rfim.rfim_freq_sigma_cut(xd, [4.0, 3.0], stream=s, variant=QUAD, workspace=ws)
    s.synchronize()
    assert np.array_equal(xd.cpu().numpy(), ref)
