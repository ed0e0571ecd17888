"""GPU parity: the streaming FDSC kernel (csrc/fd_u8_stream.cuh) through the C ABI vs the CPU oracle, bit-exact:
one bin and the paper's per-bin mean correction (8f NEXT-1),
in place (only replaced samples are written) and out of place (copy + repair)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"
STREAM = rfim.VARIANT_FD_STREAM


def noisy(shape, seed, mu=100, sigma=12):
    rng = np.random.default_rng(seed)
    return np.clip(np.rint(rng.normal(mu, sigma, shape)), 0, 255).astype(np.uint8)


def banded(shape, seed, block=32):
    """Gaussian noise on a bandpass that differs per `block` channels (what the bin correction is for), plus
    narrow-band RFI, a broadband spike and a dropout."""
    rng = np.random.default_rng(seed)
    B, C, S = shape
    band = 60 + 80 * rng.random((B, (C + block - 1) // block, 1)).repeat(block, axis=1)[:, :C]
    x = np.clip(np.rint(rng.normal(band, 8, shape)), 0, 255)
    x[0, C // 3, :] += 70
    x[:, :, S // 2] += 90
    x[B - 1, C - 1, ::5] = 0
    return np.clip(x, 0, 255).astype(np.uint8)


def check(x_np, ks, bin_size=0, inplace=False, pitch=None, want=None, base_shift=0, variant=STREAM):
    B, C, S = x_np.shape
    ref, rflags, rcounts = oracle.freq_sigma_cut(x_np, ks, bin_size=bin_size)
    P = pitch or S
    buf = torch.full((B * C * P + 64,), 0x5A, dtype=torch.uint8, device=DEV)
    xv = buf[base_shift:base_shift + B * C * P].view(B, C, P)
    xv[:, :, :S] = torch.from_numpy(x_np).to(DEV)
    x = xv[:, :, :S]
    obuf = torch.full((B * C * P + 64,), 0xAB, dtype=torch.uint8, device=DEV)
    out = None if inplace else obuf[base_shift:base_shift + B * C * P].view(B, C, P)[:, :, :S]
    flags = torch.full((B, C, S), 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((len(ks),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(x, ks, out=out, bin_size=bin_size, flags=flags, counts=counts, variant=variant)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    got = res.cpu().numpy()
    assert np.array_equal(got, ref), f"{name}: cleaned array differs at {np.argwhere(got != ref)[:5]}"
    assert np.array_equal(flags.cpu().numpy(), rflags), f"{name}: flags differ"
    assert counts.cpu().tolist() == [int(c) for c in rcounts], f"{name}: counts"
    # nothing outside the samples is written: pitch padding, the bytes before / after the buffers
    if P != S:
        assert torch.all(xv[:, :, S:] == 0x5A)
        if not inplace:
            assert torch.all(obuf[base_shift:base_shift + B * C * P].view(B, C, P)[:, :, S:] == 0xAB)
    assert torch.all(buf[:base_shift] == 0x5A) and torch.all(buf[base_shift + B * C * P:] == 0x5A)
    if not inplace:
        assert torch.all(obuf[:base_shift] == 0xAB) and torch.all(obuf[base_shift + B * C * P:] == 0xAB)
        assert torch.equal(x.cpu(), torch.from_numpy(x_np)), "input modified by an out-of-place call"
    if want:
        assert name == want, name
    return name, rcounts


@pytest.mark.parametrize("C", [512, 1024, 1536, 2048])
@pytest.mark.parametrize("S", [128, 300, 257 * 4 + 2, 44])
def test_one_bin_shapes(C, S):
    """Every supported channel count; sample counts that give whole tiles, a ragged last tile (300 = 2 x 128 + 44),
    a last word with 2 valid bytes (S = 1030: the byte-granular path) and a single ragged tile."""
    if S % 4 != 0:
        x = noisy((2, C, S), seed=C + S)
        x[0, C // 2, :] = 250
        # S not a multiple of 4: rows are not 4-byte aligned on the dense pitch -> not this kernel's request
        with pytest.raises(rfim.RfimError) as e:
            rfim.rfim_freq_sigma_cut(torch.from_numpy(x).to(DEV), [3.0], variant=STREAM)
        assert e.value.status == -2
        # ... but with a padded pitch they are, and the last word of a row has S % 4 valid bytes
        check(x, [4.0, 3.0], pitch=S + 6, want="fd_u8_stream_copy")
        check(x, [4.0, 3.0], pitch=S + 6, inplace=True, want="fd_u8_stream")
        return
    x = noisy((3, C, S), seed=C * 3 + S)
    x[0, C // 2, :] = np.minimum(x[0, C // 2, :].astype(int) + 90, 255).astype(np.uint8)   # narrow-band RFI
    x[1, 1, S // 2] = 255
    x[2, C - 1, S - 1] = 0
    x[0, :, 0] = 77                                                                          # constant column
    x[2, ::97, :] = 240
    check(x, [4.0, 3.0], want="fd_u8_stream_copy")
    check(x, [3.25, 3.25, 3.25], inplace=True, want="fd_u8_stream")


def test_config3_slice_and_many_tiles():
    """More tiles than resident CTAs (5 beams x 98 tiles > 2 x 148): ring phases across tiles, accumulator
    double-buffering, the prefetch of the next tile's boxes."""
    cfg = synth.config(3, beams=5)
    x = synth.fill_host(cfg, beam0=31, beams=5)
    check(x, cfg["thresholds"], inplace=True, want="fd_u8_stream")
    check(x[:2], cfg["thresholds"], want="fd_u8_stream_copy")


@pytest.mark.parametrize("pitch,shift", [(1008, 0), (1004, 4), (1012, 8), (1024, 12), (1000, 4)])
def test_pitch_and_base_alignment(pitch, shift):
    """Every 16-byte phase pattern of the rows (pitch mod 16) and of the base pointers (4, 8, 12 bytes past a
    16-byte boundary, src and dst alike)."""
    x = noisy((2, 512, 1000), seed=pitch + shift)
    x[:, 9, :] = 200
    x[1, :, 500] = 250
    check(x, [4.0, 3.0], pitch=pitch, base_shift=shift)
    check(x, [4.0, 3.0], pitch=pitch, base_shift=shift, inplace=True)


def test_src_and_dst_with_different_phase():
    """Unlike the strip kernel, the streaming kernel does not need src and dst to share their 16-byte phase."""
    x = noisy((1, 512, 400), seed=5)
    x[0, 3, :] = 250
    xd = torch.from_numpy(x).to(DEV)
    ref, _, _ = oracle.freq_sigma_cut(x, [3.0, 3.0])
    for shift in (4, 8, 12, 16):
        obuf = torch.zeros(512 * 400 + 64, dtype=torch.uint8, device=DEV)
        out = obuf[shift:shift + 512 * 400].view(1, 512, 400)
        rfim.rfim_freq_sigma_cut(xd, [3.0, 3.0], out=out, variant=STREAM)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), ref)
        assert int(obuf[:shift].sum()) == 0 and int(obuf[shift + 512 * 400:].sum()) == 0
    with pytest.raises(rfim.RfimError) as e:                     # dst not 4-byte aligned: not this kernel
        rfim.rfim_freq_sigma_cut(xd, [3.0], out=obuf[1:1 + 512 * 400].view(1, 512, 400), variant=STREAM)
    assert e.value.status == -2


def test_degenerate_columns():
    C = 512
    x = np.zeros((1, C, 12), dtype=np.uint8)
    x[0, :, 1] = 255
    x[0, ::2, 2] = 100; x[0, 1::2, 2] = 101        # sigma = 0.5: tiny thresholds cut everything (empty kept interval)
    x[0, :, 3] = 100; x[0, 5, 3] = 160             # single spike
    x[0, :, 4] = 0; x[0, -1, 4] = 255
    x[0, :, 5] = 255; x[0, 0, 5] = 0
    x[0, :, 6] = noisy((C,), 1, 250, 10)
    x[0, :, 7] = noisy((C,), 2, 3, 5)
    x[0, : C // 2, 8] = 10; x[0, C // 2:, 8] = 240
    x[0, :, 9] = noisy((C,), 3)
    x[0, :, 10] = (np.arange(C) % 256).astype(np.uint8)
    x[0, :, 11] = np.where(np.arange(C) % 50 < 3, 250, noisy((C,), 4))
    for ks in ([3.0], [0.4], [0.4, 0.4, 3.0], [1.0, 1.0], [4.0, 3.0], [200.0], [2.0 ** -16], [2.75] * 16):
        check(x, ks)
        check(x, ks, inplace=True)


def test_heavy_rfi_and_many_iterations():
    x = noisy((2, 1536, 300), seed=21)
    x[0, 100:600, :] = np.minimum(x[0, 100:600, :].astype(int) + 90, 255).astype(np.uint8)   # a third of the band
    x[1, ::7, :] = 255
    x[1, :, 100:110] = 3
    for ks in ([3.0], [2.75, 2.75], [1.5, 2.5, 3.5, 4.5], [1.0] * 6):
        check(x, ks)
        check(x, ks, inplace=True)


def test_worked_example_p3_along_channels():
    """15 x 100 and one 160 across channels ... embedded in 512 channels of 100: mu = 100.117, one spike:
    k = {3,3,3}: the 160 is cut to the rounded mean 100, then nothing (tests/test_oracle_pins.py P2 / P3 logic)."""
    x = np.full((1, 512, 8), 100, dtype=np.uint8)
    x[0, 5, 3] = 160
    name, counts = check(x, [3.0, 3.0, 3.0])
    assert [int(c) for c in counts] == [1, 0, 0]


# ------------------------------------------------------------------------------------------- bins
@pytest.mark.parametrize("C,nb", [(1536, 32), (1536, 16), (1536, 64), (1536, 96), (1536, 128), (512, 32), (512, 128),
                                  (1024, 256), (2048, 32), (2048, 64)])
def test_binned(C, nb):
    """PAPER.md:102 step 1 with bins of nb channels (Fig. 5: 32): bin sizes that are a multiple of 16 and divide the
    32 * (C / 128) channels of a warp quartet; two iterations at 2.75 sigma and a three-step list."""
    x = banded((2, C, 260), seed=C + nb, block=nb)
    check(x, [2.75, 2.75], nb, want="fd_u8_stream_binned_copy")
    check(x, [4.0, 3.0, 3.0], nb, inplace=True, want="fd_u8_stream_binned")
    check(x, [0.5], nb)


def test_binned_refused_shapes_fall_back():
    """Bin sizes the streaming kernel does not take run in the generic binned kernel in auto mode."""
    x = banded((1, 1536, 64), seed=3, block=24)
    xd = torch.from_numpy(x).to(DEV)
    for nb in (24, 8, 512):
        with pytest.raises(rfim.RfimError) as e:
            rfim.rfim_freq_sigma_cut(xd.clone(), [2.75], bin_size=nb, variant=STREAM)
        assert e.value.status == -2
        y = xd.clone()
        rfim.rfim_freq_sigma_cut(y, [2.75], bin_size=nb)
        torch.cuda.synchronize()
        assert rfim.rfim_last_variant() == "fd_u8_binned_generic"
        assert np.array_equal(y.cpu().numpy(), oracle.freq_sigma_cut(x, [2.75], bin_size=nb)[0])


def test_binned_config3_size_fig5_parameters():
    """BASELINE.json configs[2] shape (12 x 1536 x 12500) with the paper's FDSC parameters: bins of 32 channels at
    2.75 sigma, 3 beams compared element by element."""
    cfg = synth.config(3, beams=3)
    x = synth.fill_host(cfg, beam0=4, beams=3)
    check(x, [2.75, 2.75], 32, inplace=True, want="fd_u8_stream_binned")


def test_binned_degenerate():
    C = 512
    x = np.zeros((1, C, 8), dtype=np.uint8)
    x[0, :, 1] = 255
    x[0, :, 2] = np.repeat(np.array([10, 200] * (C // 64), dtype=np.uint8), 32)     # bin-wise constant: nothing cut
    x[0, :, 3] = x[0, :, 2]; x[0, 40, 3] = 90                                        # one outlier inside a bin
    x[0, :, 4] = noisy((C,), 5)
    x[0, ::2, 5] = 100; x[0, 1::2, 5] = 101
    x[0, :, 6] = (np.arange(C) % 256).astype(np.uint8)
    x[0, :, 7] = noisy((C,), 6, 250, 20)
    for ks in ([2.75], [0.4, 0.4], [1.0, 2.0, 3.0], [200.0], [2.0 ** -16]):
        check(x, ks, 32)
        check(x, ks, 32, inplace=True)


def test_other_stream_no_flags_no_counts():
    x = noisy((2, 1024, 700), seed=81)
    x[0, 7, :] = 255
    xd = torch.from_numpy(x).to(DEV)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rfim.rfim_freq_sigma_cut(xd, [3.0], stream=s, variant=STREAM)
    s.synchronize()
    assert np.array_equal(xd.cpu().numpy(), oracle.freq_sigma_cut(x, [3.0])[0])
