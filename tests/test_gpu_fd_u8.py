"""GPU parity: rfim_freq_sigma_cut (uint8, one bin) through the C ABI vs the CPU oracle, bit-exact.

Cleaned array, flag mask and per-iteration counts must be identical (BASELINE.json north_star).
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu

DEV = "cuda:0"
TILE, GENERIC = rfim.VARIANT_STAGED, rfim.VARIANT_GENERIC
STRIP, STRIP_BULK, STRIP_CLUSTER, STREAM = (rfim.VARIANT_FD_STRIP, rfim.VARIANT_FD_STRIP_BULK,
                                            rfim.VARIANT_FD_STRIP_CLUSTER, rfim.VARIANT_FD_STREAM)


def fast_name(C, S, inplace=False):
    """The tuned kernel auto mode picks for a dense [.][C][S] uint8 request with mean replacement and one bin."""
    if S % 4 != 0:
        return "fd_u8_generic"
    return "fd_u8_strip"          # short batches: the resident-tile kernel (large ones in place: fd_u8_quad)


def run_gpu(x_np, ks, variant=rfim.VARIANT_AUTO, inplace=False, pitch=None, want_flags=True):
    B, C, S = x_np.shape
    if pitch is None:
        x = torch.from_numpy(x_np).to(DEV)
        out = None if inplace else torch.full_like(x, 0xAB)
    else:
        buf = torch.full((B, C, pitch), 0x5A, dtype=torch.uint8, device=DEV)
        buf[:, :, :S] = torch.from_numpy(x_np).to(DEV)
        x = buf[:, :, :S]
        obuf = torch.full((B, C, pitch), 0xAB, dtype=torch.uint8, device=DEV)
        out = None if inplace else obuf[:, :, :S]
    flags = torch.full((B, C, S), 7, dtype=torch.uint8, device=DEV) if want_flags else None
    counts = torch.full((max(1, len(ks)),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(x, ks, out=out, flags=flags, counts=counts, variant=variant)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    if pitch is not None:
        assert torch.all(buf[:, :, S:] == 0x5A), "padding columns of the input were touched"
        if not inplace:
            assert torch.all(obuf[:, :, S:] == 0xAB), "padding columns of the output were touched"
    if not inplace:
        assert torch.equal(x.cpu(), torch.from_numpy(x_np)), "input modified by an out-of-place call"
    return (res.cpu().numpy(), flags.cpu().numpy() if want_flags else None,
            counts.cpu().numpy()[:len(ks)], name)


def check(x_np, ks, **kw):
    ref, rflags, rcounts = oracle.freq_sigma_cut(x_np, ks)
    got, gflags, gcounts, name = run_gpu(x_np, ks, **kw)
    assert np.array_equal(got, ref), f"{name}: cleaned array differs at {np.argwhere(got != ref)[:5]}"
    assert np.array_equal(gflags, rflags), f"{name}: flags differ at {np.argwhere(gflags != rflags)[:5]}"
    assert gcounts.tolist() == [int(c) for c in rcounts], f"{name}: counts {gcounts} vs {rcounts}"
    return name, rcounts


def noisy(shape, seed, mu=100, sigma=12):
    rng = np.random.default_rng(seed)
    return np.clip(np.rint(rng.normal(mu, sigma, shape)), 0, 255).astype(np.uint8)


# ----------------------------------------------------------------------------------- configs
@pytest.mark.parametrize("variant", [TILE, GENERIC])
def test_config1_shape_fd(variant):
    """BASELINE.json configs[0] data through FDSC: the +60 channels 7 and 40 ARE outliers across
    channels (FDSC removes bright narrow-band signals) -- SURVEY.md pin P13."""
    cfg = synth.config(1)
    x = synth.fill_host(cfg)
    name, counts = check(x, [3.0], variant=variant)
    assert name == ("fd_u8_strip1" if variant == TILE else "fd_u8_generic")
    # (the oracle-side pin P13 lives in tests/test_oracle_pins.py::test_p13_config1_behaviour)


def test_config3_arts_like_all_beams():
    """BASELINE.json configs[2]: 12 x 1536 x 12500 uint8, FDSC k = {4,3}; every element compared."""
    cfg = synth.config(3)
    B, C, S = cfg["beams"], cfg["channels"], cfg["samples"]
    x = torch.empty((B, C, S), dtype=torch.uint8, device=DEV)
    synth.fill_device(cfg, x)
    x_np = x.cpu().numpy()
    name, counts = check(x_np, cfg["thresholds"], inplace=True)      # auto: the strip kernel on a 12-beam batch
    assert name in ("fd_u8_strip1", "fd_u8_quad", "fd_u8_stream")
    assert all(int(c) > 0 for c in counts)
    name, _ = check(x_np[:3], cfg["thresholds"])                      # auto, out of place
    assert name in ("fd_u8_strip1", "fd_u8_quad_copy", "fd_u8_stream_copy")
    name, _ = check(x_np[:3], cfg["thresholds"], inplace=True, variant=STREAM)
    assert name == "fd_u8_stream"
    name, _ = check(x_np[:2], cfg["thresholds"], variant=STREAM)      # out of place: copy + repair
    assert name == "fd_u8_stream_copy"
    name, _ = check(x_np[:2], cfg["thresholds"], inplace=True, variant=STRIP)
    assert name == "fd_u8_strip1"
    check(x_np[:1], cfg["thresholds"], variant=GENERIC)


def test_config4_chain_two_beams():
    """BASELINE.json configs[3] on a 2-beam slice: TDSC {5,4,3} then FDSC {4,3}, in place."""
    cfg = synth.config(4, beams=2)
    x = synth.fill_host(cfg, beam0=17, beams=2)
    xd = torch.from_numpy(x).to(DEV)
    rfim.rfim_time_sigma_cut(xd, cfg["thresholds"])
    rfim.rfim_freq_sigma_cut(xd, cfg["freq_thresholds"])
    torch.cuda.synchronize()
    ref, _, _ = oracle.time_sigma_cut(x, cfg["thresholds"])
    ref, _, _ = oracle.freq_sigma_cut(ref, cfg["freq_thresholds"])
    assert np.array_equal(xd.cpu().numpy(), ref)


# --------------------------------------------------------------------- shapes, tails, alignment
@pytest.mark.parametrize("C,S", [(1, 40), (2, 64), (4, 1), (8, 63), (12, 65), (64, 100), (100, 257), (384, 1000),
                                 (1536, 212), (2000, 96), (4096, 70), (7000, 33)])
@pytest.mark.parametrize("variant", [rfim.VARIANT_AUTO, GENERIC])
def test_shapes(C, S, variant):
    """Row pitch S runs through every 16-byte phase pattern (S mod 16 = 0, 8, 4, 12; S not a multiple of 4 takes
    the generic path); channel counts that are not multiples of the row groups or the cluster size; ragged tiles."""
    x = noisy((2, C, S), seed=C * 7 + S)
    if C >= 8:
        x[0, C // 2, :] = np.minimum(x[0, C // 2, :].astype(int) + 90, 255).astype(np.uint8)   # narrow-band RFI
        x[1, 1, S // 2] = 255
        x[1, C - 1, S - 1] = 0
        x[0, :, 0] = 77                                                                          # constant column
    name, _ = check(x, [4.0, 3.0], variant=variant)
    assert name.startswith("fd_u8_generic" if variant == GENERIC else fast_name(C, S)), name
    check(x, [3.25, 3.25, 3.25], variant=variant, inplace=True)


@pytest.mark.parametrize("pitch", [1008, 1004, 1002, 1001, 1024])
def test_padded_pitch(pitch):
    x = noisy((3, 64, 1000), seed=pitch)
    x[:, 9, :] = 200
    x[1, :, 500] = 250
    check(x, [4.0, 3.0], pitch=pitch)
    check(x, [4.0, 3.0], pitch=pitch, inplace=True)


def test_misaligned_out():
    """out with another 16-byte phase than data: the aligned interiors of the rows do not coincide, so only the
    generic kernel can run; a whole 16 bytes off is fine for the cluster kernel."""
    x = noisy((1, 16, 1000), seed=12)
    x[0, 3, :] = 250
    xd = torch.from_numpy(x).to(DEV)
    ref, _, _ = oracle.freq_sigma_cut(x, [3.0])
    for shift, want in ((4, "fd_u8_generic"), (1, "fd_u8_generic"), (16, "fd_u8_strip1")):
        obuf = torch.zeros(16 * 1000 + 64, dtype=torch.uint8, device=DEV)
        out = obuf[shift:shift + 16000].view(1, 16, 1000)
        rfim.rfim_freq_sigma_cut(xd, [3.0], out=out)
        torch.cuda.synchronize()
        assert rfim.rfim_last_variant().startswith(want)
        assert np.array_equal(out.cpu().numpy(), ref)
        assert int(obuf[:shift].sum()) == 0 and int(obuf[shift + 16000:].sum()) == 0
    out = obuf[4:4 + 16000].view(1, 16, 1000)
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_freq_sigma_cut(xd, [3.0], out=out, variant=TILE)
    assert e.value.status == -2
    # out overlapping data without being data is refused (include/rfim.h)
    big = torch.zeros(2 * 16000, dtype=torch.uint8, device=DEV)
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_freq_sigma_cut(big[:16000].view(1, 16, 1000), [3.0], out=big[8000:24000].view(1, 16, 1000))
    assert e.value.status == -1


def test_unaligned_base_pointer_tile_path():
    """data and out both 4 bytes past a 16-byte boundary: the class offsets absorb it."""
    x = noisy((2, 32, 500), seed=13)
    x[:, 5, :] = 230
    buf = torch.zeros(2 * 32 * 500 + 16, dtype=torch.uint8, device=DEV)
    v = buf[4:4 + 2 * 32 * 500].view(2, 32, 500)
    v.copy_(torch.from_numpy(x).to(DEV))
    rfim.rfim_freq_sigma_cut(v, [4.0, 3.0])
    torch.cuda.synchronize()
    assert rfim.rfim_last_variant().startswith("fd_u8_strip")
    ref, _, _ = oracle.freq_sigma_cut(x, [4.0, 3.0])
    assert np.array_equal(v.cpu().numpy(), ref)
    assert int(buf[:4].sum()) == 0 and int(buf[4 + 2 * 32 * 500:].sum()) == 0


# ----------------------------------------------------------------------------- degenerate data
@pytest.mark.parametrize("variant", [rfim.VARIANT_AUTO, GENERIC])
def test_degenerate_columns(variant):
    C = 776
    x = np.zeros((1, C, 12), dtype=np.uint8)
    x[0, :, 0] = 0
    x[0, :, 1] = 255
    x[0, ::2, 2] = 100; x[0, 1::2, 2] = 101        # sigma = 0.5: tiny thresholds cut everything
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
        check(x, ks, variant=variant)


def test_worked_example_p3_along_channels():
    """15 x 100 and one 160 across channels, k = {3,3,3} -> 104 -> 100 (tests/test_oracle_pins.py P3)."""
    x = np.full((1, 16, 8), 100, dtype=np.uint8)
    x[0, 5, 3] = 160
    for variant in (rfim.VARIANT_AUTO, GENERIC):
        got, flags, counts, _ = run_gpu(x, [3.0, 3.0, 3.0], variant=variant)
        assert (got == 100).all() and counts.tolist() == [1, 1, 0] and flags.sum() == 1
        got, _, _, _ = run_gpu(x, [3.0], variant=variant)
        assert got[0, 5, 3] == 104


def test_heavy_rfi():
    x = noisy((2, 1536, 300), seed=21)
    x[0, 100:600, :] = np.minimum(x[0, 100:600, :].astype(int) + 90, 255).astype(np.uint8)   # a third of the band
    x[1, ::7, :] = 255
    x[1, :, 100:110] = 3
    for ks in ([3.0], [2.75, 2.75], [1.5, 2.5, 3.5, 4.5]):
        check(x, ks)
        check(x, ks, variant=GENERIC)


def test_many_tiles_grid_wraps():
    """More tiles than resident CTAs: the persistent loop reuses the tile buffer (mbarrier phase, bulk groups)."""
    x = noisy((40, 64, 2100), seed=71)
    x[:, 9, ::5] = 255
    name, _ = check(x, [4.0, 3.0])
    assert name == "fd_u8_strip1"
    name, _ = check(np.ascontiguousarray(x[:, :, :2096]), [4.0, 3.0])
    assert name == "fd_u8_strip1"
    check(x[:13], [4.0, 3.0], variant=STRIP_CLUSTER)


def test_no_flags_no_counts_other_stream():
    x = noisy((1, 256, 2000), seed=81)
    x[0, 7, :] = 255
    xd = torch.from_numpy(x).to(DEV)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rfim.rfim_freq_sigma_cut(xd, [3.0], stream=s)
    s.synchronize()
    ref, _, _ = oracle.freq_sigma_cut(x, [3.0])
    assert np.array_equal(xd.cpu().numpy(), ref)


def test_zero_thresholds_is_copy():
    x = noisy((2, 3, 100), seed=61)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.zeros_like(xd)
    rfim.rfim_freq_sigma_cut(xd, [], out=out)
    torch.cuda.synchronize()
    assert torch.equal(out, xd)


def test_unsupported_requests_fail_loudly():
    x = torch.zeros((1, 64, 128), dtype=torch.uint8, device=DEV)
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_freq_sigma_cut(x, [3.0], policy="median", bin_size=16, variant=TILE)   # no tuned kernel for median with bins
    assert e.value.status == -2


# ------------------------------------------------------------------------ strip kernel: cluster sizes by channel count
@pytest.mark.parametrize("C,name", [(700, "fd_u8_strip1_bulk"), (768, "fd_u8_strip1"), (1537, "fd_u8_strip1_bulk"), (3001, "fd_u8_strip4_bulk"),
                                    (6100, "fd_u8_strip8_bulk"), (1536, "fd_u8_strip1"), (3072, "fd_u8_strip4"),
                                    (6144, "fd_u8_strip8"), (1028, "fd_u8_strip1_bulk"), (1024, "fd_u8_strip1"),
                                    (1280, "fd_u8_strip1"), (1152, "fd_u8_strip1")])
def test_strip_cluster_sizes(C, name):
    """The strip kernel splits the channels over the smallest cluster whose CTAs fit two to an SM: uneven splits,
    a ragged last tile (S = 300 = 2 x 128 + 44), RFI channels in every CTA, empty kept intervals."""
    x = noisy((2, C, 300), seed=C)
    x[0, ::97, :] = 250
    x[1, C // 2:C // 2 + 40, 17:60] = 0
    x[1, :, 299] = 7
    got, _ = check(x, [4.0, 3.0], variant=STRIP)
    assert got == name
    got, _ = check(x, [4.0, 3.0])                      # auto: short batches go to the strip kernel too
    assert got == name
    check(x, [0.5, 3.0, 3.0], inplace=True, variant=STRIP)
    got, _ = check(x, [4.0, 3.0], variant=STRIP_BULK)  # the same kernel with per-row bulk copies
    assert got == name.replace("_bulk", "") + "_bulk"
    got, _ = check(x, [4.0, 3.0], variant=STRIP_CLUSTER)   # never the whole tile in one CTA: clusters, two CTAs per SM
    assert got.startswith("fd_u8_strip2" if C in (1536, 1537, 1028, 1024, 1280, 1152) else name.replace("_bulk", ""))


# ----------------------------------------------------------------------------------- median replacement (NEXT-3)
def check_median(x_np, ks, inplace=False, variant=rfim.VARIANT_AUTO, want=None):
    ref, rflags, rcounts = oracle.freq_sigma_cut(x_np, ks, policy=oracle.MEDIAN)
    x = torch.from_numpy(x_np).to(DEV)
    out = None if inplace else torch.full_like(x, 0xAB)
    flags = torch.full(x_np.shape, 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((len(ks),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_freq_sigma_cut(x, ks, "median", out=out, flags=flags, counts=counts, variant=variant)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    got = res.cpu().numpy()
    assert np.array_equal(got, ref), f"{name}: cleaned array differs at {np.argwhere(got != ref)[:5]}"
    assert np.array_equal(flags.cpu().numpy(), rflags), f"{name}: flags differ"
    assert counts.cpu().tolist() == [int(c) for c in rcounts], f"{name}: counts"
    if want:
        assert name == want, name
    return name


@pytest.mark.parametrize("C,S,want", [(1536, 300, "fd_u8_strip1_median"), (1536, 128, "fd_u8_strip1_median"),
                                      (512, 212, "fd_u8_strip1_median"), (64, 100, "fd_u8_strip1_median"),
                                      (30, 44, "fd_u8_strip1_bulk_median"), (2, 64, "fd_u8_strip1_bulk_median"),
                                      (4096, 140, "fd_u8_binned_generic")])
def test_median_replacement_in_the_strip_kernel(C, S, want):
    """FDSC with the median strategy on the resident tile: the lower median of every column by
    bisection over the byte values, once per column; the oracle recomputes it in every iteration.  4096 channels
    do not fit one CTA: the definition kernel."""
    x = noisy((2, C, S), seed=C + S)
    if C >= 8:
        x[0, C // 2, :] = np.minimum(x[0, C // 2, :].astype(int) + 90, 255).astype(np.uint8)   # narrow-band RFI
        x[1, ::3, S // 2] = 255                       # a third of a column saturated: median far from the noise
        x[1, C - 1, S - 1] = 0
        x[0, :, 0] = 77                               # constant column
        x[0, : C // 2, 1] = 10                        # two-level column with an even split (lower median = 10)
        x[0, C // 2:, 1] = 200
    check_median(x, [4.0, 3.0], want=want)
    check_median(x, [3.25, 3.25, 3.25], inplace=True, want=want)
    check_median(x, [0.5, 1.0, 2.0, 3.0], inplace=True, want=want)     # k < 1: the kept interval may miss the median


def test_median_config3_slice():
    cfg = synth.config(3, beams=2)
    x = synth.fill_host(cfg, beam0=3, beams=2)
    check_median(x, cfg["thresholds"], inplace=True, want="fd_u8_strip1_median")
    check_median(x[:1], [2.75, 2.75], want="fd_u8_strip1_median")
