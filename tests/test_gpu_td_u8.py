"""GPU parity: rfim_time_sigma_cut (uint8) through the C ABI vs the CPU oracle, bit-exact.

Cleaned array, flag mask and per-iteration counts must be identical (BASELINE.json north_star:
"The flag mask and the cleaned array must therefore be bit-exact against the oracle").
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def run_gpu(x_np, ks, variant=rfim.VARIANT_AUTO, inplace=False, policy="mean", window=0, pitch=None):
    """x_np: [B][C][S] uint8.  Returns (cleaned, flags, counts, variant_name) as numpy."""
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
    flags = torch.full((B, C, S), 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((max(1, len(ks)),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_time_sigma_cut(x, ks, policy, out=out, window=window, flags=flags, counts=counts,
                                   variant=variant)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    if pitch is not None:
        # padding columns must be untouched
        assert torch.all(buf[:, :, S:] == 0x5A)
        if not inplace:
            assert torch.all(obuf[:, :, S:] == 0xAB)
    if not inplace:
        assert torch.equal(x.cpu(), torch.from_numpy(x_np)), "input modified by an out-of-place call"
    return res.cpu().numpy(), flags.cpu().numpy(), counts.cpu().numpy()[:len(ks)], name


def check(x_np, ks, **kw):
    policy = kw.get("policy", "mean")
    ref, rflags, rcounts = oracle.time_sigma_cut(
        x_np, ks, policy=oracle.MEDIAN if policy == "median" else oracle.MEAN, window=kw.get("window", 0))
    got, gflags, gcounts, name = run_gpu(x_np, ks, **kw)
    assert np.array_equal(got, ref), f"{name}: cleaned array differs at {np.argwhere(got != ref)[:5]}"
    assert np.array_equal(gflags, rflags), f"{name}: flags differ"
    assert gcounts.tolist() == [int(c) for c in rcounts], f"{name}: counts {gcounts} vs {rcounts}"
    return name, rcounts


def noisy(shape, seed, mu=100, sigma=12):
    rng = np.random.default_rng(seed)
    return np.clip(np.rint(rng.normal(mu, sigma, shape)), 0, 255).astype(np.uint8)


# ----------------------------------------------------------------------------------- configs
@pytest.mark.parametrize("variant", [rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC])
def test_config1_tiny(variant):
    """BASELINE.json configs[0]: 1 x 64 x 1024, k = 3, mean."""
    cfg = synth.config(1)
    x = synth.fill_host(cfg)
    name, counts = check(x, cfg["thresholds"], variant=variant)
    assert name == {rfim.VARIANT_STAGED_1W: "td_u8_staged", rfim.VARIANT_STAGED_2W: "td_u8_staged_team2",
                    rfim.VARIANT_GENERIC: "td_u8_generic"}[variant]
    # (the oracle-side pin P13 lives in tests/test_oracle_pins.py::test_p13_config1_behaviour)
    # a constant +60 offset (channels 7, 40) only moves the mean: TDSC leaves it
    got, _, _, _ = run_gpu(x, cfg["thresholds"], variant=variant)
    assert abs(got[0, 7].mean() - 160) < 2 and abs(got[0, 40].mean() - 160) < 2


def test_config2_arts_like_all_beams():
    """BASELINE.json configs[1]: 12 x 1536 x 12500 uint8, k = {5,4,3}; every element compared."""
    cfg = synth.config(2)
    B, C, S = cfg["beams"], cfg["channels"], cfg["samples"]
    x = torch.empty((B, C, S), dtype=torch.uint8, device=DEV)
    synth.fill_device(cfg, x)
    x_np = x.cpu().numpy()
    name, counts = check(x_np, cfg["thresholds"], inplace=True)
    assert name == "td_u8_staged"
    check(x_np[:2], cfg["thresholds"], variant=rfim.VARIANT_STAGED_2W)
    assert all(int(c) > 0 for c in counts)


def test_device_generator_matches_host_twin():
    cfg = synth.config(2)
    x = torch.empty((1, cfg["channels"], cfg["samples"]), dtype=torch.uint8, device=DEV)
    synth.fill_device(cfg, x, beam0=3, beams=1)
    assert np.array_equal(x.cpu().numpy(), synth.fill_host(cfg, beam0=3, beams=1))


# --------------------------------------------------------------------- shapes, tails, alignment
@pytest.mark.parametrize("S", [1, 2, 15, 16, 17, 31, 33, 100, 255, 1000, 4099, 12500])
@pytest.mark.parametrize("variant", [rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC])
def test_row_lengths_and_misalignment(S, variant):
    """Odd S makes consecutive rows start at every 16-byte phase; several 16-byte groups and a ragged tail."""
    x = noisy((2, 19, S), seed=S)
    if S >= 16:
        x[0, 3, S // 2] = 255
        x[1, 5, : S // 8 + 1] = 230
        x[1, 7, 0] = 0
        x[1, 8, S - 1] = 255
        x[0, 0, :] = 42                 # constant row
    name, _ = check(x, [5.0, 4.0, 3.0], variant=variant)
    check(x, [3.25, 3.25, 3.25], variant=variant, inplace=True)


@pytest.mark.parametrize("variant", [rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC])
@pytest.mark.parametrize("pitch", [1040, 1027])
def test_padded_pitch(variant, pitch):
    x = noisy((3, 8, 1000), seed=11)
    x[:, :, 500] = 250
    check(x, [4.0, 3.0], variant=variant, pitch=pitch)
    check(x, [4.0, 3.0], variant=variant, pitch=pitch, inplace=True)


def test_misaligned_out_falls_back_to_generic():
    """out and data with different 16-byte phases cannot share a TMA interior: auto must pick generic."""
    x = noisy((1, 4, 1000), seed=12)
    x[0, :, 10] = 250
    xd = torch.from_numpy(x).to(DEV)
    obuf = torch.zeros(4 * 1000 + 16, dtype=torch.uint8, device=DEV)
    out = obuf[4:4 + 4000].view(1, 4, 1000)
    rfim.rfim_time_sigma_cut(xd, [3.0], out=out)
    torch.cuda.synchronize()
    assert rfim.rfim_last_variant() == "td_u8_generic"
    ref, _, _ = oracle.time_sigma_cut(x, [3.0])
    assert np.array_equal(out.cpu().numpy(), ref)
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_time_sigma_cut(xd, [3.0], out=out, variant=rfim.VARIANT_STAGED)
    assert e.value.status == -2


# ----------------------------------------------------------------------------- degenerate data
@pytest.mark.parametrize("variant", [rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC])
def test_degenerate_rows(variant):
    S = 777
    x = np.zeros((1, 10, S), dtype=np.uint8)
    x[0, 0, :] = 0                                 # all zero
    x[0, 1, :] = 255                               # all saturated
    x[0, 2, ::2] = 100; x[0, 2, 1::2] = 101        # sigma = 0.5: tiny thresholds cut everything
    x[0, 3, :] = 100; x[0, 3, 5] = 160             # single spike (closed form: cut iff N > k^2 + 1)
    x[0, 4, :] = 0; x[0, 4, -1] = 255              # spike at the last byte
    x[0, 5, :] = 255; x[0, 5, 0] = 0               # negative spike at the first byte
    x[0, 6, :] = noisy((S,), 1, 250, 10)           # clipped at 255
    x[0, 7, :] = noisy((S,), 2, 3, 5)              # clipped at 0
    x[0, 8, : S // 2] = 10; x[0, 8, S // 2:] = 240  # bimodal: sigma ~ 115, bounds beyond [0,255]
    x[0, 9, :] = noisy((S,), 3)
    for ks in ([3.0], [0.4], [0.4, 0.4, 3.0], [1.0, 1.0], [5.0, 4.0, 3.0], [200.0], [2.0 ** -16]):
        check(x, ks, variant=variant)


def test_worked_example_p3_on_gpu():
    """15 x 100 and one 160, k = {3,3,3} -> 104 -> 100 (hand-computed in tests/test_oracle_pins.py)."""
    x = np.full((1, 1, 16), 100, dtype=np.uint8)
    x[0, 0, 5] = 160
    for variant in (rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC):
        got, flags, counts, _ = run_gpu(x, [3.0, 3.0, 3.0], variant=variant)
        assert got[0, 0].tolist() == [100] * 16 and counts.tolist() == [1, 1, 0]
        got, _, counts, _ = run_gpu(x, [3.0], variant=variant)
        assert got[0, 0, 5] == 104


@pytest.mark.parametrize("ks", [[3.0], [2.75, 2.75], [3.25, 3.25, 3.25], [4.0] * 16, [1.5, 2.5, 3.5, 4.5]])
def test_heavy_rfi_rows(ks):
    """Rows where a large fraction is cut: bursts, steps, ramps (queue nearly full)."""
    S = 5000
    x = noisy((1, 12, S), seed=21)
    x[0, 0, 1000:1500] += 90
    x[0, 1, ::7] = 255
    x[0, 2, :] = (np.arange(S) % 256).astype(np.uint8)
    x[0, 3, : S // 3] = 0
    x[0, 4, 100:4900] = 200
    x[0, 5, :] = np.where(np.arange(S) % 50 < 3, 250, x[0, 5, :])
    for variant in (rfim.VARIANT_STAGED_1W, rfim.VARIANT_STAGED_2W, rfim.VARIANT_GENERIC):
        check(x, ks, variant=variant)


# ------------------------------------------------------------------ generic-only functionality
@pytest.mark.parametrize("window", [64, 256, 1000, 4096])
def test_windows_u8(window):
    x = noisy((2, 5, 4099), seed=31)
    x[0, 2, 100:130] = 240
    x[1, 4, 4090:] = 0
    name, _ = check(x, [4.0, 3.0], window=window)
    assert name == "td_u8_generic"


def test_median_policy_u8():
    """PAPER.md:110 median replacement.  Whole rows run in the staged kernel (lower median by counting passes over
    the staged row, taken at the first hit of an iteration, i.e. from the snapshot); windows in the generic one."""
    x = noisy((2, 6, 3000), seed=41)
    x[0, 1, 50:400] = 220                       # a long burst: the median (100) is far from the mean (114)
    x[1, 2, ::11] = 0
    x[1, 3, :] = 7                              # constant row
    x[1, 4, :1400] = 30; x[1, 4, 1400:] = 200   # bimodal: median on the lower mode, rank (3000 - 1) // 2 = 1499
    x[1, 5, 1000:1010] = 255
    name, counts = check(x, [3.0, 3.0], policy="median")
    assert name == "td_u8_staged_median" and counts[0] > 0
    name, _ = check(x, [1.0, 1.0, 1.0], policy="median", inplace=True)
    assert name == "td_u8_staged_median"
    name, _ = check(x, [3.0, 3.0], policy="median", variant=rfim.VARIANT_GENERIC)
    assert name == "td_u8_generic"
    name, _ = check(x, [4.0, 3.0], policy="median", window=500)
    assert name == "td_u8_generic"
    with pytest.raises(rfim.RfimError) as e:    # two warps per row: the snapshot median needs the one owner
        run_gpu(x, [3.0], policy="median", variant=rfim.VARIANT_STAGED_2W)
    assert e.value.status == -2


@pytest.mark.parametrize("S", [15, 16, 17, 100, 1023, 12500, 20001])
def test_median_policy_u8_lengths_and_ranks(S):
    """Odd and even lengths (rank (S - 1) // 2), every head / tail padding of the staged row (the padding copies of
    the first / last sample must not be counted), values at both ends of the byte range."""
    x = noisy((1, 9, S), seed=S)
    x[0, 0, :] = noisy((S,), S + 1, 3, 4)          # clipped at 0
    x[0, 1, :] = noisy((S,), S + 2, 252, 4)        # clipped at 255
    x[0, 2, : S // 2] = 0; x[0, 2, S // 2:] = 255  # the rank decides between 0 and 255
    x[0, 3, ::3] = 255
    x[0, 4, 0] = 255; x[0, 4, S - 1] = 0           # outliers in the first / last sample (the padding copies)
    x[0, 5, : S // 3] = 250
    for ks in ([3.0, 3.0], [1.0], [0.5, 2.0]):
        name, _ = check(x, ks, policy="median")
        assert name == "td_u8_staged_median"


def test_config2_median_two_beams():
    """BASELINE.json configs[1] data with the median policy: 2 beams, every element."""
    cfg = synth.config(2, beams=2)
    x = synth.fill_host(cfg, beam0=3, beams=2)
    name, counts = check(x, cfg["thresholds"], policy="median", inplace=True)
    assert name == "td_u8_staged_median" and all(int(c) > 0 for c in counts)


def test_long_rows_use_generic():
    x = noisy((1, 3, 300_000), seed=51)
    x[0, 1, 1000:3000] = 255
    name, _ = check(x, [5.0, 4.0, 3.0])
    assert name == "td_u8_generic"


def test_zero_thresholds_is_copy():
    x = noisy((2, 3, 100), seed=61)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.zeros_like(xd)
    flags = torch.ones_like(xd)
    rfim.rfim_time_sigma_cut(xd, [], out=out, flags=flags)
    torch.cuda.synchronize()
    assert torch.equal(out, xd) and int(flags.sum()) == 0


def test_many_rows_grid_wraps():
    """More rows than resident warps: the persistent loop and slot reuse (mbarrier phase, bulk groups)."""
    x = noisy((4, 3000, 257), seed=71)
    x[:, ::5, 100] = 255
    check(x, [4.0, 3.0], variant=rfim.VARIANT_STAGED_1W)
    check(x, [4.0, 3.0], variant=rfim.VARIANT_STAGED_2W)


def test_other_stream():
    x = noisy((1, 64, 2000), seed=81)
    x[0, :, 7] = 255
    xd = torch.from_numpy(x).to(DEV)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        rfim.rfim_time_sigma_cut(xd, [3.0], stream=s)
    s.synchronize()
    ref, _, _ = oracle.time_sigma_cut(x, [3.0])
    assert np.array_equal(xd.cpu().numpy(), ref)
