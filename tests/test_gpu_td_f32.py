"""GPU parity: rfim_time_sigma_cut (float32, windows, mean / median) through the C ABI vs the CPU oracle.

Tolerance (BASELINE.json north_star; reading R21): replaced values within 1e-5 relative;
a flag may differ from the oracle only where | |x - mu| - k sigma | < 1e-5 sigma.  A window that holds
such a borderline sample is "excused" (its later iterations legitimately diverge); excused windows
must stay below 1e-6 of all windows (at least one is tolerated in small cases).  Everything else --
kept samples, flags, counts -- must be identical.
"""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu

DEV = "cuda:0"


def run_gpu(x_np, ks, policy="median", window=0, variant=rfim.VARIANT_AUTO, inplace=False, pitch=None):
    B, C, S = x_np.shape
    if pitch is None:
        x = torch.from_numpy(x_np).to(DEV)
        out = None if inplace else torch.full_like(x, -7.0)
    else:
        buf = torch.full((B, C, pitch), 1234.5, dtype=torch.float32, device=DEV)
        buf[:, :, :S] = torch.from_numpy(x_np).to(DEV)
        x = buf[:, :, :S]
        obuf = torch.full((B, C, pitch), -7.0, dtype=torch.float32, device=DEV)
        out = None if inplace else obuf[:, :, :S]
    flags = torch.full((B, C, S), 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((max(1, len(ks)),), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_time_sigma_cut(x, ks, policy, out=out, window=window, flags=flags, counts=counts,
                                   variant=variant)
    torch.cuda.synchronize()
    name = rfim.rfim_last_variant()
    if pitch is not None:
        assert torch.all(buf[:, :, S:] == 1234.5)
        if not inplace:
            assert torch.all(obuf[:, :, S:] == -7.0)
    if not inplace:
        assert torch.equal(x.cpu(), torch.from_numpy(x_np)), "input modified by an out-of-place call"
    return res.cpu().numpy(), flags.cpu().numpy(), counts.cpu().numpy()[:len(ks)], name


def window_is_borderline(w, ks, policy="median"):
    """Re-derive one window in numpy float64: does any iteration hold a sample within 1e-5 sigma of the cut?"""
    x = w.astype(np.float64).copy()
    for k in ks:
        mu = x.mean()
        sg = x.std()
        dev = np.abs(x - mu)
        if np.any(np.abs(dev - k * sg) < 1e-5 * sg):
            return True
        f = dev > k * sg
        if f.any():
            x[f] = np.sort(x)[(x.size - 1) // 2] if policy == "median" else np.float64(np.float32(mu))
    return False


def compare(x_np, ks, got, gflags, gcounts, ref, rflags, rcounts, window, name, policy="median"):
    B, C, S = x_np.shape
    W = S if window == 0 or window > S else window
    nwin_total = B * C * ((S + W - 1) // W)
    close = np.isclose(got, ref, rtol=1e-5, atol=0.0) | (got == ref)
    bad = ~close | (gflags != rflags)
    excused = 0
    if bad.any():
        rows = np.argwhere(bad.any(axis=2))
        for (b, c) in rows:
            cols = np.nonzero(bad[b, c])[0]
            for w in sorted(set(int(i) // W for i in cols)):
                seg = x_np[b, c, w * W:min(S, (w + 1) * W)]
                assert window_is_borderline(seg, ks, policy), (
                    f"{name}: beam {b} channel {c} window {w}: GPU differs from the oracle without a borderline "
                    f"sample; first at {cols[:5]}, got {got[b, c, cols[:5]]}, ref {ref[b, c, cols[:5]]}")
                excused += 1
        assert excused <= max(1, int(1e-6 * nwin_total)), f"{name}: {excused} excused windows of {nwin_total}"
    if excused == 0 and gcounts is not None:
        assert gcounts.tolist() == [int(v) for v in rcounts], f"{name}: counts {gcounts} vs {rcounts}"
    # replaced samples of one window and iteration share one value; kept samples are untouched bit for bit
    kept = (gflags == 0) & (rflags == 0)
    assert np.array_equal(got[kept].view(np.uint32), x_np[kept].view(np.uint32)), f"{name}: a kept sample changed"
    return excused


def check(x_np, ks, policy="median", window=0, **kw):
    ref, rflags, rcounts = oracle.time_sigma_cut(
        x_np, ks, policy=oracle.MEDIAN if policy == "median" else oracle.MEAN, window=window)
    got, gflags, gcounts, name = run_gpu(x_np, ks, policy=policy, window=window, **kw)
    compare(x_np, ks, got, gflags, gcounts, ref, rflags, rcounts, window, name, policy)
    return name, rcounts


def gauss(shape, seed, mu=0.0, sigma=1.0):
    rng = np.random.default_rng(seed)
    return rng.normal(mu, sigma, shape).astype(np.float32)


# (config 5 at full size: tests/test_gpu_full_size.py)


@pytest.mark.parametrize("policy", ["mean", "median"])
@pytest.mark.parametrize("window", [0, 256, 1000])
def test_config5_shape_small(policy, window):
    cfg = synth.config(5, beams=1, channels=48)
    x = synth.fill_host(cfg)
    check(x, cfg["thresholds"], policy=policy, window=window)
    check(x, [3.25, 3.25, 3.25], policy=policy, window=window, inplace=True)


# ------------------------------------------------------------------------ shapes, tails, alignment
@pytest.mark.parametrize("S", [1, 2, 3, 5, 31, 33, 100, 255, 1000, 4099])
@pytest.mark.parametrize("window", [0, 1, 7, 32, 100])
@pytest.mark.parametrize("policy", ["mean", "median"])
def test_row_lengths_windows(S, window, policy):
    x = gauss((2, 9, S), seed=S * 131 + window)
    if S >= 16:
        x[0, 3, S // 2] = 40.0
        x[1, 5, : S // 8 + 1] += 9.0
        x[1, 7, 0] = -30.0
        x[1, 8, S - 1] = 1e6
        x[0, 0, :] = 0.25                # constant row
    check(x, [4.0, 3.0], policy=policy, window=window)


@pytest.mark.parametrize("variant", [rfim.VARIANT_AUTO, rfim.VARIANT_GENERIC])
@pytest.mark.parametrize("pitch", [1040, 1027])
@pytest.mark.parametrize("inplace", [False, True])
def test_padded_pitch_and_global_variant(variant, pitch, inplace):
    """pitch 1040: 16-byte aligned rows (TMA bulk path); 1027: rows at every 4-byte phase (plain loads)."""
    x = gauss((2, 7, 1000), seed=pitch)
    x[0, 2, 100:110] += 12.0
    name, _ = check(x, [4.0, 3.0], policy="median", window=256, variant=variant, pitch=pitch, inplace=inplace)
    assert name.startswith("td_f32_global" if variant == rfim.VARIANT_GENERIC else ("td_f32_staged", "td_f32_fast"))


@pytest.mark.parametrize("window,expect", [(0, "td_f32_global_w8"), (1024, "td_f32_staged_w1"),
                                           (16000, "td_f32_staged_w2"), (20000, "td_f32_staged_w4"),
                                           (50000, "td_f32_staged_w8")])
def test_rows_longer_than_shared_memory(window, expect):
    """S = 120001 floats = 480 KB per row: segments of whole windows; window = row falls back to global memory."""
    x = gauss((1, 3, 120001), seed=5)
    x[0, 1, 7000:7020] += 15.0
    x[0, 2, 119990:] -= 9.0
    name, _ = check(x, [4.0, 3.0], policy="median", window=window)
    assert name == expect


# ---------------------------------------------------------------------------------- value structure
@pytest.mark.parametrize("policy", ["mean", "median"])
def test_large_offset_and_scale(policy):
    """mu = 1e4 with sigma = 1 (pivoted statistics), and values of 1e-20 and 1e20."""
    x = gauss((1, 6, 5000), seed=11, mu=1.0e4, sigma=1.0)
    x[0, 1] = gauss((5000,), seed=12) * np.float32(1e-20)
    x[0, 2] = gauss((5000,), seed=13) * np.float32(1e20)
    x[0, 3, 17] = 1.0e4 + 50
    check(x, [4.0, 3.0, 3.0], policy=policy, window=0)
    check(x, [4.0, 3.0, 3.0], policy=policy, window=500)


@pytest.mark.parametrize("window", [0, 64, 999])
def test_median_with_heavy_ties_and_odd_distributions(window):
    """Quantised values (many equal samples), a bimodal row, a geometric cluster, half zeros: the median
    selection must split bins again / fall back to bisection and still return the exact lower median."""
    rng = np.random.default_rng(3)
    S = 6000
    x = np.zeros((1, 8, S), dtype=np.float32)
    x[0, 0] = np.rint(rng.normal(100, 12, S))                                     # integers stored as floats
    x[0, 1] = np.where(rng.random(S) < 0.5, rng.normal(-50, 1, S), rng.normal(80, 1, S))   # bimodal
    x[0, 2] = np.ldexp(1.0, -rng.integers(0, 120, S)).astype(np.float32)          # geometric cluster at 0
    x[0, 3] = np.where(rng.random(S) < 0.6, 0.0, rng.normal(0, 1, S))             # mostly exact zeros
    x[0, 4] = rng.standard_cauchy(S).astype(np.float32)                           # heavy tails
    x[0, 5] = np.where(rng.random(S) < 0.5, -0.0, 0.0); x[0, 5, ::97] = 5.0       # signed zeros
    x[0, 6] = np.rint(rng.normal(0, 2, S)) * np.float32(1e-42)                    # denormals
    x[0, 7] = rng.normal(0, 1, S); x[0, 7, ::50] += 25.0
    x = x.astype(np.float32)
    check(x, [4.0, 3.0, 2.0], policy="median", window=window)
    check(x, [1.5, 1.0], policy="median", window=window)


def test_p1_constant_and_p2_single_spike():
    """P1: constant rows untouched.  P2: (N-1) copies of c plus one spike are cut iff N > k^2 + 1."""
    x = np.full((1, 4, 300), 3.5, dtype=np.float32)
    got, gflags, gcounts, _ = run_gpu(x, [3.0], policy="mean")
    assert np.array_equal(got, x) and gflags.sum() == 0 and gcounts.tolist() == [0]
    for n, cut in ((9, False), (11, True), (12, True)):
        x = np.full((1, 1, n), 2.0, dtype=np.float32)
        x[0, 0, n // 2] = 1000.0
        got, gflags, gcounts, _ = run_gpu(x, [3.0], policy="median")
        assert bool(gflags.sum()) == cut
        if cut:
            assert got[0, 0, n // 2] == 2.0 and gcounts.tolist() == [1]


def test_iterations_equal_repeated_calls():
    """P9: {k,k,k} in one call equals three calls with {k}."""
    x = gauss((1, 16, 3000), seed=21)
    x[0, :, 100] += 10
    a, fa, ca, _ = run_gpu(x, [3.0, 3.0, 3.0], policy="median", window=500)
    y = x
    tot = []
    for _ in range(3):
        y, f, c, _ = run_gpu(y, [3.0], policy="median", window=500)
        tot.append(int(c[0]))
    assert np.array_equal(a, y) and ca.tolist() == tot


@pytest.mark.parametrize("policy", ["mean", "median"])
@pytest.mark.parametrize("window", [0, 256, 1000])
def test_huge_spike_at_the_first_sample_of_a_window(policy, window):
    """An RFI spike of 1e6 .. 1e8 sigma that lands on a window's FIRST sample (a broadband impulse on a window
    boundary does this to every channel at once).  The statistics must not be taken around that sample: with the
    pivot 1e8 sigma away, sigma^2 = B/n - (A/n)^2 cancels completely in the iterations after the spike is replaced.
    Three thresholds, so that two iterations run on statistics updated after the replacement."""
    S = 12500
    x = gauss((1, 24, S), seed=77)
    W = S if window == 0 else window
    amps = [1e6, 1e7, 1e8, -1e8, 3e7, 1e6]
    for c in range(24):
        a = np.float32(amps[c % len(amps)])
        x[0, c, 0] = a                                   # first sample of the row = first sample of window 0
        if W < S:
            x[0, c, W * (1 + c % 5)] = a                 # first sample of another window
            x[0, c, W * 7 + W // 2] = -a                 # and one in the middle of a window, for contrast
    check(x, [4.0, 3.0, 3.0], policy=policy, window=window)
    check(x, [5.0, 4.0, 3.0, 3.0], policy=policy, window=window, inplace=True)


@pytest.mark.parametrize("policy", ["mean", "median"])
@pytest.mark.parametrize("window", [0, 256, 1000])
def test_segment_kernel_forced(policy, window):
    """The tuned kernel (td_f32_fast.cuh) takes these requests in auto mode; variant 3 keeps the segment kernel
    (td_f32.cuh), which still serves rows longer than shared memory, windows that are not multiples of 4 samples
    and unaligned rows, under test on the same inputs."""
    cfg = synth.config(5, beams=1, channels=32)
    x = synth.fill_host(cfg)
    name, _ = check(x, cfg["thresholds"], policy=policy, window=window, variant=rfim.VARIANT_STAGED_1W)
    assert name.startswith("td_f32_staged")
    name, _ = check(x, cfg["thresholds"], policy=policy, window=window)
    assert name.startswith("td_f32_fast")


@pytest.mark.parametrize("window,team", [(4, 4), (64, 4), (256, 4), (260, 16), (1024, 16), (1028, 64), (4096, 64),
                                         (4100, 256), (12500, 256)])
def test_fast_kernel_team_sizes(window, team):
    """Every team size of the tuned kernel, windows at the edges of each range, a ragged last window."""
    x = gauss((1, 12, 12500), seed=window)
    x[0, 1, 5000:5040] += 9.0
    x[0, 2, ::1250] = 30.0
    x[0, 3, 12499] = -1e4
    for policy in ("mean", "median"):
        name, _ = check(x, [4.0, 3.0, 3.0], policy=policy, window=window)
        assert name == f"td_f32_fast_g{team}"
