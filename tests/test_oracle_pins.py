"""Pins for the CPU oracle (oracle/rfim_oracle.c) -- CPU only.

The paper prints no worked numeric example (PAPER.md has no table of outputs;
its figures are images), so the oracle is pinned against what the definition
(PAPER.md:100 TDSC, PAPER.md:102-108 FDSC) and the mathematics fix:

  P1  invariant      constant input is untouched
  P2  closed form    one spike among N-1 equal samples is cut iff N > k^2 + 1
  P3  worked example 15 x 100 + one 160, k = {3,3,3}  (hand-computed below)
  P4  hand array     {2,4,4,4,5,5,7,9}: mu = 5, sigma = 2
  P5  tie / rounding |x-mu| == k sigma is kept; mean 100.5 is replaced by 101
  P6  Samuelson      k >= sqrt(N-1) never flags
  P7  Chebyshev      #flagged < N / k^2
  P8  symmetries     shift, permutation, row independence
  P9  reductions     {k,k,k} == three calls; window == reshape; FD(1 bin) == TD on transpose
  P10 library        numpy mean/std/sort; exact rational brute force (fractions.Fraction)
  P11 idempotence    a fixed point stays fixed
  P12 monotone       flagged(k2) subset of flagged(k1) for k1 < k2
  F*  FDSC           hand-computed binned column; bin-wise constant column
  M*  median + bins  replacement = lower median of the flagged sample's own bin SNAPSHOT:
                     rational brute force with sorted(), hand-computed columns, numpy (f32)
  P13 behaviour      config 1: the 192 broadband-spike samples are cut by TDSC, the +60 channels by FDSC
Every expected value in this file is derived by hand or by exact rational
arithmetic in the test itself, never read back from the oracle.
"""
from fractions import Fraction

import numpy as np
import pytest
from hypothesis import given, settings, strategies as st

import oracle

K316 = 2 ** 16


def td(x, ks, **kw):
    a = np.asarray(x)
    if a.ndim == 1:
        a = a[None, None, :]
    out, flags, counts = oracle.time_sigma_cut(a, ks, **kw)
    return out, flags, counts


def fd(x, ks, **kw):
    a = np.asarray(x)
    if a.ndim == 1:  # a single column: channels along the given axis
        a = a[None, :, None]
    return oracle.freq_sigma_cut(a, ks, **kw)


# ---------------------------------------------------------------- brute force
def brute_td_iteration(x, k):
    """One TDSC iteration in exact rationals, straight from PAPER.md:100:
    |x - mu| > k sigma with population sigma; decided as (x-mu)^2 > k^2 sigma^2.
    k is the rational p/2^16 (reading R17).  Returns (new list, flags)."""
    n = len(x)
    kq = Fraction(int(round(k * K316)), K316)  # exact for the k used here
    mu = Fraction(sum(x), n)
    var = Fraction(sum(v * v for v in x), n) - mu * mu
    flags = [(Fraction(v) - mu) ** 2 > kq * kq * var for v in x]
    r = (2 * sum(x) + n) // (2 * n)  # round half up (reading R6)
    return [r if f else v for v, f in zip(x, flags)], flags


def brute_fd_iteration(col, k, nb, policy="mean"):
    """One FDSC iteration on a column in exact rationals.  policy "median": a flagged
    sample is replaced by the lower median (rank (nb-1)//2 of sorted()) of ITS bin's snapshot, i.e. of the
    bin's values at the start of the iteration ("mean of its respective bin" + PAPER.md:110)."""
    C = len(col)
    kq = Fraction(int(round(k * K316)), K316)
    means = [Fraction(sum(col[b:b + nb]), nb) for b in range(0, C, nb)]
    d = [Fraction(col[c]) - means[c // nb] for c in range(C)]
    mu = sum(d) / C
    var = sum((v - mu) ** 2 for v in d) / C
    flags = [(v - mu) ** 2 > kq * kq * var for v in d]
    if policy == "median":
        rep = [sorted(col[b:b + nb])[(nb - 1) // 2] for b in range(0, C, nb)]
    else:
        rep = [(2 * sum(col[b:b + nb]) + nb) // (2 * nb) for b in range(0, C, nb)]
    return [rep[c // nb] if flags[c] else col[c] for c in range(C)], flags


# ------------------------------------------------------------------------ P1
@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
@pytest.mark.parametrize("k", [0.5, 1.0, 3.0, 5.0])
def test_p1_constant_untouched(dtype, k):
    x = np.full((2, 3, 50), 77, dtype=dtype)
    for fn in (oracle.time_sigma_cut, oracle.freq_sigma_cut):
        out, flags, counts = fn(x, [k, k])
        assert np.array_equal(out, x)
        assert flags.sum() == 0 and counts.sum() == 0


# ------------------------------------------------------------------------ P2
@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
@pytest.mark.parametrize("n,k,cut", [(10, 3.0, False), (11, 3.0, True), (17, 4.0, False), (18, 4.0, True),
                                      (5, 2.0, False), (6, 2.0, True), (26, 5.0, False), (27, 5.0, True)])
@pytest.mark.parametrize("c,amp", [(100, 60), (100, -90), (3, 200), (7, 1)])
def test_p2_single_spike_closed_form(dtype, n, k, cut, c, amp):
    """(N-1) samples equal to c and one equal to c+A: mu = c + A/N, sigma = |A| sqrt(N-1)/N,
    spike deviation = |A|(N-1)/N, so the spike is cut iff sqrt(N-1) > k iff N > k^2+1,
    for any A and c; for k >= 1 nothing else is ever cut.  N = k^2+1 is exact equality and
    pins the strict '>' of PAPER.md:100."""
    if dtype == np.float32 and n == int(k * k) + 1:
        pytest.skip("equality case is not exactly representable in floating point")
    x = np.full(n, c, dtype=dtype)
    pos = n // 3
    x[pos] = c + amp
    out, flags, counts = td(x, [k])
    expect_flags = np.zeros(n, dtype=np.uint8)
    expect = x.copy()
    if cut:
        expect_flags[pos] = 1
        if dtype == np.uint8:
            s = int(x.astype(np.int64).sum())
            expect[pos] = (2 * s + n) // (2 * n)
        else:
            expect[pos] = np.float32(np.float64(x.astype(np.float64).sum()) / n)
    assert np.array_equal(flags[0, 0], expect_flags)
    assert int(counts[0]) == int(cut)
    if dtype == np.uint8:
        assert np.array_equal(out[0, 0], expect)
    else:
        np.testing.assert_allclose(out[0, 0], expect, rtol=1e-6)


# ------------------------------------------------------------------------ P3
def test_p3_worked_example_three_iterations():
    """15 x 100 and one 160, k = {3,3,3}, worked by hand:
    it 1: S=1660, mu=103.75, N^2 var = 16*175600-1660^2 = 54000 (var = 3375/16, sigma=14.52);
          spike dev 56.25 > 43.57 -> cut, r = floor((3320+16)/32) = 104; others dev 3.75 keep.
    it 2: S=1604, mu=100.25, var = 15/16 (sigma=0.968); the 104 deviates 3.75 > 2.905 -> cut again,
          r = floor((3208+16)/32) = 100; the 100s deviate 0.25, keep.
    it 3: all 100, sigma = 0, nothing.
    Pins: the replacement mean includes the outlier (R5), round half up (R6), statistics are
    refreshed between iterations (R7), count semantics (R8)."""
    x = np.full(16, 100, dtype=np.uint8)
    x[5] = 160
    out1, _, c1 = td(x, [3.0])
    assert out1[0, 0, 5] == 104 and c1.tolist() == [1]
    out2, _, c2 = td(x, [3.0, 3.0])
    assert out2[0, 0, 5] == 100 and c2.tolist() == [1, 1]
    out3, flags3, c3 = td(x, [3.0, 3.0, 3.0])
    assert np.array_equal(out3[0, 0], np.full(16, 100, dtype=np.uint8))
    assert c3.tolist() == [1, 1, 0]
    assert flags3[0, 0].tolist() == [0] * 5 + [1] + [0] * 10
    # the same statistics, from the oracle's exposed helper
    s, q = oracle.stats_u8(x)
    assert (s, q) == (1660, 175600)


# ------------------------------------------------------------------------ P4
def test_p4_hand_array():
    """{2,4,4,4,5,5,7,9}: S=40, Q=232, mu=5, sigma^2 = 232/8-25 = 4, sigma=2.
    k=2: the 9 is exactly 2 sigma away -> kept (strict).  k=1.5 (cut at 3.0): the 9 (dev 4) is
    cut and becomes the mean 5; the 2 (dev exactly 3) is kept."""
    x = np.array([2, 4, 4, 4, 5, 5, 7, 9], dtype=np.uint8)
    assert oracle.stats_u8(x) == (40, 232)
    out, flags, counts = td(x, [2.0])
    assert np.array_equal(out[0, 0], x) and counts.tolist() == [0]
    out, flags, counts = td(x, [1.5])
    assert out[0, 0].tolist() == [2, 4, 4, 4, 5, 5, 7, 5]
    assert flags[0, 0].tolist() == [0, 0, 0, 0, 0, 0, 0, 1] and counts.tolist() == [1]
    # float32 path, same array: mean 5, sigma 2 exactly representable
    xf = x.astype(np.float32)
    m, sg = oracle.stats_f32(xf)
    assert m == 5.0 and sg == 2.0
    out, flags, counts = td(xf, [1.5])
    assert out[0, 0].tolist() == [2, 4, 4, 4, 5, 5, 7, 5] and counts.tolist() == [1]
    out, flags, counts = td(xf, [2.0])
    assert counts.tolist() == [0]


# ------------------------------------------------------------------------ P5
def test_p5_ties_and_rounding():
    x = np.array([10] * 4 + [20] * 4, dtype=np.uint8)  # mu 15, sigma 5: every sample exactly 1 sigma away
    out, flags, counts = td(x, [1.0])
    assert np.array_equal(out[0, 0], x) and counts.tolist() == [0]
    # just below 1 sigma everything is cut, and replaced by the mean 15
    out, flags, counts = td(x, [1.0 - 2.0 ** -16])
    assert out[0, 0].tolist() == [15] * 8 and counts.tolist() == [8]
    # 19 x 100 and one 110: S = 2010, mu = 100.5 -> replacement 101 (half up)
    y = np.array([100] * 19 + [110], dtype=np.uint8)
    out, flags, counts = td(y, [3.0])
    assert out[0, 0, 19] == 101 and counts.tolist() == [1]
    assert out[0, 0, :19].tolist() == [100] * 19
    # 19 x 100 and one 109: mu = 100.45 -> 100 (round down); one 111: mu = 100.55 -> 101
    y[19] = 109
    assert td(y, [3.0])[0][0, 0, 19] == 100
    y[19] = 111
    assert td(y, [3.0])[0][0, 0, 19] == 101


def test_threshold_quantisation():
    """R17: p = round-half-even(k 2^16); exact for every threshold the paper uses
    (2.75, 3.25, 4.00: PAPER.md:126,140,144) and the configs' 3, 4, 5."""
    for k in (2.75, 3.0, 3.25, 4.0, 5.0, 1.5):
        assert oracle.quantise_threshold(k) == int(k * K316)
    assert oracle.quantise_threshold(2.0 ** -17) == 0            # half -> even (0)
    assert oracle.quantise_threshold(3 * 2.0 ** -17) == 2        # 1.5 -> 2
    assert oracle.quantise_threshold(5 * 2.0 ** -17) == 2        # 2.5 -> 2
    assert oracle.quantise_threshold(1.0 + 2.0 ** -18) == K316   # rounds to nearest


# --------------------------------------------------------------------- P6, P7
@settings(max_examples=150, deadline=None)
@given(st.lists(st.integers(0, 255), min_size=2, max_size=60), st.sampled_from([1.0, 1.5, 2.0, 3.0, 4.0]))
def test_p6_p7_samuelson_chebyshev(vals, k):
    x = np.array(vals, dtype=np.uint8)
    n = len(vals)
    out, flags, counts = td(x, [k])
    nflag = int(counts[0])
    if k >= np.sqrt(n - 1):          # Samuelson: max |x-mu| <= sigma sqrt(N-1)
        assert nflag == 0
    if nflag:
        assert nflag * k * k < n      # Chebyshev, strict
    # same bounds along the channel axis
    out, flags, counts = fd(x, [k])
    nflag = int(counts[0])
    if k >= np.sqrt(n - 1):
        assert nflag == 0
    if nflag:
        assert nflag * k * k < n


# ------------------------------------------------------------------------ P10
@settings(max_examples=300, deadline=None)
@given(st.lists(st.integers(0, 255), min_size=1, max_size=40),
       st.lists(st.sampled_from([0.75, 1.0, 1.25, 1.5, 2.0, 2.75, 3.0, 3.25]), min_size=1, max_size=3))
def test_p10_td_u8_vs_exact_rationals(vals, ks):
    x = np.array(vals, dtype=np.uint8)
    out, flags, counts = td(x, ks)
    cur = list(vals)
    anyflag = [False] * len(vals)
    exp_counts = []
    for k in ks:
        cur, fl = brute_td_iteration(cur, k)
        anyflag = [a or f for a, f in zip(anyflag, fl)]
        exp_counts.append(sum(fl))
    assert out[0, 0].tolist() == cur
    assert flags[0, 0].tolist() == [int(f) for f in anyflag]
    assert counts.tolist() == exp_counts


@settings(max_examples=200, deadline=None)
@given(st.integers(1, 6), st.sampled_from([1, 2, 4, 8]), st.data(),
       st.lists(st.sampled_from([0.75, 1.0, 1.5, 2.0, 2.75]), min_size=1, max_size=2))
def test_p10_fd_u8_vs_exact_rationals(nbins, nb, data, ks):
    C = nbins * nb
    vals = data.draw(st.lists(st.integers(0, 255), min_size=C, max_size=C))
    x = np.array(vals, dtype=np.uint8)
    out, flags, counts = fd(x, ks, bin_size=nb)
    cur = list(vals)
    anyflag = [False] * C
    exp_counts = []
    for k in ks:
        cur, fl = brute_fd_iteration(cur, k, nb)
        anyflag = [a or f for a, f in zip(anyflag, fl)]
        exp_counts.append(sum(fl))
    assert out[0, :, 0].tolist() == cur
    assert flags[0, :, 0].tolist() == [int(f) for f in anyflag]
    assert counts.tolist() == exp_counts


@settings(max_examples=300, deadline=None)
@given(st.integers(1, 6), st.sampled_from([1, 2, 3, 4, 5, 8]), st.data(),
       st.lists(st.sampled_from([0.75, 1.0, 1.5, 2.0, 2.75]), min_size=1, max_size=3))
def test_m1_fd_u8_median_with_bins_vs_exact_rationals(nbins, nb, data, ks):
    """The median-with-bins branch of fdsc_iter_u8 (policy MEDIAN, bin_size < channels) against the brute
    force: flags from exact rationals, replacement = sorted(bin snapshot)[(nb-1)//2].  A wrong bin offset, a
    median taken after an earlier bin of the same iteration was modified, or an upper median fails here."""
    C = nbins * nb
    vals = data.draw(st.lists(st.integers(0, 255), min_size=C, max_size=C))
    x = np.array(vals, dtype=np.uint8)
    out, flags, counts = fd(x, ks, bin_size=nb, policy=oracle.MEDIAN)
    cur = list(vals)
    anyflag = [False] * C
    exp_counts = []
    for k in ks:
        cur, fl = brute_fd_iteration(cur, k, nb, policy="median")
        anyflag = [a or f for a, f in zip(anyflag, fl)]
        exp_counts.append(sum(fl))
    assert out[0, :, 0].tolist() == cur
    assert flags[0, :, 0].tolist() == [int(f) for f in anyflag]
    assert counts.tolist() == exp_counts


@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_m2_fd_median_with_bins_hand_computed(dtype):
    """C = 8, bins of 4, column {1,2,3,40, 9,9,9,9}, k = 1.5, worked by hand.
    Bin means 11.5 and 9; corrected {-10.5,-9.5,-8.5,28.5, 0,0,0,0}; their mean is 0 and
    sigma'^2 = (110.25+90.25+72.25+812.25)/8 = 135.625, sigma' = 11.646, cut = 17.47: only the 40 is cut.
    MEDIAN: sorted bin {1,2,3,40}, rank (4-1)//2 = 1 -> 2 (the LOWER median; the upper would be 3, the bin
    mean 11.5 -> 12, the other bin's median 9, the whole column's lower median 9).
    Second iteration (k = 1.5 again) on {1,2,3,2, 9,9,9,9}: bin means 2 and 9; corrected {-1,0,1,0,0,0,0,0};
    sigma'^2 = 2/8, cut = 0.75: the 1 and the 3 are cut (dev 1) and replaced by the median of the snapshot
    {1,2,3,2}: sorted {1,2,2,3}[1] = 2 -> {2,2,2,2, 9,9,9,9}; counts {1, 2}."""
    col = np.array([1, 2, 3, 40, 9, 9, 9, 9], dtype=dtype)
    out, flags, counts = fd(col, [1.5], bin_size=4, policy=oracle.MEDIAN)
    assert out[0, :, 0].tolist() == [1, 2, 3, 2, 9, 9, 9, 9]
    assert flags[0, :, 0].tolist() == [0, 0, 0, 1, 0, 0, 0, 0] and counts.tolist() == [1]
    out, flags, counts = fd(col, [1.5, 1.5], bin_size=4, policy=oracle.MEDIAN)
    assert out[0, :, 0].tolist() == [2, 2, 2, 2, 9, 9, 9, 9]
    assert flags[0, :, 0].tolist() == [1, 0, 1, 1, 0, 0, 0, 0] and counts.tolist() == [1, 2]
    # the mean policy on the same column: 40 -> round-half-up(11.5) = 12 (u8), 11.5 (f32)
    out, _, _ = fd(col, [1.5], bin_size=4, policy=oracle.MEAN)
    assert out[0, :, 0].tolist() == [1, 2, 3, 12 if dtype == np.uint8 else 11.5, 9, 9, 9, 9]
    # flagged samples in BOTH bins of one iteration: each takes the median of its OWN bin's snapshot.
    # {10,10,10,90, 50,50,52,120}, k = 1.5: bin means 30 and 68; corrected {-20,-20,-20,60,-18,-18,-16,52};
    # sigma'^2 = (3*400+3600+324+324+256+2704)/8 = 1051, cut = 48.63: the 90 and the 120 are cut;
    # medians: sorted {10,10,10,90}[1] = 10, sorted {50,50,52,120}[1] = 50.
    col2 = np.array([10, 10, 10, 90, 50, 50, 52, 120], dtype=dtype)
    out, flags, counts = fd(col2, [1.5], bin_size=4, policy=oracle.MEDIAN)
    assert out[0, :, 0].tolist() == [10, 10, 10, 10, 50, 50, 52, 50]
    assert flags[0, :, 0].tolist() == [0, 0, 0, 1, 0, 0, 0, 1] and counts.tolist() == [2]


@pytest.mark.parametrize("policy", [oracle.MEAN, oracle.MEDIAN])
@pytest.mark.parametrize("nb", [4, 8, 32])
def test_m3_fd_f32_bins_vs_numpy(policy, nb):
    """f32 FDSC with bins against numpy: bin means, np.std(ddof=0) of the mean-corrected values, np.sort per bin.
    Samples closer than 1e-9 sigma to the cut are excluded (summation order)."""
    rng = np.random.default_rng(11)
    B, C, S = 2, 64, 40
    x = rng.normal(0.0, 1.0, (B, C, S)).astype(np.float32)
    x += np.repeat(rng.normal(0.0, 5.0, (B, C // nb, 1)), nb, axis=1).astype(np.float32)   # a bandpass shape
    x[0, 13, :] += 7.0
    x[1, 40, 5:25] -= 6.0
    out, flags, counts = oracle.freq_sigma_cut(x, [2.75], policy=policy, bin_size=nb)
    x64 = x.astype(np.float64).reshape(B, C // nb, nb, S)
    m = x64.mean(axis=2, keepdims=True)
    d = (x64 - m).reshape(B, C, S)
    mu = d.mean(axis=1, keepdims=True)
    sg = d.std(axis=1, ddof=0, keepdims=True)
    dev = np.abs(d - mu)
    safe = np.abs(dev - 2.75 * sg) > 1e-9 * sg
    exp_flags = dev > 2.75 * sg
    assert exp_flags.sum() > 40
    assert np.array_equal(flags.astype(bool)[safe], exp_flags[safe])
    if policy == oracle.MEAN:
        rep = np.broadcast_to(m.astype(np.float32), x64.shape).reshape(B, C, S)
    else:
        srt = np.sort(x.reshape(B, C // nb, nb, S), axis=2)[:, :, (nb - 1) // 2, :]
        rep = np.repeat(srt, nb, axis=1)
    expect = np.where(flags.astype(bool), rep, x)
    if policy == oracle.MEDIAN:
        assert np.array_equal(out, expect)               # an element of the bin: exact
    else:
        np.testing.assert_allclose(out, expect, rtol=1e-6, atol=1e-6)
    assert int(counts[0]) == int(flags.sum())


def test_p10_f32_statistics_vs_numpy():
    rng = np.random.default_rng(1)
    for n in (1, 2, 7, 256, 12500):
        x = rng.normal(3.0, 2.0, n).astype(np.float32)
        m, sg = oracle.stats_f32(x)
        x64 = x.astype(np.float64)
        assert m == pytest.approx(np.mean(x64), rel=1e-13, abs=1e-13)
        assert sg == pytest.approx(np.std(x64, ddof=0), rel=1e-12, abs=1e-13)
    x = rng.integers(0, 256, 5000).astype(np.uint8)
    s, q = oracle.stats_u8(x)
    assert s == int(x.astype(np.int64).sum()) and q == int((x.astype(np.int64) ** 2).sum())


def test_p10_f32_flags_and_median_vs_numpy():
    """f32: statistics via numpy.mean / numpy.std(ddof=0) in float64, median via numpy.sort.
    Samples closer than 1e-9 sigma to the cut are excluded (summation order)."""
    rng = np.random.default_rng(2)
    x = rng.normal(0.0, 1.0, (2, 3, 1000)).astype(np.float32)
    x[0, 1, 17] = 9.0
    x[1, 2, 400:420] += 6.0
    for policy in (oracle.MEAN, oracle.MEDIAN):
        out, flags, counts = oracle.time_sigma_cut(x, [3.0], policy=policy)
        x64 = x.astype(np.float64)
        mu = x64.mean(axis=2, keepdims=True)
        sg = x64.std(axis=2, ddof=0, keepdims=True)
        dev = np.abs(x64 - mu)
        safe = np.abs(dev - 3.0 * sg) > 1e-9 * sg
        exp_flags = dev > 3.0 * sg
        assert np.array_equal(flags.astype(bool)[safe], exp_flags[safe])
        assert exp_flags.sum() > 20
        if policy == oracle.MEAN:
            rep = np.broadcast_to(mu.astype(np.float32), x.shape)
        else:
            srt = np.sort(x, axis=2)
            rep = np.broadcast_to(srt[:, :, (x.shape[2] - 1) // 2][:, :, None], x.shape)
        expect = np.where(flags.astype(bool), rep, x)
        if policy == oracle.MEDIAN:
            assert np.array_equal(out, expect)           # the median is an element: exact
        else:
            np.testing.assert_allclose(out, expect, rtol=1e-6, atol=1e-7)


def test_median_u8_policy():
    """R12/R13: the test still uses mean and sigma; only the replacement is the lower median.
    {1,1,2,2,3,3,50}: mu = 62/7, the 50 is cut at k=2; ascending rank (7-1)//2 = 3 -> 2.
    Even count {1,2,3,4,5,100}: rank (6-1)//2 = 2 -> 3 (lower of 3 and 4)."""
    x = np.array([3, 1, 50, 2, 1, 3, 2], dtype=np.uint8)
    out, flags, counts = td(x, [2.0], policy=oracle.MEDIAN)
    assert out[0, 0].tolist() == [3, 1, 2, 2, 1, 3, 2] and counts.tolist() == [1]
    y = np.array([5, 100, 1, 4, 2, 3], dtype=np.uint8)
    out, flags, counts = td(y, [2.0], policy=oracle.MEDIAN)
    assert out[0, 0].tolist() == [5, 3, 1, 4, 2, 3] and counts.tolist() == [1]


# ------------------------------------------------------------------------ P8
def test_p8_symmetries():
    rng = np.random.default_rng(3)
    x = np.clip(np.rint(rng.normal(100, 10, (2, 4, 300))), 0, 255).astype(np.uint8)
    x[0, 1, 50:60] = 200
    x[1, 3, 7] = 0
    ks = [4.0, 3.0]
    out, flags, counts = oracle.time_sigma_cut(x, ks)
    assert counts.sum() > 10
    # shift by a constant (no clipping: values stay inside 0..255)
    assert x.max() <= 235
    out_s, flags_s, _ = oracle.time_sigma_cut((x + 20).astype(np.uint8), ks)
    assert np.array_equal(flags_s, flags) and np.array_equal(out_s, out + 20)
    # permutation of the samples of every row
    perm = rng.permutation(x.shape[2])
    out_p, flags_p, _ = oracle.time_sigma_cut(np.ascontiguousarray(x[:, :, perm]), ks)
    assert np.array_equal(out_p, out[:, :, perm]) and np.array_equal(flags_p, flags[:, :, perm])
    # rows do not influence each other
    y = x.copy()
    y[1, 2] = 255 - y[1, 2]
    out_y, _, _ = oracle.time_sigma_cut(y, ks)
    keep = np.ones((2, 4), dtype=bool)
    keep[1, 2] = False
    assert np.array_equal(out_y[keep], out[keep])
    # FDSC: columns do not influence each other, permuting channels permutes the result
    out_f, flags_f, _ = oracle.freq_sigma_cut(x, ks)
    permc = rng.permutation(x.shape[1])
    out_fp, flags_fp, _ = oracle.freq_sigma_cut(np.ascontiguousarray(x[:, permc, :]), ks)
    assert np.array_equal(out_fp, out_f[:, permc, :])


# ------------------------------------------------------------------------ P9
def test_p9_iterations_equal_repeated_calls():
    rng = np.random.default_rng(4)
    x = np.clip(np.rint(rng.normal(100, 12, (1, 40, 300))), 0, 255).astype(np.uint8)
    x[0, :, 100] = 250            # broadband impulse (TDSC's target)
    x[0, 2, 200:260] = 180        # narrow-band burst (FDSC's target; 40 channels > 3.25^2+1, Samuelson)
    for fn in (oracle.time_sigma_cut, oracle.freq_sigma_cut):
        out3, flags3, counts3 = fn(x, [3.25, 3.25, 3.25])   # PAPER.md:178 "three iterations with 3.25 sigma"
        cur = x
        fl = np.zeros_like(flags3)
        cs = []
        for _ in range(3):
            cur, f1, c1 = fn(cur, [3.25])
            fl |= f1
            cs.append(int(c1[0]))
        assert np.array_equal(out3, cur) and np.array_equal(flags3, fl) and counts3.tolist() == cs
        assert cs[0] > 0


@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
def test_p9_window_equals_reshape(dtype):
    rng = np.random.default_rng(5)
    x = np.clip(np.rint(rng.normal(100, 12, (2, 3, 512))), 0, 255).astype(dtype)
    x[1, 1, 300] = 255
    x[0, 2, 10:20] = 190
    for W in (64, 128, 512):
        out_w, flags_w, counts_w = oracle.time_sigma_cut(x, [4.0, 3.0], window=W)
        xr = np.ascontiguousarray(x.reshape(2, 3 * 512 // W, W))
        out_r, flags_r, counts_r = oracle.time_sigma_cut(xr, [4.0, 3.0])
        assert np.array_equal(out_w.reshape(xr.shape), out_r)
        assert np.array_equal(flags_w.reshape(xr.shape), flags_r)
        assert counts_w.tolist() == counts_r.tolist()
    # ragged tail: 500 = 3*128 + 116 -> the tail is its own window (R11)
    y = np.ascontiguousarray(x[:, :, :500])
    out_t, _, _ = oracle.time_sigma_cut(y, [3.0], window=128)
    for w0 in (0, 128, 256, 384):
        seg = np.ascontiguousarray(y[:, :, w0:w0 + 128])
        assert np.array_equal(out_t[:, :, w0:w0 + 128], oracle.time_sigma_cut(seg, [3.0])[0])


@pytest.mark.parametrize("dtype", [np.uint8, np.float32])
@pytest.mark.parametrize("policy", [oracle.MEAN, oracle.MEDIAN])
def test_p9_fd_single_bin_equals_td_on_transpose(dtype, policy):
    """The FDSC loop (gather column, bins, corrected statistics) and the TDSC loop are written
    independently in the oracle; with one bin they must agree on the transposed beam."""
    rng = np.random.default_rng(6)
    x = np.clip(np.rint(rng.normal(100, 12, (2, 48, 70))), 0, 255).astype(dtype)
    x[:, 7, :] += 60
    x[1, 40, 20:30] += 80
    ks = [4.0, 3.0]
    out_f, flags_f, counts_f = oracle.freq_sigma_cut(x, ks, policy=policy)
    xt = np.ascontiguousarray(x.transpose(0, 2, 1))
    out_t, flags_t, counts_t = oracle.time_sigma_cut(xt, ks, policy=policy)
    if dtype == np.uint8 or policy == oracle.MEDIAN:
        assert np.array_equal(out_f, out_t.transpose(0, 2, 1))
    else:
        np.testing.assert_allclose(out_f, out_t.transpose(0, 2, 1), rtol=1e-6)
    assert np.array_equal(flags_f, flags_t.transpose(0, 2, 1))
    assert counts_f.tolist() == counts_t.tolist() and counts_f[0] > 0


# ----------------------------------------------------------------------- P11
def test_p11_idempotent_at_fixed_point():
    rng = np.random.default_rng(7)
    x = np.clip(np.rint(rng.normal(100, 12, (1, 6, 800))), 0, 255).astype(np.uint8)
    x[0, :, 300:303] = 240
    cur = x
    for _ in range(50):                       # iterate k=3 to a fixed point
        nxt, _, c = oracle.time_sigma_cut(cur, [3.0])
        if c[0] == 0:
            break
        cur = nxt
    assert c[0] == 0
    again, flags, counts = oracle.time_sigma_cut(cur, [3.0, 3.0])
    assert np.array_equal(again, cur) and flags.sum() == 0 and counts.sum() == 0


# ----------------------------------------------------------------------- P12
def test_p12_monotone_in_k():
    rng = np.random.default_rng(8)
    x = np.clip(np.rint(rng.normal(100, 12, (1, 4, 2000))), 0, 255).astype(np.uint8)
    prev = None
    for k in (5.0, 4.0, 3.25, 3.0, 2.75, 2.0):
        _, flags, _ = oracle.time_sigma_cut(x, [k])
        if prev is not None:
            assert np.all(flags >= prev)      # smaller k flags a superset
        prev = flags
    assert prev.sum() > 0


# ------------------------------------------------------------------------ F*
def test_fdsc_hand_computed_bins():
    """C = 8, bins of 4 (PAPER.md:102 step 1).  Column {10,10,10,10, 50,50,50,90}:
    bin means 10 and 60; corrected {0,0,0,0,-10,-10,-10,30}; their mean is 0 and
    sigma'^2 = (3*100 + 900)/8 = 150, sigma' = 12.247.  k = 2 (cut 24.49): only the 90 is cut and
    the ORIGINAL value is replaced by ITS bin's mean, 60.
    With a single bin instead: mu = 35, sigma^2 = 775, sigma = 27.84, cut 55.68: the 90 (dev 55) stays."""
    col = np.array([10, 10, 10, 10, 50, 50, 50, 90], dtype=np.uint8)
    out, flags, counts = fd(col, [2.0], bin_size=4)
    assert out[0, :, 0].tolist() == [10, 10, 10, 10, 50, 50, 50, 60]
    assert flags[0, :, 0].tolist() == [0] * 7 + [1] and counts.tolist() == [1]
    out, flags, counts = fd(col, [2.0], bin_size=0)
    assert np.array_equal(out[0, :, 0], col) and counts.tolist() == [0]
    out, flags, counts = fd(col, [2.0], bin_size=8)
    assert np.array_equal(out[0, :, 0], col)
    # float32, same numbers
    out, flags, counts = fd(col.astype(np.float32), [2.0], bin_size=4)
    assert out[0, :, 0].tolist() == [10, 10, 10, 10, 50, 50, 50, 60] and counts.tolist() == [1]


def test_fdsc_binwise_constant_column_untouched():
    """If every bin is constant (a pure bandpass shape) all corrected values are 0, sigma' = 0 and
    nothing is cut, although without step 1 the levels differ by far more than k sigma."""
    col = np.repeat(np.array([10, 200, 10, 10, 10, 10, 10, 10], dtype=np.uint8), 4)
    out, flags, counts = fd(col, [1.0], bin_size=4)
    assert np.array_equal(out[0, :, 0], col) and counts.sum() == 0
    out, flags, counts = fd(col, [1.0], bin_size=0)      # single bin: the 200s are 2.6 sigma out
    assert counts[0] == 4 and set(out[0, :, 0].tolist()) == {10, 34}   # mean = (28*10+4*200)/32 = 33.75 -> 34


def test_fdsc_touches_only_its_column_and_td_only_its_row():
    x = np.full((1, 16, 16), 100, dtype=np.uint8)
    x[0, 3, :] = 160                     # a narrow-band channel: constant in time
    out_t, _, ct = oracle.time_sigma_cut(x, [3.0])
    assert np.array_equal(out_t, x)      # TDSC cannot see a constant offset
    out_f, flags_f, cf = oracle.freq_sigma_cut(x, [3.0])
    assert cf[0] == 16 and np.all(flags_f[0, 3, :] == 1) and flags_f.sum() == 16
    assert np.all(out_f[0, 3, :] == 104)  # column mean (15*100+160)/16 = 103.75 -> 104
    y = np.full((1, 16, 16), 100, dtype=np.uint8)
    y[0, :, 5] = 160                     # a broadband impulse: constant in frequency
    out_f, _, cf = oracle.freq_sigma_cut(y, [3.0])
    assert np.array_equal(out_f, y)      # FDSC does not affect broadband signal
    out_t, flags_t, ct = oracle.time_sigma_cut(y, [3.0])
    assert ct[0] == 16 and np.all(out_t[0, :, 5] == 104)


# ----------------------------------------------------------------------- P13
def test_p13_config1_behaviour():
    """SURVEY.md 8c P13 on the seeded config-1 input (BASELINE.json configs[0]): every one of the 3 x 64 = 192
    broadband-spike samples (+80 = 8 sigma) is cut by TDSC at k = 3; the +60 channels 7 and 40 are NOT cleaned by
    TDSC (a constant offset only moves the row mean) but are outliers across channels for FDSC."""
    from paper_2001_03389_b200 import synth
    cfg = synth.config(1)
    x = synth.fill_host(cfg)
    d = synth.Descriptor(cfg)
    spikes = np.nonzero(d.imp_amp[0])[0]
    assert len(spikes) == 3
    out, flags, counts = oracle.time_sigma_cut(x, cfg["thresholds"])
    assert flags[0][:, spikes].sum() == 64 * 3
    assert abs(out[0, 7].astype(np.float64).mean() - 160) < 2 and abs(out[0, 40].astype(np.float64).mean() - 160) < 2
    assert flags[0, 7].sum() <= 3 + 8 and flags[0, 40].sum() <= 3 + 8     # the spikes plus at most a few tail samples
    _, fflags, _ = oracle.freq_sigma_cut(x, [3.0])
    assert fflags[0, 7].mean() > 0.9 and fflags[0, 40].mean() > 0.9
    others = np.ones(64, dtype=bool)
    others[[7, 40]] = False
    assert fflags[0, others].mean() < 0.02


# --------------------------------------------------------------- ABI details
def test_out_of_place_stride_and_errors():
    import ctypes
    rng = np.random.default_rng(9)
    B, C, S, P = 2, 3, 37, 48
    buf = np.zeros((B, C, P), dtype=np.uint8)
    x = np.clip(np.rint(rng.normal(100, 10, (B, C, S))), 0, 255).astype(np.uint8)
    x[0, 0, 5] = 255
    buf[:, :, :S] = x
    buf[:, :, S:] = 7                    # padding must not be read or written
    outbuf = np.full((B, C, P), 9, dtype=np.uint8)
    o = oracle.Opts(P, 0, 0, outbuf.ctypes.data, None, None, None)
    st_ = oracle.raw_call("rfim_oracle_time_sigma_cut", buf.ctypes.data, B, C, S, oracle.U8, [3.0], oracle.MEAN, o)
    assert st_ == 0
    ref, _, _ = oracle.time_sigma_cut(x, [3.0])
    assert np.array_equal(outbuf[:, :, :S], ref) and np.all(outbuf[:, :, S:] == 9)
    assert np.array_equal(buf[:, :, :S], x) and np.all(buf[:, :, S:] == 7)
    # errors: nothing touched, -1 returned
    bad = [
        dict(beams=0), dict(channels=-1), dict(samples=0), dict(dtype=5), dict(policy=2),
        dict(thresholds=[0.0]), dict(thresholds=[-1.0]), dict(thresholds=[float("nan")]), dict(thresholds=[256.0]),
        dict(thresholds=[3.0] * 17),
    ]
    for kw in bad:
        args = dict(beams=B, channels=C, samples=S, dtype=oracle.U8, thresholds=[3.0], policy=oracle.MEAN)
        args.update(kw)
        st_ = oracle.raw_call("rfim_oracle_time_sigma_cut", buf.ctypes.data, args["beams"], args["channels"],
                              args["samples"], args["dtype"], args["thresholds"], args["policy"], None)
        assert st_ == -1, kw
    o = oracle.Opts(S - 1, 0, 0, None, None, None, None)
    assert oracle.raw_call("rfim_oracle_time_sigma_cut", buf.ctypes.data, B, C, S, 0, [3.0], 0, o) == -1
    o = oracle.Opts(0, 0, 2, None, None, None, None)     # 3 channels, bins of 2
    assert oracle.raw_call("rfim_oracle_freq_sigma_cut", buf.ctypes.data, B, C, S, 0, [3.0], 0, o) == -1
    assert oracle.raw_call("rfim_oracle_time_sigma_cut", None, B, C, S, 0, [3.0], 0, None) == -1
    # zero thresholds: a valid no-op
    y, f, c = oracle.time_sigma_cut(x, [])
    assert np.array_equal(y, x) and f.sum() == 0


# ----------------------------------------------------------------------------------------------------------------
# R22: with median replacement the snapshot median never changes from one iteration to the next --
# with L samples < m and E samples = m (L <= rank < L + E), replacing l samples from below and u from above by m
# leaves L - l <= rank < L + E + u.  The kernels take the median once per row / window / column on the strength of
# this; here the recomputing oracle is checked against the property (it is a theorem about the definition, so a
# failure would mean a wrong median or replacement step in the oracle).
@pytest.mark.parametrize("dtype", ["u8", "f32"])
def test_r22_median_is_invariant_under_median_replacement(dtype):
    rng = np.random.default_rng(22)
    for trial in range(40):
        n = int(rng.integers(5, 400))
        if dtype == "u8":
            row = np.clip(np.rint(rng.normal(100, 12, n)), 0, 255)
            row[rng.random(n) < 0.08] = rng.integers(0, 256)
            x = row.astype(np.uint8).reshape(1, 1, n)
        else:
            row = rng.normal(0, 1, n)
            row[rng.random(n) < 0.08] *= 30.0
            x = row.astype(np.float32).reshape(1, 1, n)
        ks = [float(k) for k in rng.choice([1.0, 1.5, 2.0, 3.0], size=4)]
        med = np.sort(x[0, 0])[(n - 1) // 2]
        out, flags, counts = oracle.time_sigma_cut(x, ks, policy=oracle.MEDIAN)
        assert np.all(out[0, 0][flags[0, 0] != 0] == med), (trial, ks)
        # the same along the channel axis, per bin
        nb = int(rng.choice([0, 1]))
        xc = np.ascontiguousarray(x.reshape(1, n, 1))
        outc, flagsc, _ = oracle.freq_sigma_cut(xc, ks, policy=oracle.MEDIAN)
        assert np.all(outc[0, :, 0][flagsc[0, :, 0] != 0] == med)
        if sum(int(c) for c in counts) > 0:
            assert np.sort(out[0, 0])[(n - 1) // 2] == med          # and the cleaned row still has that median
