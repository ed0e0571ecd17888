"""The seeded input generator: determinism, beam-range independence, and the stated recipe."""
import numpy as np

from paper_2001_03389_b200 import synth


def test_config1_recipe():
    cfg = synth.config(1)
    x = synth.fill_host(cfg)
    assert x.shape == (1, 64, 1024) and x.dtype == np.uint8
    d = synth.Descriptor(cfg)
    spikes = np.nonzero(d.imp_amp[0])[0]
    assert len(spikes) == 3 and np.all(d.imp_amp[0][spikes] == 80)
    clean = [c for c in range(64) if c not in (7, 40)]
    body = np.delete(x[0], spikes, axis=1)
    assert abs(body[clean].mean() - 100) < 0.3 and abs(body[clean].std() - 10) < 0.3
    assert abs(body[7].mean() - 160) < 1.5 and abs(body[40].mean() - 160) < 1.5
    assert np.array_equal(x, synth.fill_host(cfg))               # deterministic


def test_beam_ranges_are_independent_and_strided_fill():
    cfg = synth.config(2, beams=3, channels=64, samples=500)
    full = synth.fill_host(cfg)
    part = synth.fill_host(cfg, beam0=1, beams=2)
    assert np.array_equal(full[1:], part)
    padded = synth.fill_host(cfg, sample_stride=512)
    assert np.array_equal(padded[:, :, :500], full) and np.all(padded[:, :, 500:] == 0)


def test_arts_structure():
    cfg = synth.config(2, beams=2)
    d = synth.Descriptor(cfg, 0, 2)
    C, S = cfg["channels"], cfg["samples"]
    for b in range(2):
        persistent = np.count_nonzero(d.row_offset[b])
        bursty = sum(1 for c in range(C) if d.burst_ptr[b * C + c + 1] > d.burst_ptr[b * C + c])
        assert persistent + bursty == 77                           # 5 % of 1536 channels
        assert d.row_offset[b][d.row_offset[b] > 0].min() >= 40 and d.row_offset[b].max() <= 100
        assert 20 <= np.count_nonzero(d.imp_amp[b]) <= 100         # 20 impulses of 1..5 samples
    assert d.burst_len[:-1].min() >= 1 and d.burst_len.max() <= 500
    # Eq. 2: DM 500 sweep across 1220-1520 MHz is 0.496 s = 6055 samples at 81.92 us
    assert d.pulse_start[-1] - 1000 in (0, 1) and abs((d.pulse_start[0] - d.pulse_start[-1]) - 6051) < 10
    assert np.all(np.diff(d.pulse_start) <= 0)


def test_noise_cdf_is_the_rounded_clipped_gaussian():
    t = synth.noise_cdf(100.0, 12.0).astype(np.float64) / 2 ** 32
    assert np.all(np.diff(t) >= 0) and abs(t[99] - 0.4834) < 1e-3 and abs(t[100] - 0.5166) < 1e-3
    x = synth.fill_host(synth.config(2, beams=1, channels=8, samples=50000, kind="noise"))
    assert abs(x.mean() - 100) < 0.1 and abs(x.std() - np.sqrt(144 + 1 / 12)) < 0.1


def test_f32_config():
    cfg = synth.config(5, beams=1, channels=16, samples=2000)
    x = synth.fill_host(cfg)
    assert x.dtype == np.float32 and np.isfinite(x).all()
    d = synth.Descriptor(cfg, 0, 1)
    quiet = [c for c in range(16) if d.row_offset[0, c] == 0 and d.burst_ptr[c + 1] == d.burst_ptr[c]]
    body = x[0][quiet][:, d.imp_amp[0] == 0]
    assert abs(body.mean()) < 0.05 and abs(body.std() - 1) < 0.05
