"""GPU parity of the two composite entry points through the C ABI vs the CPU oracle, bit-exact:
rfim_time_freq_sigma_cut (TDSC then FDSC on its result; device pointers) and
rfim_sigma_cut_host (host buffers streamed through device staging buffers)."""
import numpy as np
import pytest
import torch

import oracle
import paper_2001_03389_b200 as rfim
from paper_2001_03389_b200 import synth

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def noisy(shape, seed, mu=100, sigma=12):
    rng = np.random.default_rng(seed)
    return np.clip(np.rint(rng.normal(mu, sigma, shape)), 0, 255).astype(np.uint8)


def oracle_chain(x, tks, fks, window=0, bin_size=0, policy=oracle.MEAN):
    y, tf, tc = oracle.time_sigma_cut(x, tks, window=window, policy=policy)
    z, ff, fc = oracle.freq_sigma_cut(y, fks, bin_size=bin_size, policy=policy)
    return z, tf | ff, [int(c) for c in tc] + [int(c) for c in fc]


@pytest.mark.parametrize("inplace", [False, True])
def test_chain_config4_slice(inplace):
    """BASELINE.json configs[3] on a 3-beam slice: TDSC {5,4,3} then FDSC {4,3}; cleaned array, the OR of both flag
    masks and the five per-iteration counts."""
    cfg = synth.config(4, beams=3)
    x = synth.fill_host(cfg, beam0=101, beams=3)
    ref, rflags, rcounts = oracle_chain(x, cfg["thresholds"], cfg["freq_thresholds"])
    xd = torch.from_numpy(x).to(DEV)
    out = None if inplace else torch.full_like(xd, 0xAB)
    flags = torch.full(x.shape, 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((5,), -1, dtype=torch.int64, device=DEV)
    res = rfim.rfim_time_freq_sigma_cut(xd, cfg["thresholds"], cfg["freq_thresholds"], out=out, flags=flags, counts=counts)
    torch.cuda.synchronize()
    assert rfim.rfim_last_variant() in ("fd_u8_quad", "fd_u8_stream", "fd_u8_strip1")
    assert np.array_equal(res.cpu().numpy(), ref)
    assert np.array_equal(flags.cpu().numpy(), rflags)
    assert counts.cpu().tolist() == rcounts and min(rcounts) > 0
    if not inplace:
        assert torch.equal(xd.cpu(), torch.from_numpy(x))


def test_chain_other_shapes_policies_and_empty_lists():
    x = noisy((2, 40, 300), seed=4)
    x[0, :, 100] = 250
    x[1, 2, 200:260] = 180
    xd = torch.from_numpy(x).to(DEV)
    for tks, fks, kw in (([3.25] * 3, [2.75, 2.75], {}), ([3.0], [3.0], dict(policy="median")),
                         ([4.0, 3.0], [3.0], dict(window=100, bin_size=8)), ([], [3.0], {}), ([3.0], [], {}), ([], [], {})):
        pol = oracle.MEDIAN if kw.get("policy") == "median" else oracle.MEAN
        ref, rflags, rcounts = oracle_chain(x, tks, fks, kw.get("window", 0), kw.get("bin_size", 0), pol)
        out = torch.full_like(xd, 0xAB)
        flags = torch.full(x.shape, 7, dtype=torch.uint8, device=DEV)
        counts = torch.full((max(1, len(tks) + len(fks)),), -1, dtype=torch.int64, device=DEV)
        rfim.rfim_time_freq_sigma_cut(xd, tks, fks, out=out, flags=flags, counts=counts, **kw)
        torch.cuda.synchronize()
        assert np.array_equal(out.cpu().numpy(), ref), (tks, fks, kw)
        assert np.array_equal(flags.cpu().numpy(), rflags), (tks, fks, kw)
        assert counts.cpu().tolist()[:len(rcounts)] == rcounts, (tks, fks, kw)
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_time_freq_sigma_cut(xd, [3.0], [3.0], variant=rfim.VARIANT_FD_STREAM)
    assert e.value.status == -2


def test_chain_and_host_path_with_the_papers_parameters():
    """The pipeline of PAPER.md:126,178 on a config-4 slice: TDSC three times at 3.25 sigma, then FDSC with bins of
    32 channels twice at 2.75 sigma -- through rfim_time_freq_sigma_cut (the binned streaming kernel behind the
    composite entry point) and through rfim_sigma_cut_host."""
    cfg = synth.config(4, beams=3)
    x = synth.fill_host(cfg, beam0=100, beams=3)
    tks, fks = [3.25, 3.25, 3.25], [2.75, 2.75]
    ref, rflags, rcounts = oracle_chain(x, tks, fks, 0, 32)
    xd = torch.from_numpy(x).to(DEV)
    out = torch.full_like(xd, 0xAB)
    flags = torch.full(x.shape, 7, dtype=torch.uint8, device=DEV)
    counts = torch.full((5,), -1, dtype=torch.int64, device=DEV)
    rfim.rfim_time_freq_sigma_cut(xd, tks, fks, out=out, bin_size=32, flags=flags, counts=counts)
    torch.cuda.synchronize()
    assert rfim.rfim_last_variant() == "fd_u8_qbin"
    assert np.array_equal(out.cpu().numpy(), ref)
    assert np.array_equal(flags.cpu().numpy(), rflags)
    assert counts.cpu().tolist() == rcounts and min(rcounts) > 0
    h = torch.from_numpy(x.copy()).pin_memory()
    hout = torch.empty_like(h).pin_memory()
    rfim.rfim_sigma_cut_host(h, tks, fks, out=hout, bin_size=32)
    assert np.array_equal(hout.numpy(), ref)


def test_chain_float32():
    rng = np.random.default_rng(9)
    x = rng.normal(0, 1, (2, 32, 500)).astype(np.float32)
    x[0, :, 77] += 9.0
    x[1, 5, :] += 6.0
    y, _, _ = oracle.time_sigma_cut(x, [4.0, 3.0], policy=oracle.MEDIAN, window=250)
    ref, _, _ = oracle.freq_sigma_cut(y, [3.0], policy=oracle.MEDIAN, bin_size=8)
    xd = torch.from_numpy(x).to(DEV)
    rfim.rfim_time_freq_sigma_cut(xd, [4.0, 3.0], [3.0], "median", window=250, bin_size=8)
    torch.cuda.synchronize()
    np.testing.assert_allclose(xd.cpu().numpy(), ref, rtol=1e-5, atol=0)


# ------------------------------------------------------------------------------------------ host path
@pytest.mark.parametrize("pinned", [True, False])
@pytest.mark.parametrize("use_workspace", [True, False])
def test_host_path_ragged_chunks(pinned, use_workspace):
    """15 beams of 1536 x 12500 in chunks of 6: a ragged last chunk (3 beams), three staging slots reused, pinned and
    pageable host memory, caller-provided and self-allocated staging buffers; a sample of beams against the oracle
    and the whole result against the device entry point."""
    cfg = synth.config(4, beams=15)
    x = synth.fill_host(cfg, beam0=200, beams=15)
    h_in = torch.from_numpy(x)
    h_out = torch.empty_like(h_in)
    if pinned:
        h_in = h_in.pin_memory()
        h_out = h_out.pin_memory()
    ws = None
    if use_workspace:
        need = rfim.rfim_workspace_bytes(rfim.OP_HOST, 15, 1536, 12500)
        ws = torch.empty(need, dtype=torch.uint8, device=DEV)
    n0 = rfim.rfim_launch_count()
    rfim.rfim_sigma_cut_host(h_in, cfg["thresholds"], cfg["freq_thresholds"], out=h_out, workspace=ws)
    assert rfim.rfim_launch_count() - n0 == 2 * 3
    assert torch.equal(h_in, torch.from_numpy(x)), "host input modified"
    xd = torch.from_numpy(x).to(DEV)
    rfim.rfim_time_freq_sigma_cut(xd, cfg["thresholds"], cfg["freq_thresholds"])
    torch.cuda.synchronize()
    assert torch.equal(h_out, xd.cpu())
    for b in (0, 5, 6, 14):
        ref, _, _ = oracle_chain(x[b:b + 1], cfg["thresholds"], cfg["freq_thresholds"])
        assert np.array_equal(h_out[b:b + 1].numpy(), ref), b


def test_host_path_pitch_in_place_single_ops_and_f32():
    x = noisy((5, 64, 1000), seed=12)
    x[:, 9, :] = 200
    x[1, :, 500] = 250
    pitch = 1008
    buf = np.full((5, 64, pitch), 0x5A, dtype=np.uint8)
    buf[:, :, :1000] = x
    h = torch.from_numpy(buf)
    view = h[:, :, :1000]
    rfim.rfim_sigma_cut_host(view, [4.0, 3.0], [3.0])                     # in place, padded pitch (2-D copies)
    ref, _, _ = oracle_chain(x, [4.0, 3.0], [3.0])
    assert np.array_equal(view.numpy(), ref) and np.all(h.numpy()[:, :, 1000:] == 0x5A)
    # TDSC only / FDSC only; a bin size that does not divide the channels is fine as long as FDSC does not run
    h2 = torch.from_numpy(x.copy())
    out = torch.empty_like(h2)
    rfim.rfim_sigma_cut_host(h2, [3.0], [], out=out, bin_size=7)
    assert np.array_equal(out.numpy(), oracle.time_sigma_cut(x, [3.0])[0])
    rfim.rfim_sigma_cut_host(h2, [], [3.0, 3.0], out=out, bin_size=16)
    assert np.array_equal(out.numpy(), oracle.freq_sigma_cut(x, [3.0, 3.0], bin_size=16)[0])
    with pytest.raises(rfim.RfimError) as e:
        rfim.rfim_sigma_cut_host(h2, [3.0], [3.0], out=out, bin_size=7)
    assert e.value.status == -1
    # float32, median, windows
    rng = np.random.default_rng(3)
    xf = rng.normal(0, 1, (3, 16, 700)).astype(np.float32)
    xf[0, :, 50] += 8
    hf = torch.from_numpy(xf.copy())
    rfim.rfim_sigma_cut_host(hf, [4.0, 3.0], [], "median", window=350)
    reff, _, _ = oracle.time_sigma_cut(xf, [4.0, 3.0], policy=oracle.MEDIAN, window=350)
    np.testing.assert_allclose(hf.numpy(), reff, rtol=1e-5, atol=0)
