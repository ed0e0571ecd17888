#!/usr/bin/env python
"""bench.py -- one JSON line for the RFIm sigma-cut hot path on B200 ("Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--beams B]

A step is one pass of the whole hot path over one batch of synthetic ARTS-shaped input:
TDSC k = {5,4,3} (rows T1..T6 of SURVEY.md 8a) followed by FDSC k = {4,3} (rows F1..F6) on
BASELINE.json configs[3]: 480 beams x 1536 channels x 12500 samples uint8 (9.216 GB resident in HBM).
TDSC reads the pristine input and writes a second buffer, FDSC cleans that buffer in place, so every
timed step sees the same input.  These are exactly the two enqueues rfim_time_freq_sigma_cut makes; they
are issued separately here so that a CUDA event can sit between them.  `value` is the cleaned data rate of
the whole step (batch bytes / step time); per stage the JSON also carries GB/s against the HBM roofline.

After the timed region the line gets a `table`: the other BASELINE.json configs (1, 2, 3, 5) and the NEXT rows
(binned FDSC, median TDSC) timed on their own, out of place with rotating buffers (or restored + L2 flushed
when in place), so that every number in BASELINE.md section 4 is in the driver's BENCH file.

N > 1 (torchrun): one process per GPU, each cleans its own 480-beam batch (beams are independent, there
is no exchange step: SURVEY.md 8e), barrier + device timing, max over ranks, scaling "weak".

`--impl reference` times the CPU oracle (oracle/, as it stands, one core) on a bounded sample of the
same workload; rank 0 only.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

TD_KS = [5.0, 4.0, 3.0]
FD_KS = [4.0, 3.0]
BATCH_SECONDS = 1.024            # one ARTS batch: 12500 samples at 81.92 us
FALLBACK_HBM_GBS = 6650.0        # /opt/skills/guides/B200_PROFILING.md, used only without MEASURED_PEAKS.json
NCU_TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.json")


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(kernel: str, beams: int):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel`, from the committed `ncu --set full`
    capture listed in profiles/ncu_traffic.json (kernel -> bytes, beams of that launch, source file), scaled
    linearly to the launch bench.py times.  None when no capture of this kernel is tracked."""
    try:
        with open(NCU_TRAFFIC_FILE) as f:
            ent = json.load(f)["kernels"].get(kernel)
        if not ent:
            return None, None
        return (ent["dram_bytes_read"] + ent["dram_bytes_write"]) * (beams / ent["beams"]), ent["source"]
    except Exception:
        return None, None


class ClockSampler:
    """nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index = index
        self.rows = []
        self.proc = None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, mx, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------ CPU oracle legs
def oracle_sample(cfg, beam0: int, beams: int):
    """Time the oracle as it stands (single thread) on `beams` beams of the workload: TDSC then FDSC.
    Input generation is outside the timed region.  Returns (seconds, bytes cleaned)."""
    import oracle
    from paper_2001_03389_b200 import synth
    x = synth.fill_host(cfg, beam0=beam0, beams=beams)
    t0 = time.perf_counter()
    y, _, _ = oracle.time_sigma_cut(x, TD_KS, want_flags=False, want_counts=False)
    y, _, _ = oracle.freq_sigma_cut(y, FD_KS, want_flags=False, want_counts=False)
    return time.perf_counter() - t0, x.size


def run_reference(args, cfg):
    """--impl reference: the oracle on the host cores, bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    total = args.steps + args.warmup
    beams = max(1, min(4, int(90.0 / (max(total, 1) * 1.0))))      # about 1 s of oracle time per beam
    beams = min(beams, cfg["beams"])
    times, nbytes = [], 0
    for i in range(total):
        dt, nbytes = oracle_sample(cfg, beam0=(i * beams) % max(1, cfg["beams"] - beams + 1), beams=beams)
        if i >= args.warmup:
            times.append(dt)
    sec = sum(times) / len(times)
    gbs = nbytes / sec / 1e9
    sample = f"{beams} of {cfg['beams']} beams per step ({nbytes / 1e6:.1f} MB), TDSC {TD_KS} then FDSC {FD_KS}"
    line = {
        "impl": "reference", "metric": "cleaned_GB_per_s", "value": gbs, "unit": "GB/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u8", "data": "synthetic",
        "config": workload_config(cfg),
        "samples_per_s": nbytes / sec,
        "realtime_margin": BATCH_SECONDS / (sec * cfg["beams"] / beams),
        "cpu_baseline": {"value": gbs, "unit": "GB/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": gbs, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }
    print(json.dumps(line), flush=True)


def workload_config(cfg):
    return {"workload": f"BASELINE.json configs[3]: {cfg['beams']} beams x {cfg['channels']} channels x "
                        f"{cfg['samples']} samples uint8, dense rows; TDSC k={TD_KS} then FDSC k={FD_KS}, mean "
                        "replacement",
            "beams": cfg["beams"], "channels": cfg["channels"], "samples": cfg["samples"],
            "time_thresholds": TD_KS, "freq_thresholds": FD_KS, "policy": "mean",
            "l2": "inputs larger than L2 (9.2 GB per buffer vs 126 MB): no flush needed",
            "seed": cfg["seed"]}


# ------------------------------------------------------------------------------------------- our arm
def run_ours(args, cfg):
    import numpy as np
    import torch

    import paper_2001_03389_b200 as rfim
    from paper_2001_03389_b200 import shard, synth

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; librfim has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    B, C, S = cfg["beams"], cfg["channels"], cfg["samples"]
    x = torch.empty((B, C, S), dtype=torch.uint8, device=dev)     # pristine input, resident in HBM
    y = torch.empty_like(x)                                       # TDSC output, cleaned in place by FDSC
    gen_chunk = 48
    for b0 in range(0, B, gen_chunk):                             # rank r holds beams [r*B, (r+1)*B) of the stream
        nb = min(gen_chunk, B - b0)
        synth.fill_device(cfg, x[b0:b0 + nb], beam0=shard.weak_scaling_beam0(B, rank) + b0, beams=nb)
    torch.cuda.synchronize()

    names = ["", ""]                                              # kernels the two calls of a step selected
    # scratch of the FDSC call (its tile dispenser): the caller's, so that the timed calls allocate nothing
    ws = torch.zeros(max(256, rfim.rfim_workspace_bytes(rfim.OP_FREQ, B, C, S)), dtype=torch.uint8, device=dev)

    def step(evs=None):
        if evs:
            evs[0].record()
        rfim.rfim_time_sigma_cut(x, TD_KS, out=y, variant=args.td_variant)
        names[0] = rfim.rfim_last_variant()
        if evs:
            evs[1].record()
        rfim.rfim_freq_sigma_cut(y, FD_KS, variant=args.fd_variant, workspace=ws)
        names[1] = rfim.rfim_last_variant()
        if evs:
            evs[2].record()

    for _ in range(args.warmup):
        step()
    td_name = fd_name = ""
    barrier()
    K = args.steps
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.25)
    launches0 = rfim.rfim_launch_count()
    t0 = time.time()
    e0.record()
    for i in range(K):
        step(evs[i])
    e1.record()
    barrier()
    t1 = time.time()
    launches = rfim.rfim_launch_count() - launches0
    clocks = sampler.stop(t0, t1)
    td_name, fd_name = names
    ms_total = e0.elapsed_time(e1)
    ms_total = shard.max_over_ranks(ms_total, dev)
    ms_step = ms_total / K
    td_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    fd_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    batch_bytes = B * C * S
    value = world * batch_bytes / (ms_step * 1e-3) / 1e9

    # the composite entry point makes the same two enqueues: same result (checked on the whole buffer)
    chain_ok = None
    if not args.no_e2e:
        z = torch.empty_like(x)
        rfim.rfim_time_freq_sigma_cut(x, TD_KS, FD_KS, out=z)
        torch.cuda.synchronize()
        chain_ok = bool(torch.equal(z, y))
        del z

    # ---- end to end through the C ABI with HOST buffers (rank-local; same metric)
    e2e = None if args.no_e2e else e2e_leg(rfim, torch, x, y, cfg, world, dist, dev)

    # ---- roofline of the dominant kernel.  Algorithmic bytes: one read + one
    # write per sample for every stage.  (In place the streaming FDSC kernel does not rewrite a sample it leaves
    # alone, so its measured DRAM traffic is below the algorithmic bytes; the fraction is still quoted against them.)
    peak, peak_src = hbm_peak()
    td_bytes = 2 * batch_bytes
    fd_bytes = 2 * batch_bytes       # 2 B per uint8 sample, whatever the kernel manages to skip
    fd_skips_writes = fd_name in ("fd_u8_quad", "fd_u8_stream", "fd_u8_stream_binned", "fd_u8_qbin")
    dom_name, dom_ms, dom_bytes = (td_name, td_ms, td_bytes) if td_ms >= fd_ms else (fd_name, fd_ms, fd_bytes)
    achieved = dom_bytes / (dom_ms * 1e-3) / 1e9
    traffic, traffic_src = ncu_traffic(dom_name, B)
    roofline = {"bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": dom_bytes, "ms_per_launch": dom_ms,
                "frac_of_nominal_8000": achieved / 8000.0}

    def stage(name, ms, nbytes, what):
        t, src = ncu_traffic(name, B)
        return {"kernel": name, "ms": ms, "algorithmic_bytes": nbytes, "bytes_counted": what,
                "GBps": nbytes / (ms * 1e-3) / 1e9, "frac_of_measured_peak": nbytes / (ms * 1e-3) / 1e9 / peak,
                "frac_of_nominal_8000": nbytes / (ms * 1e-3) / 1e9 / 8000.0,
                "realtime_margin": BATCH_SECONDS / (ms * 1e-3), "ncu_dram_bytes": t, "ncu_source": src}
    stages = {
        "td": stage(td_name, td_ms, td_bytes, "one read + one write per sample (out of place)"),
        "fd": stage(fd_name, fd_ms, fd_bytes,
                    "one read + one write per sample (in place; the kernel itself writes only replaced samples)"
                    if fd_skips_writes else "one read + one write per sample (in place)"),
        "chain": {"ms": ms_step, "algorithmic_bytes": 4 * batch_bytes,
                  "bytes_counted": "TDSC read + write, FDSC read + write (the intermediate goes through HBM: two "
                                   "launches)",
                  "GBps": 4 * batch_bytes / (ms_step * 1e-3) / 1e9,
                  "frac_of_measured_peak": 4 * batch_bytes / (ms_step * 1e-3) / 1e9 / peak,
                  "rfim_time_freq_sigma_cut_matches": chain_ok},
    }

    cpu = cpu_all = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_leg(torch, x, y, cfg)
        cpu_all = cpu_baseline_all_cores_leg(torch, x, y, cfg)
    table = None
    if rank == 0 and world == 1 and not args.no_table:
        del x, y
        torch.cuda.empty_cache()
        table = run_table(quiet=True)

    if rank == 0:
        line = {
            "metric": "cleaned_GB_per_s", "value": value, "unit": "GB/s", "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic", "config": workload_config(cfg),
            "samples_per_s": world * batch_bytes / (ms_step * 1e-3),
            "realtime_margin": BATCH_SECONDS / (ms_step * 1e-3),
            "stages": stages, "roofline": roofline, "cpu_baseline": cpu, "cpu_baseline_all_cores": cpu_all,
            "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks, "table": table,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def e2e_leg(rfim, torch, x, y, cfg, world, dist, dev):
    """rfim_sigma_cut_host: pinned host input -> H2D -> TDSC -> FDSC -> D2H -> pinned host output, wall clock.
    The device staging buffers are the caller's (opts->workspace): nothing is allocated inside the timed call."""
    B, C, S = cfg["beams"], cfg["channels"], cfg["samples"]
    nb = B
    h_in = h_out = None
    while nb >= 1:
        try:
            h_in = torch.empty((nb, C, S), dtype=torch.uint8, pin_memory=True)
            h_out = torch.empty((nb, C, S), dtype=torch.uint8, pin_memory=True)
            break
        except RuntimeError:
            h_in = h_out = None
            nb //= 2
    if h_in is None:
        return {"value": None, "unit": "GB/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0,
                "note": "pinned host allocation failed"}
    ws = torch.empty(rfim.rfim_workspace_bytes(rfim.OP_HOST, nb, C, S), dtype=torch.uint8, device=dev)
    h_in.copy_(x[:nb])
    torch.cuda.synchronize()
    rfim.rfim_sigma_cut_host(h_in, TD_KS, FD_KS, out=h_out, workspace=ws)   # warm-up (also checks the result below)
    ok = bool(torch.equal(h_out[:2].to(dev), y[:2])) and bool(torch.equal(h_out[nb - 1:].to(dev), y[nb - 1:nb]))
    times = []
    for _ in range(3):
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        rfim.rfim_sigma_cut_host(h_in, TD_KS, FD_KS, out=h_out, workspace=ws)
        times.append(time.perf_counter() - t0)
    sec = sum(times) / len(times)
    if dist is not None:
        t = torch.tensor([sec], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        sec = float(t.item())
    nbytes = nb * C * S
    del h_in, h_out, ws
    return {"value": world * nbytes / sec / 1e9, "unit": "GB/s", "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "ms_per_step": sec * 1e3, "beams": nb, "steps": 3,
            "matches_device_path": ok,
            "api": "rfim_sigma_cut_host (pinned host buffers, beams streamed through 3 caller-provided staging "
                   "buffers on 3 streams)"}


def cpu_baseline_leg(torch, x, y, cfg, beams: int = 16):
    """The oracle, as it stands, one core, on the first `beams` beams of the same input (about 6 s)."""
    import numpy as np

    import oracle
    oracle.build()
    beams = min(beams, cfg["beams"])
    xs = x[:beams].cpu().numpy()
    t0 = time.perf_counter()
    r, _, _ = oracle.time_sigma_cut(xs, TD_KS, want_flags=False, want_counts=False)
    r, _, _ = oracle.freq_sigma_cut(r, FD_KS, want_flags=False, want_counts=False)
    sec = time.perf_counter() - t0
    same = bool(np.array_equal(r, y[:beams].cpu().numpy()))
    return {"value": xs.size / sec / 1e9, "unit": "GB/s", "cores": 1, "kind": "oracle",
            "sample": f"first {beams} of {cfg['beams']} beams ({xs.size / 1e6:.1f} MB), TDSC {TD_KS} then FDSC "
                      f"{FD_KS}, {sec:.1f} s",
            "gpu_output_bit_exact_on_sample": same}


def cpu_baseline_all_cores_leg(torch, x, y, cfg):
    """The same unmodified oracle calls fanned out over beams on all host cores (oracle/fanout.py: threads around the
    ctypes calls, no arithmetic of its own).  Sample: the LAST beams of the batch, 4 per core, at most 96."""
    import numpy as np

    from oracle import fanout
    cores = fanout.host_cores()
    beams = min(cfg["beams"], max(16, min(96, 4 * cores)))
    b0 = cfg["beams"] - beams
    xs = x[b0:].cpu().numpy()
    t0 = time.perf_counter()
    r, nthreads = fanout.chain(xs, TD_KS, FD_KS, workers=cores)
    sec = time.perf_counter() - t0
    same = bool(np.array_equal(r, y[b0:].cpu().numpy()))
    return {"value": xs.size / sec / 1e9, "unit": "GB/s", "cores": nthreads, "kind": "oracle, fanned out over beams",
            "sample": f"last {beams} of {cfg['beams']} beams ({xs.size / 1e6:.1f} MB), TDSC {TD_KS} then FDSC "
                      f"{FD_KS}, {sec:.1f} s on {nthreads} threads ({cores} cores available)",
            "gpu_output_bit_exact_on_sample": same}


TABLE_CASES = [
    # (label, config, op, kwargs of the call, in place?)
    ("cfg1 TDSC u8 {3}", 1, "time", {}, False),
    ("cfg2 TDSC u8 {5,4,3}", 2, "time", {}, False),
    ("cfg2 TDSC u8 {5,4,3} median", 2, "time", {"policy": "median"}, False),
    ("cfg3 FDSC u8 {4,3} out of place", 3, "freq", {}, False),
    ("cfg3 FDSC u8 {4,3} in place", 3, "freq", {}, True),
    ("cfg3 FDSC u8 bins of 32, {2.75,2.75} out of place", 3, "freq", {"bin_size": 32, "ks": [2.75, 2.75]}, False),
    ("cfg3 FDSC u8 bins of 32, {2.75,2.75} in place", 3, "freq", {"bin_size": 32, "ks": [2.75, 2.75]}, True),
    ("cfg3 FDSC u8 {4,3} median, in place", 3, "freq", {"policy": "median"}, True),
    ("cfg4 x 96 beams FDSC u8 {4,3} in place", 4, "freq", {"beams": 96, "ks": [4.0, 3.0]}, True),
    ("cfg4 x 96 beams FDSC u8 {4,3} out of place", 4, "freq", {"beams": 96, "ks": [4.0, 3.0]}, False),
    ("cfg4 x 96 beams FDSC u8 bins of 32, {2.75,2.75} in place", 4, "freq",
     {"beams": 96, "bin_size": 32, "ks": [2.75, 2.75]}, True),
    ("cfg4 x 96 beams TDSC u8 {5,4,3} median", 4, "time", {"beams": 96, "policy": "median"}, False),
    ("cfg5 TDSC f32 W=256 median", 5, "time", {"window": 256}, False),
    ("cfg5 TDSC f32 W=1024 median", 5, "time", {"window": 1024}, False),
    ("cfg5 TDSC f32 W=12500 median", 5, "time", {"window": 12500}, False),
    ("cfg5 TDSC f32 W=256 mean", 5, "time", {"window": 256, "policy": "mean"}, False),
    ("cfg5 TDSC f32 W=1024 mean", 5, "time", {"window": 1024, "policy": "mean"}, False),
    ("cfg5 TDSC f32 W=12500 mean", 5, "time", {"window": 12500, "policy": "mean"}, False),
    ("cfg5-shaped FDSC f32 {4,3} mean", 5, "freq", {"policy": "mean"}, False),
    ("cfg5-shaped FDSC f32 {4,3} median", 5, "freq", {"policy": "median"}, False),
    ("cfg5-shaped FDSC f32 bins of 32, {2.75,2.75} mean", 5, "freq", {"policy": "mean", "bin_size": 32, "ks": [2.75, 2.75]},
     False),
]


def run_table(quiet: bool = False, only: str = ""):
    """The other BASELINE.json configs (1, 2, 3, 5: the parity-test configurations; the bench line proper is
    config 4) and the NEXT rows, each timed on its own: 3 warm-ups, 20 timed repetitions, each between its own pair
    of CUDA events, median and best; the repetitions of a case are enqueued back to back and synchronised once.
    Out of place: four rotating buffer pairs, so that no repetition finds its input in L2 (a pair comes round again
    after more than 1 GB of other traffic).  In place: the buffer is restored from a pristine copy and L2 is flushed
    (a 512 MB write) before every repetition, outside the events."""
    import numpy as np
    import torch

    import paper_2001_03389_b200 as rfim
    from paper_2001_03389_b200 import synth
    dev = torch.device("cuda", torch.cuda.current_device())
    peak, _ = hbm_peak()
    rows = []
    flush = torch.empty(512 << 20, dtype=torch.uint8, device=dev)
    inputs = {}
    for (label, n, op, kw, inplace) in TABLE_CASES:
        if only and only not in label:
            continue
        cfg = synth.config(n, **({"beams": kw["beams"]} if "beams" in kw else {}))
        if n not in inputs:
            inputs.clear()
            torch.cuda.empty_cache()
            host = synth.fill_host(cfg) if cfg["dtype"] == "f32" or cfg["beams"] * cfg["channels"] < 4096 else None
            xs = []
            for _ in range(4):
                if host is not None:
                    xi = torch.from_numpy(host).to(dev)
                else:
                    xi = torch.empty((cfg["beams"], cfg["channels"], cfg["samples"]), dtype=torch.uint8, device=dev)
                    synth.fill_device(cfg, xi)
                xs.append(xi)
            inputs[n] = (xs, [torch.empty_like(xs[0]) for _ in range(4)])
        xs, ys = inputs[n]
        ks = kw.get("ks", cfg["thresholds"])
        policy = kw.get("policy", cfg["policy"])

        def call(i):
            xi, yi = xs[i % 4], ys[i % 4]
            if inplace:
                xi, yi = ys[0], None
            if op == "time":
                rfim.rfim_time_sigma_cut(xi, ks, policy, out=yi, window=kw.get("window", 0))
            else:
                rfim.rfim_freq_sigma_cut(xi, ks, policy, out=yi, bin_size=kw.get("bin_size", 0))

        def prepare():
            if inplace:
                ys[0].copy_(xs[0])
                flush.fill_(1)
        # all repetitions are enqueued back to back (the device never idles between them, so short kernels are not
        # timed on a GPU that has just dropped its clocks); every repetition has its own pair of events
        evs = []
        for i in range(23):
            prepare()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); call(i); e1.record()
            evs.append((e0, e1))
        torch.cuda.synchronize()
        ms = [a.elapsed_time(b) for (a, b) in evs[3:]]
        med, best = float(np.median(ms)), float(min(ms))
        elems = xs[0].numel()
        es = xs[0].element_size()
        name = rfim.rfim_last_variant()
        nbytes = elems * es * 2                          # one read + one write per sample
        row = {"case": label, "config": n, "op": op, "kernel": name, "thresholds": ks, "policy": policy,
               "window": kw.get("window"), "bin_size": kw.get("bin_size"), "in_place": inplace,
               "ms_median": med, "ms_best": best, "samples_per_s": elems / (med * 1e-3),
               "algorithmic_bytes": nbytes,
               "bytes_counted": "one read + one write per sample",
               "GBps": nbytes / (med * 1e-3) / 1e9, "frac_of_measured_peak": nbytes / (med * 1e-3) / 1e9 / peak,
               "frac_of_nominal_8000": nbytes / (med * 1e-3) / 1e9 / 8000.0,
               "realtime_margin": BATCH_SECONDS / (med * 1e-3)}
        rows.append(row)
        if not quiet:
            print(json.dumps(row), flush=True)
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--beams", type=int, default=0, help="override the beam count (testing only)")
    ap.add_argument("--td-variant", type=int, default=0, help="kernel variant for TDSC (tuning only; 0 = auto)")
    ap.add_argument("--fd-variant", type=int, default=0, help="kernel variant for FDSC (tuning only; 0 = auto)")
    ap.add_argument("--table", action="store_true", help="only the table (one JSON line per case)")
    ap.add_argument("--cases", default="", help="with --table: only the cases whose label contains this text")
    ap.add_argument("--no-table", action="store_true", help="skip the table (profiling runs)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle legs (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    from paper_2001_03389_b200 import synth
    cfg = synth.config(4, **({"beams": args.beams} if args.beams else {}))
    if args.table:
        run_table(only=args.cases)
    elif args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
