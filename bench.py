#!/usr/bin/env python
"""bench.py -- one JSON line for the RFIm sigma-cut hot path on B200 ("Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--beams B]

A step is one pass of the whole hot path over one batch of synthetic ARTS-shaped input:
TDSC k = {5,4,3} (rows T1..T6 of SURVEY.md 8a) followed by FDSC k = {4,3} (rows F1..F6) on
BASELINE.json configs[3]: 480 beams x 1536 channels x 12500 samples uint8 (9.216 GB resident in HBM).
TDSC reads the pristine input and writes a second buffer, FDSC cleans that buffer in place, so every
timed step sees the same input.  `value` is the cleaned data rate of the whole step (batch bytes /
step time); per stage the JSON also carries read+write GB/s against the HBM roofline.

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

# dram__bytes_read.sum + dram__bytes_write.sum per launch from the committed `ncu --set full` captures
# (profiles/): kernel name -> (bytes per launch, beams in that launch, source file).  Scaled linearly to the
# launch bench.py times.  None until a capture exists.
NCU_TRAFFIC = {
    "td_u8_staged": (9.253756e9 + 9.172766e9, 480, "profiles/r1b_td_details.txt"),
    "fd_u8_strip1": (10.159767e9 + 9.180238e9, 480, "profiles/r1d_fd_details.txt"),
}


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


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

    def step(evs=None):
        if evs:
            evs[0].record()
        rfim.rfim_time_sigma_cut(x, TD_KS, out=y, variant=args.td_variant)
        if evs:
            evs[1].record()
        rfim.rfim_freq_sigma_cut(y, FD_KS, variant=args.fd_variant)
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
    rfim.rfim_time_sigma_cut(x[:1], TD_KS, out=y[:1]); td_name = rfim.rfim_last_variant()
    rfim.rfim_freq_sigma_cut(y[:1], FD_KS); fd_name = rfim.rfim_last_variant()
    torch.cuda.synchronize()
    ms_total = e0.elapsed_time(e1)
    ms_total = shard.max_over_ranks(ms_total, dev)
    ms_step = ms_total / K
    td_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in evs]))
    fd_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in evs]))
    batch_bytes = B * C * S
    value = world * batch_bytes / (ms_step * 1e-3) / 1e9

    # ---- end to end through the C ABI with HOST buffers (rank-local; same metric)
    e2e = None if args.no_e2e else e2e_leg(rfim, torch, x, y, cfg, world, dist, dev)

    # ---- roofline of the dominant kernel (algorithmic bytes: one read + one write per sample)
    peak, peak_src = hbm_peak()
    dom_name, dom_ms = (td_name, td_ms) if td_ms >= fd_ms else (fd_name, fd_ms)
    achieved = 2 * batch_bytes / (dom_ms * 1e-3) / 1e9
    traffic = None
    if dom_name in NCU_TRAFFIC:
        tb, tbeams, _ = NCU_TRAFFIC[dom_name]
        traffic = tb * (B / tbeams)
    roofline = {"bound": "hbm", "kernel": dom_name, "achieved": achieved, "peak": peak, "unit": "GB/s",
                "frac": achieved / peak, "traffic": traffic, "peak_source": peak_src,
                "algorithmic_bytes_per_launch": 2 * batch_bytes, "ms_per_launch": dom_ms,
                "frac_of_nominal_8000": achieved / 8000.0}
    stages = {
        "td": {"kernel": td_name, "ms": td_ms, "GBps_rw": 2 * batch_bytes / (td_ms * 1e-3) / 1e9,
               "frac_of_measured_peak": 2 * batch_bytes / (td_ms * 1e-3) / 1e9 / peak,
               "frac_of_nominal_8000": 2 * batch_bytes / (td_ms * 1e-3) / 1e9 / 8000.0,
               "realtime_margin": BATCH_SECONDS / (td_ms * 1e-3)},
        "fd": {"kernel": fd_name, "ms": fd_ms, "GBps_rw": 2 * batch_bytes / (fd_ms * 1e-3) / 1e9,
               "frac_of_measured_peak": 2 * batch_bytes / (fd_ms * 1e-3) / 1e9 / peak,
               "frac_of_nominal_8000": 2 * batch_bytes / (fd_ms * 1e-3) / 1e9 / 8000.0,
               "realtime_margin": BATCH_SECONDS / (fd_ms * 1e-3)},
    }

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline_leg(torch, x, y, cfg)

    if rank == 0:
        line = {
            "metric": "cleaned_GB_per_s", "value": value, "unit": "GB/s", "n_gpus": world, "steps": K,
            "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u8", "data": "synthetic", "config": workload_config(cfg),
            "samples_per_s": world * batch_bytes / (ms_step * 1e-3),
            "realtime_margin": BATCH_SECONDS / (ms_step * 1e-3),
            "stages": stages, "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks,
        }
        print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def e2e_leg(rfim, torch, x, y, cfg, world, dist, dev):
    """rfim_sigma_cut_host: pinned host input -> H2D -> TDSC -> FDSC -> D2H -> pinned host output, wall clock."""
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
    h_in.copy_(x[:nb])
    torch.cuda.synchronize()
    rfim.rfim_sigma_cut_host(h_in, TD_KS, FD_KS, out=h_out)       # warm-up (also checks the result below)
    ok = bool(torch.equal(h_out[:2].to(dev), y[:2]))
    times = []
    for _ in range(3):
        if dist is not None:
            dist.barrier()
        t0 = time.perf_counter()
        rfim.rfim_sigma_cut_host(h_in, TD_KS, FD_KS, out=h_out)
        times.append(time.perf_counter() - t0)
    sec = sum(times) / len(times)
    if dist is not None:
        t = torch.tensor([sec], device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        sec = float(t.item())
    nbytes = nb * C * S
    del h_in, h_out
    return {"value": world * nbytes / sec / 1e9, "unit": "GB/s", "h2d_bytes_per_step": nbytes,
            "d2h_bytes_per_step": nbytes, "ms_per_step": sec * 1e3, "beams": nb, "steps": 3,
            "matches_device_path": ok,
            "api": "rfim_sigma_cut_host (pinned host buffers, beams streamed through 3 staging buffers)"}


def cpu_baseline_leg(torch, x, y, cfg, beams: int = 16):
    """The oracle, as it stands, one core, on the first `beams` beams of the same input (about 15 s)."""
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


def run_table(args):
    """--table: one JSON line per BASELINE.json config 1, 2, 3, 5 (the parity-test configurations; the bench line
    proper is config 4).  Out of place, four rotating buffer pairs so that no repetition finds its input in L2,
    3 warm-ups, 20 timed repetitions on CUDA events, median and best."""
    import numpy as np
    import torch

    import paper_2001_03389_b200 as rfim
    from paper_2001_03389_b200 import synth
    dev = torch.device("cuda", 0)
    peak, _ = hbm_peak()
    cases = [(1, "time", None), (2, "time", None), (3, "freq", None), (5, "time", 256), (5, "time", 1024),
             (5, "time", 12500)]
    for (n, op, window) in cases:
        cfg = synth.config(n)
        host = synth.fill_host(cfg) if cfg["dtype"] == "f32" or cfg["beams"] * cfg["channels"] < 4096 else None
        pairs = []
        for _ in range(4):
            if host is not None:
                x = torch.from_numpy(host).to(dev)
            else:
                x = torch.empty((cfg["beams"], cfg["channels"], cfg["samples"]), dtype=torch.uint8, device=dev)
                synth.fill_device(cfg, x)
            pairs.append((x, torch.empty_like(x)))
        ks = cfg["thresholds"]

        def call(i):
            x, y = pairs[i % 4]
            if op == "time":
                rfim.rfim_time_sigma_cut(x, ks, cfg["policy"], out=y, window=window or 0)
            else:
                rfim.rfim_freq_sigma_cut(x, ks, cfg["policy"], out=y)
        for i in range(3):
            call(i)
        torch.cuda.synchronize()
        ms = []
        for i in range(20):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(); call(i); e1.record(); torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        med, best = float(np.median(ms)), float(min(ms))
        nbytes = 2 * pairs[0][0].numel() * pairs[0][0].element_size()
        print(json.dumps({"config": n, "op": op, "window": window, "kernel": rfim.rfim_last_variant(),
                          "thresholds": ks, "policy": cfg["policy"], "ms_median": med, "ms_best": best,
                          "samples_per_s": pairs[0][0].numel() / (med * 1e-3), "GBps_rw": nbytes / (med * 1e-3) / 1e9,
                          "frac_of_measured_peak": nbytes / (med * 1e-3) / 1e9 / peak,
                          "frac_of_nominal_8000": nbytes / (med * 1e-3) / 1e9 / 8000.0,
                          "realtime_margin": BATCH_SECONDS / (med * 1e-3)}), flush=True)
        del pairs


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--beams", type=int, default=0, help="override the beam count (testing only)")
    ap.add_argument("--td-variant", type=int, default=0, help="kernel variant for TDSC (tuning only; 0 = auto)")
    ap.add_argument("--fd-variant", type=int, default=0, help="kernel variant for FDSC (tuning only; 0 = auto)")
    ap.add_argument("--table", action="store_true", help="time configs 1, 2, 3, 5 instead (one JSON line each)")
    ap.add_argument("--no-cpu-baseline", action="store_true", help="skip the oracle leg (profiling runs)")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer leg (profiling runs)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    from paper_2001_03389_b200 import synth
    cfg = synth.config(4, **({"beams": args.beams} if args.beams else {}))
    if args.table:
        run_table(args)
    elif args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_ours(args, cfg)


if __name__ == "__main__":
    main()
