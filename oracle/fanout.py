"""All-host-cores fan-out around the UNMODIFIED oracle calls -- TEST INFRASTRUCTURE ONLY.

Beams are independent in both sigma cuts (TDSC statistics are per (beam, channel) row, FDSC statistics per
(beam, sample) column), so a batch can be split along the beam axis and every slice handed to the plain,
single-threaded oracle (oracle/rfim_oracle.c) as it stands; ctypes releases the GIL for the duration of a
call, so plain threads are enough.  None of the method's arithmetic lives here: this module only slices,
calls and concatenates.  Used by the full-size parity tests and by bench.py's `cpu_baseline_all_cores` leg.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np

from . import freq_sigma_cut, lib, time_sigma_cut


def host_cores() -> int:
    try:
        return max(1, len(os.sched_getaffinity(0)))
    except AttributeError:  # pragma: no cover
        return max(1, os.cpu_count() or 1)


def _slices(beams: int, workers: int):
    per = (beams + workers - 1) // workers
    return [(b0, min(beams, b0 + per)) for b0 in range(0, beams, per)]


def fan_out(fn, data, thresholds, workers: int | None = None, **kw):
    """fn(data[b0:b1], thresholds, **kw) for beam slices on `workers` threads; returns what fn returns, with the
    arrays concatenated along the beam axis and the counts summed.  Also returns the thread count used."""
    lib()                                   # build / load once, outside the threads
    data = np.ascontiguousarray(data)
    workers = min(workers or host_cores(), data.shape[0])
    parts = _slices(data.shape[0], workers)
    with ThreadPoolExecutor(max_workers=len(parts)) as pool:
        res = list(pool.map(lambda p: fn(data[p[0]:p[1]], thresholds, **kw), parts))
    out = np.concatenate([r[0] for r in res], axis=0)
    flags = np.concatenate([r[1] for r in res], axis=0) if res[0][1] is not None else None
    counts = sum(r[2].astype(np.uint64) for r in res) if res[0][2] is not None else None
    return out, flags, counts, len(parts)


def chain(data, time_thresholds, freq_thresholds, workers: int | None = None, policy=0, window=0, bin_size=0,
          want_flags=False, want_counts=False):
    """TDSC then FDSC on its result, fanned out over beams.  Returns (cleaned, threads used)."""
    def one(x, _):
        y, _, _ = time_sigma_cut(x, time_thresholds, policy=policy, window=window, want_flags=want_flags,
                                 want_counts=want_counts)
        z, _, _ = freq_sigma_cut(y, freq_thresholds, policy=policy, bin_size=bin_size, want_flags=want_flags,
                                 want_counts=want_counts)
        return z, None, None
    out, _, _, n = fan_out(one, data, None, workers)
    return out, n
