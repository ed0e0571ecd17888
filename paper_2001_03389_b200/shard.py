"""Multi-GPU host logic: the sigma cuts shard by beam with no exchange step.

TDSC units are (beam, channel) rows, FDSC units are (beam, sample) columns and the chain needs whole
beams, so a global batch is partitioned over ranks by contiguous beam ranges and every rank runs the
single-GPU library on its slice.  Nothing here moves sample data between ranks; the only collectives
are on metadata (replacement counts, timings), so they work on any backend (NCCL on GPUs, gloo in the
CPU tests).
"""
from __future__ import annotations

from typing import Optional, Sequence, Tuple

import torch
import torch.distributed as dist


def beam_slice(beams: int, rank: int, world: int) -> Tuple[int, int]:
    """(first beam, number of beams) of `rank`: contiguous, balanced, the remainder goes to the first ranks."""
    if beams < 0 or world <= 0 or not (0 <= rank < world):
        raise ValueError("beam_slice: bad arguments")
    base, rem = divmod(beams, world)
    b0 = rank * base + min(rank, rem)
    return b0, base + (1 if rank < rem else 0)


def weak_scaling_beam0(beams_per_rank: int, rank: int) -> int:
    """bench.py's weak-scaling layout: rank r holds beams [r * B, (r + 1) * B) of the generator's stream."""
    return rank * beams_per_rank


def _world(group=None) -> Tuple[int, int]:
    if dist.is_available() and dist.is_initialized():
        return dist.get_rank(group), dist.get_world_size(group)
    return 0, 1


def sum_counts(counts: torch.Tensor, group=None) -> torch.Tensor:
    """Global replacement counts per threshold: the sum of every rank's local `counts` (int64)."""
    out = counts.clone()
    if _world(group)[1] > 1:
        dist.all_reduce(out, op=dist.ReduceOp.SUM, group=group)
    return out


def max_over_ranks(value: float, device: Optional[torch.device] = None, group=None) -> float:
    """Timing rule: a multi-GPU time is the maximum over ranks."""
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if _world(group)[1] > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX, group=group)
    return float(t.item())


def sigma_cut_sharded(local: torch.Tensor, time_thresholds: Sequence[float], freq_thresholds: Sequence[float],
                      policy="mean", *, window: int = 0, bin_size: int = 0, group=None) -> torch.Tensor:
    """Clean this rank's beams (a CUDA tensor [local beams][channels][samples]) in place with TDSC then FDSC and
    return the GLOBAL per-threshold replacement counts (time thresholds first).  No sample data is exchanged."""
    from . import binding
    nt, nf = len(time_thresholds), len(freq_thresholds)
    counts = torch.zeros(max(1, nt + nf), dtype=torch.int64, device=local.device)
    if local.shape[0] > 0:
        if nt:
            binding.rfim_time_sigma_cut(local, time_thresholds, policy, window=window, counts=counts[:nt])
        if nf:
            binding.rfim_freq_sigma_cut(local, freq_thresholds, policy, bin_size=bin_size, counts=counts[nt:nt + nf])
    return sum_counts(counts[:nt + nf], group)
