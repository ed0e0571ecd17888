"""World-size-2 gloo tests (CPU) of the multi-GPU host logic: beam partition, weak-scaling generator layout,
metadata collectives.  The sigma cuts shard by beam with no exchange step, which is
checked here with the oracle: cleaning each rank's beams separately equals cleaning the whole batch."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import oracle
from paper_2001_03389_b200 import shard, synth


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        cfg = synth.config(2, beams=5, channels=40, samples=700)
        b0, nb = shard.beam_slice(cfg["beams"], rank, world)
        x = synth.fill_host(cfg, beam0=b0, beams=nb)                      # this rank's beams only
        y, _, c1 = oracle.time_sigma_cut(x, [5.0, 4.0, 3.0])
        y, _, c2 = oracle.freq_sigma_cut(y, [4.0, 3.0])
        local_counts = torch.from_numpy(np.concatenate([c1, c2]).astype(np.int64))
        total = shard.sum_counts(local_counts)
        tmax = shard.max_over_ranks(10.0 + rank)
        gathered = [None] * world
        dist.all_gather_object(gathered, (b0, nb, y))
        if rank == 0:
            q.put((total.tolist(), tmax, gathered))
    finally:
        dist.destroy_process_group()


def test_beam_slice_partitions():
    for beams in (0, 1, 5, 12, 480, 481):
        for world in (1, 2, 3, 8):
            got = [shard.beam_slice(beams, r, world) for r in range(world)]
            assert got[0][0] == 0 and sum(n for _, n in got) == beams
            for (a0, an), (b0, _) in zip(got, got[1:]):
                assert a0 + an == b0
            assert max(n for _, n in got) - min(n for _, n in got) <= 1
    with pytest.raises(ValueError):
        shard.beam_slice(4, 2, 2)
    assert shard.weak_scaling_beam0(480, 3) == 1440


def test_world2_sharded_equals_whole_batch():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.SimpleQueue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    total, tmax, gathered = q.get()
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    cfg = synth.config(2, beams=5, channels=40, samples=700)
    x = synth.fill_host(cfg)
    ref, _, c1 = oracle.time_sigma_cut(x, [5.0, 4.0, 3.0])
    ref, _, c2 = oracle.freq_sigma_cut(ref, [4.0, 3.0])
    assert total == [int(v) for v in c1] + [int(v) for v in c2]
    assert tmax == 11.0
    pieces = sorted(gathered, key=lambda t: t[0])
    assert [p[:2] for p in pieces] == [(0, 3), (3, 2)]
    assert np.array_equal(np.concatenate([p[2] for p in pieces]), ref)


def test_single_process_helpers_without_process_group():
    c = torch.tensor([3, 4], dtype=torch.int64)
    assert shard.sum_counts(c).tolist() == [3, 4]
    assert shard.max_over_ranks(2.5) == 2.5
