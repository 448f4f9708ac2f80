"""world_size-2 `gloo` tests (CPU) of the N>1 host logic: F-sharding is a partition, sharded results
concatenate to the unsharded result with no exchange of data, and the timing reduction is a max.
The per-rank compute here is the oracle (this is a test); on the GPU box each rank runs
corr_execute on its shard instead."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads
from paper_1503_06203_b200 import shard


def test_channel_range_is_a_partition():
    for F in (0, 1, 2, 7, 8, 64, 1000):
        for world in (1, 2, 3, 4, 8):
            seen = []
            sizes = []
            for r in range(world):
                f0, f1 = shard.channel_range(F, r, world)
                assert 0 <= f0 <= f1 <= F
                seen += list(range(f0, f1))
                sizes.append(f1 - f0)
            assert seen == list(range(F))
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard.channel_range(8, 2, 2)


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, N, F, T, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        import oracle
        oracle.build()
        packed = workloads.uniform_bytes(N, F, T, seed=321)      # every rank draws the same stream ...
        mine = shard.shard_packed(packed, rank, world)            # ... and keeps only its channels
        f0, f1 = shard.channel_range(F, rank, world)
        assert mine.shape == (T, f1 - f0, N) and mine.flags["C_CONTIGUOUS"]
        vis_local = oracle.level1(mine)                           # no communication on the data path
        # test-only gather to compare with the unsharded result (not part of the product path)
        parts = [None] * world
        dist.all_gather_object(parts, vis_local)
        t = shard.max_over_ranks(1.0 + rank)                      # slowest rank decides
        if rank == 0:
            full = np.concatenate(parts, axis=0)
            want = oracle.level1(packed)
            out.put((bool(np.array_equal(full, want)), t))
        dist.barrier()
    finally:
        dist.destroy_process_group()


def test_two_ranks_shard_channels_without_collective():
    world, N, F, T = 2, 24, 5, 96          # odd F: ranks get 3 and 2 channels
    ctx = mp.get_context("spawn")
    out = ctx.SimpleQueue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, N, F, T, out)) for r in range(world)]
    for p in procs:
        p.start()
    for p in procs:
        p.join(120)
        assert p.exitcode == 0
    equal, t = out.get()
    assert equal
    assert t == 2.0


def test_max_over_ranks_without_group_is_identity():
    assert shard.max_over_ranks(0.25) == 0.25


def test_shard_packed_torch_tensor():
    packed = torch.arange(2 * 6 * 4, dtype=torch.uint8).reshape(2, 6, 4)
    a, b = shard.shard_packed(packed, 0, 2), shard.shard_packed(packed, 1, 2)
    assert a.is_contiguous() and b.is_contiguous()
    assert torch.equal(torch.cat([a, b], dim=1), packed)
