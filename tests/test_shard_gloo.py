"""N>1 host logic on CPU: world_size-2 gloo (shard whole ROM groups, no data-path collective;
the only reductions are the max step time and the cycle sum of the bench line)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_22447_b200.shard import shard_range, shard_envs, rank_seeds, reduce_job


def test_shard_range_partitions_every_group_once():
    for n in (0, 1, 7, 256, 257):
        for world in (1, 2, 3, 8):
            got = [shard_range(n, world, r) for r in range(world)]
            assert got[0][0] == 0 and got[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(got, got[1:]))
            sizes = [hi - lo for lo, hi in got]
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        shard_range(4, 2, 2)


def test_shard_envs_keeps_rom_groups_whole():
    env_rom = (np.arange(65536) >> 8).astype(np.int32)          # config 4: 256 envs per ROM
    parts = [shard_envs(env_rom, 256, 3, r) for r in range(3)]
    assert np.array_equal(np.concatenate(parts), np.arange(65536))
    for p in parts:
        roms, counts = np.unique(env_rom[p], return_counts=True)
        assert (counts == 256).all()
    with pytest.raises(ValueError):
        shard_envs(env_rom[:100], 256, 2, 0)


def _worker(rank, world, port, out):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        env_rom = (np.arange(2048) >> 8).astype(np.int32)
        mine = shard_envs(env_rom, 256, world, rank)
        seeds = rank_seeds(np.arange(4, dtype=np.uint64), rank)
        # every env is owned by exactly one rank: gather the owners' index lists
        gathered = [None] * world
        dist.all_gather_object(gathered, mine.tolist())
        t, c = reduce_job(dist, 10.0 + 5.0 * rank, 1000.0 * (rank + 1))
        out.put((rank, sorted(sum(gathered, [])) == list(range(2048)), t, c, int(seeds[1])))
    finally:
        dist.destroy_process_group()


def test_two_ranks_gloo():
    s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs: p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs: p.join(timeout=60)
    assert all(p.exitcode == 0 for p in procs)
    for rank, covered, t, c, seed1 in res:
        assert covered
        assert t == 15.0                      # max over ranks, the number bench.py divides by
        assert c == 3000.0                    # sum over ranks
        assert seed1 == (1 ^ (0x1000000 * rank))
    assert reduce_job(None, 3.0, 4.0) == (3.0, 4.0)
