"""N>1 path on CPU: world_size-2 gloo run of the band-sharding + max-over-ranks timing logic bench.py uses."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2308_07277_b200 import dist_util as du


def test_shard_range_partitions_exactly():
    for n in (0, 1, 7, 16, 512, 513):
        for world in (1, 2, 3, 8):
            parts = [du.shard_range(n, r, world) for r in range(world)]
            assert parts[0][0] == 0 and parts[-1][1] == n
            assert all(a[1] == b[0] for a, b in zip(parts[:-1], parts[1:]))
            sizes = [b - a for a, b in parts]
            assert max(sizes) - min(sizes) <= 1
    assert du.units_per_step(512, 4, "weak") == 2048 and du.units_per_step(512, 4, "strong") == 512
    with pytest.raises(ValueError):
        du.shard_range(4, 2, 2)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        a, b = du.shard_range(513, rank, world)
        # every rank "times" its shard; the job time is the max over ranks
        ms = [10.0 + rank, 100.0 - rank]
        got = du.max_over_ranks(ms)
        # the shards cover the range exactly once
        cover = torch.zeros(513, dtype=torch.int64)
        cover[a:b] += 1
        dist.all_reduce(cover)
        dist.barrier()
        q.put((rank, got, int(cover.min()), int(cover.max()), b - a))
    finally:
        dist.destroy_process_group()


def test_world_size_two_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, got, lo, hi, size in res:
        assert got == [11.0, 100.0]            # max over ranks of [10+r, 100-r]
        assert lo == 1 and hi == 1
        assert size in (256, 257)
