"""N>1 host logic on CPU: world_size-2 gloo process group (tier framing (5)): chunk sharding covers the input
exactly once, and the timing reduction is max-over-ranks / sum-of-units."""
import os
import socket

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2511_11337_b200 import shard


def test_chunk_ranges_partition_exactly():
    for nc in (0, 1, 2, 7, 4096, 65537):
        for world in (1, 2, 3, 8):
            r = [shard.chunk_range(nc, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == nc
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1
    assert shard.byte_range(1000, 300, 0, 2) == (0, 600) and shard.byte_range(1000, 300, 1, 2) == (600, 1000)


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    shard.barrier()
    ms, units = shard.reduce_stats(10.0 + 5.0 * rank, 100.0 * (rank + 1))
    lo, hi = shard.byte_range(1000, 300, rank, world)
    t = torch.tensor([hi - lo], dtype=torch.int64)
    dist.all_reduce(t)
    q.put((rank, ms, units, int(t.item())))
    dist.destroy_process_group()


def test_reduce_stats_world2_gloo():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    got = sorted(q.get(timeout=120) for _ in ps)
    [p.join(60) for p in ps]
    assert got == [(0, 15.0, 300.0, 1000), (1, 15.0, 300.0, 1000)]
    assert shard.reduce_stats(3.0, 4.0) == (3.0, 4.0)      # no process group: identity
