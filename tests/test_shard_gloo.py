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


# ---- one container from N ranks (8(f) NEXT-4): the host exchange + boa_container_assemble, on CPU ----
def _assemble_worker(rank, world, port, q, n, chunk):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    import numpy as np
    from oracle import codec, container, model
    from paper_2511_11337_b200 import boa, synth
    cfg = synth.CONFIGS[1]
    w = model.load_weights(cfg.weights(emb_std=0.25))
    data = cfg.data(n)
    fp = codec.fingerprint(w)
    # this rank's parts, made by the ORACLE from the bytes of its chunk range alone (chunks are independent)
    lo, hi = shard.byte_range(n, chunk, rank, world)
    _, _, _, first, payloads = container.unpack(codec.compress(w, data[lo:hi], chunk), fp)
    sizes = torch.tensor([len(p) for p in payloads], dtype=torch.int32)
    first_t = torch.frombuffer(bytearray(first), dtype=torch.uint8) if first else torch.empty(0, dtype=torch.uint8)
    pay = b"".join(payloads)
    payload = torch.frombuffer(bytearray(pay), dtype=torch.uint8) if pay else torch.empty(0, dtype=torch.uint8)
    blob = shard.exchange_and_assemble(lambda *a: boa.container_assemble(fp, *a), boa.container_index_bytes(n, chunk),
                                       n, chunk, sizes, first_t, payload, rank, world, torch.device("cpu"))
    whole = codec.compress(w, data, chunk) if rank == 0 else b""          # the single-process container of the same input
    q.put((rank, bytes(blob.numpy().tobytes()), whole))
    dist.destroy_process_group()


def _run_assemble(world, n, chunk):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    ps = [ctx.Process(target=_assemble_worker, args=(r, world, port, q, n, chunk)) for r in range(world)]
    [p.start() for p in ps]
    got = sorted(q.get(timeout=300) for _ in ps)
    [p.join(60) for p in ps]
    whole = got[0][2]
    assert len(whole) > 44
    for rank, blob, _ in got:
        assert blob == whole, (world, rank, len(blob), len(whole))   # byte-identical to the one-process container, on every rank


def test_one_container_from_two_ranks_gloo():
    _run_assemble(2, 7 * 40 + 13, 40)        # 8 chunks, ragged tail on the last rank


def test_one_container_from_three_ranks_with_an_empty_rank_gloo():
    _run_assemble(3, 2 * 30, 30)             # 2 chunks over 3 ranks: the last rank holds nothing


def test_container_assemble_host_only_errors():
    """boa_container_assemble with host pointers is plain host code: argument checks, and against the oracle's writer."""
    import numpy as np
    import pytest
    from oracle import container
    from paper_2511_11337_b200 import boa
    n, chunk = 10, 4                                                 # chunks of 4, 4, 2 bytes
    parts = [(torch.tensor([5, 6], dtype=torch.int32), torch.tensor([1, 2], dtype=torch.uint8)),
             (torch.tensor([4], dtype=torch.int32), torch.tensor([3], dtype=torch.uint8))]
    pays = [torch.arange(11, dtype=torch.uint8), torch.arange(100, 104, dtype=torch.uint8)]
    out = torch.zeros(200, dtype=torch.uint8)
    ln, offs = boa.container_assemble(0xABCDEF0012345678, n, chunk, parts, out, pays)
    want = container.pack(n, chunk, 0xABCDEF0012345678, bytes([1, 2, 3]),
                          [bytes(range(5)), bytes(range(5, 11)), bytes(range(100, 104))])
    assert out[:ln].numpy().tobytes() == want and offs == [boa.container_index_bytes(n, chunk), len(want) - 4, len(want)]
    with pytest.raises(boa.BoaError) as e:                           # a part whose payload is not the sum of its sizes
        boa.container_assemble(1, n, chunk, parts, out, [pays[0][:10], pays[1]])
    assert e.value.code == boa.E_FORMAT
    with pytest.raises(boa.BoaError) as e:                           # parts that do not cover the chunks
        boa.container_assemble(1, n, chunk, parts[:1], out, pays[:1])
    assert e.value.code == boa.E_ARG
    with pytest.raises(boa.BoaError) as e:
        boa.container_assemble(1, n, chunk, parts, out[:20], pays)
    assert e.value.code == boa.E_CAPACITY
