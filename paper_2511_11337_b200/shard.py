"""Multi-GPU host logic: chunks are independent, so the path shards with no data-path collective.
Each rank compresses/decompresses its own contiguous range of chunks with replicated weights.

Weak scaling (bench.py default): independent replicas; the only exchange is the timing reduction (max over ranks)
and the byte totals for the report.
Strong scaling (8(f) NEXT-4): ONE input -> ONE BOA1 container over `world` ranks.  Rank r compresses chunks
[lo_r, hi_r) into parts (boa_compress_shard: payload block, per-chunk sizes, first bytes); the counts are all-gathered,
the small index parts are gathered on rank 0, every payload block is sent straight to its final place in rank 0's
container buffer, rank 0 writes header + index + CRC around them (boa_container_assemble) and broadcasts the container;
each rank then decodes its chunk range of it (boa_decompress_shard).  The container is byte-identical to the one
boa_compress writes for the whole input on one GPU.  Works on CUDA tensors over NCCL and on CPU tensors over gloo (the
CPU test drives exchange_and_assemble with parts made by the oracle)."""
from __future__ import annotations

import torch
import torch.distributed as dist


def chunk_range(n_chunks: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous, balanced split: the first (n_chunks % world) ranks get one extra chunk."""
    base, extra = divmod(n_chunks, world)
    lo = rank * base + min(rank, extra)
    return lo, lo + base + (1 if rank < extra else 0)


def byte_range(n: int, chunk_bytes: int, rank: int, world: int) -> tuple[int, int]:
    nc = -(-n // chunk_bytes) if n else 0
    lo, hi = chunk_range(nc, rank, world)
    return lo * chunk_bytes, min(n, hi * chunk_bytes)


def reduce_stats(local_ms: float, local_units: float, device=None) -> tuple[float, float]:
    """(max over ranks of local_ms, sum over ranks of local_units).  Identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return local_ms, local_units
    t = torch.tensor([local_ms], dtype=torch.float64, device=device)
    u = torch.tensor([local_units], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def barrier():
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


def exchange_and_assemble(assemble, index_bytes: int, n: int, chunk_bytes: int, sizes: torch.Tensor, first: torch.Tensor,
                          payload: torch.Tensor, rank: int, world: int, device, out: torch.Tensor | None = None) -> torch.Tensor:
    """Every rank holds the parts of its chunk range: sizes (int32, CPU), first (uint8, CPU), payload (uint8 on `device`,
    exactly sum(sizes) bytes).  Returns the assembled container (uint8 on `device`) on every rank.
    `assemble(n, chunk_bytes, parts, out, payloads)` is boa.container_assemble bound to the model's fingerprint;
    `index_bytes` = boa.container_index_bytes(n, chunk_bytes).  On rank 0 `out` may be a preallocated buffer whose bytes
    [index_bytes, index_bytes + len(payload)) already ARE rank 0's payload (compressed in place)."""
    nc = -(-n // chunk_bytes) if n else 0
    counts = torch.tensor([sizes.numel(), payload.numel()], dtype=torch.int64, device=device)
    all_counts = [torch.zeros(2, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(all_counts, counts)
    all_counts = [[int(v) for v in c.cpu()] for c in all_counts]
    assert sum(c[0] for c in all_counts) == nc, "the ranks' chunk ranges do not cover the input"
    # the small index parts: padded all-gather (5 bytes per chunk)
    width = max(c[0] for c in all_counts)
    pad_s = torch.zeros(max(width, 1), dtype=torch.int32, device=device)
    pad_f = torch.zeros(max(width, 1), dtype=torch.uint8, device=device)
    pad_s[: sizes.numel()] = sizes.to(device)
    pad_f[: first.numel()] = first.to(device)
    gs = [torch.zeros_like(pad_s) for _ in range(world)]
    gf = [torch.zeros_like(pad_f) for _ in range(world)]
    dist.all_gather(gs, pad_s)
    dist.all_gather(gf, pad_f)
    total = index_bytes + sum(c[1] for c in all_counts)
    offs = [index_bytes]
    for c in all_counts:
        offs.append(offs[-1] + c[1])
    if rank == 0:
        if out is None:
            out = torch.empty(total, dtype=torch.uint8, device=device)
            out[offs[0]: offs[1]] = payload
        assert out.numel() >= total
        reqs = [dist.irecv(out[offs[r]: offs[r + 1]], src=r) for r in range(1, world) if all_counts[r][1]]
        for q in reqs:
            q.wait()
        parts = [(gs[r][: all_counts[r][0]].cpu(), gf[r][: all_counts[r][0]].cpu()) for r in range(world)]
        written, got_offs = assemble(n, chunk_bytes, parts, out, [out[offs[r]: offs[r + 1]] for r in range(world)])
        assert written == total and got_offs == offs
        blob = out[:total]
    else:
        if payload.numel():
            dist.send(payload.contiguous(), dst=0)
        blob = torch.empty(total, dtype=torch.uint8, device=device)
    dist.broadcast(blob, src=0)
    return blob


def compress_sharded(m, d_in: torch.Tensor, chunk_bytes: int, rank: int, world: int, device) -> torch.Tensor:
    """One container from `world` GPUs: this rank compresses its chunk range of d_in (the whole input, on `device`)."""
    from . import boa
    n = d_in.numel()
    lo, hi = byte_range(n, chunk_bytes, rank, world)
    nc_local = -(-(hi - lo) // chunk_bytes) if hi > lo else 0
    ib = boa.container_index_bytes(n, chunk_bytes)
    cap = 2 * (hi - lo) + 4 * nc_local
    out = None
    if rank == 0:
        out = torch.empty(boa.compress_bound(n, chunk_bytes), dtype=torch.uint8, device=device)
        buf = out[ib: ib + cap]                       # rank 0's payload is compressed straight into its final place
    else:
        buf = torch.empty(max(cap, 1), dtype=torch.uint8, device=device)
    plen, sizes, first = m.compress_shard(d_in[lo:hi], chunk_bytes, buf)
    return exchange_and_assemble(m.container_assemble, ib, n, chunk_bytes, sizes, first, buf[:plen], rank, world, device, out)


def decompress_sharded(m, blob: torch.Tensor, d_out: torch.Tensor, rank: int, world: int) -> tuple[int, int]:
    """This rank decodes its chunk range of the shared container into its place in d_out; returns the byte range."""
    from . import boa
    n = boa.decompressed_size(blob)
    chunk_bytes = int.from_bytes(bytes(blob[16:20].cpu().tolist()), "little")
    nc = -(-n // chunk_bytes) if n else 0
    c_lo, c_hi = chunk_range(nc, rank, world)
    lo, hi = c_lo * chunk_bytes, min(n, c_hi * chunk_bytes)
    if c_hi > c_lo:
        m.decompress_shard(blob, c_lo, c_hi - c_lo, d_out[lo:hi])
    return lo, hi
