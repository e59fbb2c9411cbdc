"""Multi-GPU host logic: chunks are independent, so the path shards with no data-path collective.
Each rank compresses/decompresses its own contiguous range of chunks with replicated weights; the only
exchange is the timing reduction (max over ranks) and the byte totals for the report."""
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
