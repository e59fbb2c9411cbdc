"""O4 — the .boa container, format `BOA1`.  Oracle; test infrastructure.

One field per item the paper lists: first byte of each stream, the compressed streams, the nominal
chunk length, the length of the final chunk, the total uncompressed length, a compact model
fingerprint, and a CRC-protected index of per-stream sizes (offsets = their exclusive prefix sum).

    0   'BOA1'            4   u32 version = 1        8   u64 n (uncompressed bytes)
    16  u32 chunk_bytes   20  u32 last_chunk_len     24  u32 n_chunks
    28  u32 freq_bits=16  32  u64 model fingerprint
    40  u8  first[n_chunks], zero-padded to a multiple of 4
    ..  u32 size[n_chunks]
    ..  u32 CRC-32 (IEEE, zlib) of every byte before it
    ..  payload: the n_chunks range-coder streams back to back
"""
from __future__ import annotations

import struct
import zlib

MAGIC = b"BOA1"
VERSION = 1
HEADER_BYTES = 40
ORACLE_ARITH = 0x4F52434C  # 'ORCL' — fp64 oracle arithmetic; never equal to a GPU arithmetic word


class FormatError(ValueError):
    pass


def n_chunks_of(n: int, chunk_bytes: int) -> int:
    return -(-n // chunk_bytes) if n else 0


def index_bytes(n_chunks: int) -> int:
    return HEADER_BYTES + n_chunks + ((-n_chunks) % 4) + 4 * n_chunks + 4


def pack(n: int, chunk_bytes: int, fingerprint: int, first: bytes, payloads: list) -> bytes:
    nc = n_chunks_of(n, chunk_bytes)
    assert len(first) == nc and len(payloads) == nc
    last = n - (nc - 1) * chunk_bytes if nc else 0
    head = struct.pack("<4sIQIIIIQ", MAGIC, VERSION, n, chunk_bytes, last, nc, 16, fingerprint)
    head += bytes(first) + b"\0" * ((-nc) % 4)
    head += struct.pack(f"<{nc}I", *[len(p) for p in payloads])
    head += struct.pack("<I", zlib.crc32(head) & 0xFFFFFFFF)
    return head + b"".join(payloads)


def unpack(buf: bytes, fingerprint: int | None = None):
    """Returns (n, chunk_bytes, last_chunk_len, first, payloads).  Raises FormatError."""
    if len(buf) < HEADER_BYTES + 4:
        raise FormatError("truncated header")
    magic, ver, n, cb, last, nc, fb, fp = struct.unpack_from("<4sIQIIIIQ", buf, 0)
    if magic != MAGIC or ver != VERSION or fb != 16:
        raise FormatError("bad magic / version / freq_bits")
    if cb == 0 or nc != n_chunks_of(n, cb) or (nc and last != n - (nc - 1) * cb) or (not nc and last):
        raise FormatError("inconsistent lengths")
    ib = index_bytes(nc)
    if len(buf) < ib:
        raise FormatError("truncated index")
    (crc,) = struct.unpack_from("<I", buf, ib - 4)
    if crc != (zlib.crc32(buf[: ib - 4]) & 0xFFFFFFFF):
        raise FormatError("index CRC mismatch")
    if fingerprint is not None and fp != fingerprint:
        raise FormatError("model fingerprint mismatch")
    first = bytes(buf[HEADER_BYTES: HEADER_BYTES + nc])
    sizes = struct.unpack_from(f"<{nc}I", buf, HEADER_BYTES + nc + ((-nc) % 4))
    if ib + sum(sizes) != len(buf):
        raise FormatError("payload length does not match the index")
    payloads, off = [], ib
    for s in sizes:
        payloads.append(bytes(buf[off: off + s]))
        off += s
    return n, cb, last, first, payloads


def split_shards(buf: bytes) -> list:
    """Streaming output (PAPER Fig. 2): a concatenation of complete containers, one per group of chunks.
    Returns the shards; each one's length follows from its own header and size index.  Raises FormatError."""
    shards, off = [], 0
    while off < len(buf):
        if len(buf) - off < HEADER_BYTES + 4:
            raise FormatError("truncated shard header")
        magic, _ver, _n, _cb, _last, nc, _fb, _fp = struct.unpack_from("<4sIQIIIIQ", buf, off)
        if magic != MAGIC:
            raise FormatError("bad shard magic")
        ib = index_bytes(nc)
        if len(buf) - off < ib:
            raise FormatError("truncated shard index")
        sizes = struct.unpack_from(f"<{nc}I", buf, off + HEADER_BYTES + nc + ((-nc) % 4))
        total = ib + sum(sizes)
        if total > len(buf) - off:
            raise FormatError("truncated shard payload")
        shards.append(bytes(buf[off: off + total]))
        off += total
    return shards
