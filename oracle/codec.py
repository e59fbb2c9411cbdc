"""Chunk-parallel compress / decompress, the oracle's whole path.  Test infrastructure.

compress: split the input into chunks of `chunk_bytes` (streams); store the first byte of each
stream raw; for t = 0 .. len-2 feed byte t to the step function, turn the logits into the integer
table, and range-code byte t+1; pack everything into the container.
decompress: load the metadata, run the same model on the bytes decoded so far, decode all
streams in lock-step; a stream that has reached its length is masked out (here: equal-length streams
are grouped, the ragged last chunk forms its own group).

The logits are fp64 (O1); they are rounded once to fp32 before the quantiser because the table rule
(O2) is defined on fp32 logits.
"""
from __future__ import annotations

import numpy as np

from . import container, model, quantise
from .rangecoder import RangeDecoder, RangeEncoder


def fingerprint(w: model.Weights) -> int:
    return (container.ORACLE_ARITH << 32) | w.blob_crc


def _groups(n: int, chunk_bytes: int):
    """Yield (first_chunk_id, n_streams, length) for the equal-length groups."""
    nc = container.n_chunks_of(n, chunk_bytes)
    if nc == 0:
        return
    last = n - (nc - 1) * chunk_bytes
    if last == chunk_bytes:
        yield 0, nc, chunk_bytes
    else:
        if nc > 1:
            yield 0, nc - 1, chunk_bytes
        yield nc - 1, 1, last


def compress(w: model.Weights, data: bytes, chunk_bytes: int) -> bytes:
    n = len(data)
    buf = np.frombuffer(data, dtype=np.uint8)
    nc = container.n_chunks_of(n, chunk_bytes)
    first = bytearray(nc)
    payloads = [b""] * nc
    for c0, s, length in _groups(n, chunk_bytes):
        if s > 1 or length == chunk_bytes:
            chunks = buf[c0 * chunk_bytes: c0 * chunk_bytes + s * length].reshape(s, length)
        else:
            chunks = buf[c0 * chunk_bytes:].reshape(1, length)
        st = model.init_state(w, s)
        encs = [RangeEncoder() for _ in range(s)]
        first[c0: c0 + s] = chunks[:, 0].tobytes()
        for t in range(length - 1):
            logits = model.step(w, st, chunks[:, t])
            C = quantise.quantise(logits.astype(np.float32))
            nxt = chunks[:, t + 1]
            for i in range(s):
                encs[i].encode(int(C[i, nxt[i]]), int(C[i, int(nxt[i]) + 1]))
        for i in range(s):
            payloads[c0 + i] = encs[i].finish()
    return container.pack(n, chunk_bytes, fingerprint(w), bytes(first), payloads)


def decompress(w: model.Weights, blob: bytes) -> bytes:
    n, chunk_bytes, _last, first, payloads = container.unpack(blob, fingerprint(w))
    out = np.zeros(n, dtype=np.uint8)
    for c0, s, length in _groups(n, chunk_bytes):
        st = model.init_state(w, s)
        decs = [RangeDecoder(payloads[c0 + i]) for i in range(s)]
        cur = np.frombuffer(first[c0: c0 + s], dtype=np.uint8).copy()
        rows = np.zeros((s, length), dtype=np.uint8)
        rows[:, 0] = cur
        for t in range(length - 1):
            logits = model.step(w, st, cur)
            C = quantise.quantise(logits.astype(np.float32))
            for i in range(s):
                x = decs[i].target()
                sym = quantise.find_symbol(C[i], x)
                decs[i].consume(int(C[i, sym]), int(C[i, sym + 1]))
                cur[i] = sym
            rows[:, t + 1] = cur
        for i in range(s):
            if decs[i].pos != len(payloads[c0 + i]):
                raise container.FormatError("stream not fully consumed")
        base = c0 * chunk_bytes
        out[base: base + s * length] = rows.reshape(-1)
    return out.tobytes()


def stream_compress(w: model.Weights, data: bytes, chunk_bytes: int, group_chunks: int) -> list:
    """Streaming pipeline (PAPER Fig. 2): the distributor cuts the sequence into groups of `group_chunks`
    fixed-size chunks and every group is compressed into its own shard (a complete container).  Returns the shards
    in order; the stream is their concatenation."""
    g = chunk_bytes * group_chunks
    return [compress(w, data[o: o + g], chunk_bytes) for o in range(0, len(data), g)]


def stream_decompress(w: model.Weights, blob: bytes) -> bytes:
    return b"".join(decompress(w, s) for s in container.split_shards(blob))


def probabilities(w: model.Weights, chunks: np.ndarray) -> np.ndarray:
    """eq. 6 on the oracle's logits: chunks [S,T] -> p [S,T-1,256] (fp64)."""
    return quantise.softmax(model.logits_for_chunks(w, chunks))


def tables(w: model.Weights, chunks: np.ndarray) -> np.ndarray:
    """Integer CDFs for every step: [S,T-1,257]."""
    return quantise.quantise(model.logits_for_chunks(w, chunks).astype(np.float32))


def ideal_bytes(C: np.ndarray, nxt: np.ndarray) -> float:
    """eq. 1 with q_t = f_t(s_t)/M:  sum_t -log256 q_t.   C [T,257], nxt [T]."""
    t = np.arange(len(nxt))
    f = (C[t, nxt.astype(np.int64) + 1] - C[t, nxt.astype(np.int64)]).astype(np.float64)
    return float(np.sum(-np.log(f / quantise.M)) / np.log(256.0))
