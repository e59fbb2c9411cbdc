"""Pins for oracle/container.py (O4), oracle/codec.py (whole path) and the reporting formulas."""
import os
import struct
import zlib

import numpy as np
import pytest

from oracle import codec, container, model, quantise
from paper_2511_11337_b200 import metrics, synth

HERE = os.path.dirname(__file__)


def test_container_layout_by_hand():
    blob = container.pack(10, 4, 0x1122334455667788, b"abc", [b"XY", b"", b"Z"])
    assert blob[:4] == b"BOA1" and struct.unpack_from("<I", blob, 4)[0] == 1
    assert struct.unpack_from("<Q", blob, 8)[0] == 10
    assert struct.unpack_from("<IIII", blob, 16) == (4, 2, 3, 16)          # chunk, last chunk, n_chunks, freq bits
    assert struct.unpack_from("<Q", blob, 32)[0] == 0x1122334455667788
    assert blob[40:44] == b"abc\0" and struct.unpack_from("<3I", blob, 44) == (2, 0, 1)
    assert struct.unpack_from("<I", blob, 56)[0] == zlib.crc32(blob[:56])
    assert blob[60:] == b"XYZ" and container.index_bytes(3) == 60
    n, cb, last, first, pay = container.unpack(blob, 0x1122334455667788)
    assert (n, cb, last, first, pay) == (10, 4, 2, b"abc", [b"XY", b"", b"Z"])


def test_container_rejects_corruption():
    blob = bytearray(container.pack(10, 4, 7, b"abc", [b"XY", b"", b"Z"]))
    with pytest.raises(container.FormatError):
        container.unpack(bytes(blob), fingerprint=8)
    for pos in (0, 9, 17, 41, 45, 57):
        bad = bytearray(blob); bad[pos] ^= 1
        with pytest.raises(container.FormatError):
            container.unpack(bytes(bad), 7)
    with pytest.raises(container.FormatError):
        container.unpack(bytes(blob[:-1]), 7)
    empty = container.pack(0, 4096, 7, b"", [])
    assert container.unpack(empty, 7) == (0, 4096, 0, b"", []) and len(empty) == 44


@pytest.mark.parametrize("emb_std", [None, 0.25])
def test_whole_path_round_trip_and_eq1_code_length(emb_std):
    # cfg-1 shape, shortened chunks, ragged tail (3 full chunks + 1 of 77 bytes)
    cfg = synth.CONFIGS[1]
    w = model.load_weights(cfg.weights(emb_std=emb_std))
    data = cfg.data(3 * 300 + 77)
    blob = codec.compress(w, data, 300)
    assert codec.decompress(w, blob) == data                                    # Fig. 6
    n, cb, last, first, payloads = container.unpack(blob, codec.fingerprint(w))
    assert (n, cb, last) == (977, 300, 77) and first == bytes(data[i * 300] for i in range(4))
    buf = np.frombuffer(data, np.uint8)
    total_ideal = 0.0
    for i, pl in enumerate(payloads):
        chunk = buf[i * 300: min((i + 1) * 300, n)][None, :]
        C = codec.tables(w, chunk)[0]
        ideal = codec.ideal_bytes(C, chunk[0, 1:])
        total_ideal += ideal
        assert 0 < len(pl) - ideal < 5                                           # eq. 1 + 4 flush bytes
    bpb = 8 * total_ideal / (n - 4)
    if emb_std is None:
        assert abs(bpb - 8.0) < 0.01      # untrained N(0,0.02) weights predict ~uniformly
    else:
        assert bpb > 8.05                  # sharp random weights are confidently wrong: expansion is exercised


def test_edge_cases():
    cfg = synth.CONFIGS[1]
    w = model.load_weights(cfg.weights())
    for data, cb in ((b"", 16), (b"A", 16), (b"AB", 1), (b"hello world", 4), (b"x" * 33, 16)):
        blob = codec.compress(w, data, cb)
        assert codec.decompress(w, blob) == data
        _, _, _, _, payloads = container.unpack(blob)
        if cb == 1:
            assert all(len(p) == 4 for p in payloads)          # a 1-byte chunk codes zero symbols: flush only
    with pytest.raises(container.FormatError):
        other = model.load_weights(cfg.weights(emb_std=0.3))
        codec.decompress(other, codec.compress(w, b"hello world", 4))


def test_streaming_shards_by_hand():
    """Fig. 2: groups of chunks become independent shards.  Pinned by hand-assembled bytes: the shard
    boundaries are where the groups end, each shard is a container of its own group, and the chunks of a group do not
    depend on other groups (streams are independent), so a shard equals the container of the group alone."""
    cfg = synth.CONFIGS[1]
    w = model.load_weights(cfg.weights(emb_std=0.25))
    data = cfg.data(5 * 12 + 7)                       # chunks of 12 bytes, groups of 2 chunks: 3 groups, ragged tail
    shards = codec.stream_compress(w, data, 12, 2)
    assert len(shards) == 3
    for k, s in enumerate(shards):
        n, cb, last, first, payloads = container.unpack(s, codec.fingerprint(w))
        part = data[24 * k: 24 * (k + 1)]
        assert (n, cb) == (len(part), 12) and first == bytes(part[i] for i in range(0, len(part), 12))
        assert len(payloads) == -(-len(part) // 12) and last == len(part) - 12 * (len(payloads) - 1)
    # hand-split of the concatenation at the lengths the indices give
    blob = b"".join(shards)
    cut, off = [], 0
    for s in shards:
        nc = struct.unpack_from("<I", blob, off + 24)[0]          # header field n_chunks
        sizes = struct.unpack_from(f"<{nc}I", blob, off + 40 + nc + (-nc) % 4)
        ln = 40 + nc + (-nc) % 4 + 4 * nc + 4 + sum(sizes)
        cut.append(blob[off: off + ln]); off += ln
    assert off == len(blob) and cut == shards == container.split_shards(blob)
    assert codec.stream_decompress(w, blob) == data
    # the payload of a chunk is the same whether its group or the whole input is compressed
    whole = container.unpack(codec.compress(w, data, 12))[4]
    assert [p for s in shards for p in container.unpack(s)[4]] == whole
    assert codec.stream_compress(w, b"", 12, 2) == [] and codec.stream_decompress(w, b"") == b""
    with pytest.raises(container.FormatError):
        container.split_shards(blob[:-1])
    with pytest.raises(container.FormatError):
        container.split_shards(blob + b"BOA1")


def test_table1_pins_the_ssr_formula():
    ok = 0
    for line in open(os.path.join(HERE, "golden", "table1.txt")):
        if line.startswith("#") or not line.strip():
            continue
        bad = line.rstrip().endswith("!")
        name, size, comp, t, cr, ssr = [s.strip() for s in line.rstrip(" !\n").split(";")]
        size, comp, t, cr, ssr = map(float, (size, comp, t, cr, ssr))
        assert abs(metrics.compression_ratio(size, comp) - cr) < 0.015
        got = metrics.sigma_ssr(size, comp, t)
        if bad:
            assert abs(got - ssr) > 0.05
        else:
            assert abs(got - ssr) < 0.011, line      # inputs are themselves rounded to 2 decimals
            ok += 1
    assert ok == 10
    assert metrics.bits_per_byte(2044.30, 46.32) == pytest.approx(0.181, abs=1e-3)


def test_synth_configs_match_baseline_shapes():
    sizes = {1: (9728, 46080), 2: (77824, 917504), 4: (155648, 1769472), 5: (622592, 13500416)}
    for k, (st, mac) in sizes.items():           # SURVEY §8(a) per-config size table
        sh = synth.CONFIGS[k].shape
        assert sh.state_bytes_per_stream() == st and sh.mac_per_byte() == mac
    d = synth.CONFIGS[2].data(100)
    rec = np.frombuffer(d, "<f4").reshape(5, 5)
    assert np.all(rec[:, 0] > 0) and np.all(np.abs(rec[:, 1]) <= 4.5) and np.all(np.abs(rec[:, 4]) == 1.0)
    r = np.frombuffer(synth.CONFIGS[3].data(96), np.uint8).reshape(2, 48)
    assert np.all(r[0, :8] == r[1, :8]) and np.all(r[:, 40:] == 0)
    assert struct.unpack_from("<4i", r[1].tobytes(), 8) == (1, 10**6 + 1, 10**7 + 2, 10**8 + 3)
    assert synth.CONFIGS[1].data(1000) == synth.CONFIGS[1].data(2000)[:1000]
    assert len(synth.mix_bytes(3 * 65536 + 5, 9)) == 3 * 65536 + 5
