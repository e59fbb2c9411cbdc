"""CPU-side checks of the boundary: libboa.so builds, loads and exports every symbol include/boa.h declares;
host-only entry points behave; nothing in the product package imports the oracle."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "boa.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(boa_[a-z_0-9]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(boa):
    lib = boa.lib()
    names = _declared_symbols()
    assert len(names) >= 14 and set(boa.EXPORTS) == set(names)
    for n in names:
        assert hasattr(lib, n), n


def test_host_only_entry_points(boa):
    lib = boa.lib()
    assert boa.strerror(0) == "ok" and "CRC" in boa.strerror(boa.E_CRC)
    # bound = index + 2 bytes/symbol + 4 flush bytes per stream
    assert boa.compress_bound(0, 4096) == 44
    assert boa.compress_bound(10, 4) == 40 + 4 + 12 + 4 + 20 + 12
    assert lib.boa_compress(None, None, 0, 0, None, None, None) == boa.E_ARG
    n = ctypes.c_size_t()
    buf = ctypes.create_string_buffer(b"XXXX" + b"\0" * 60)
    assert lib.boa_decompressed_size(ctypes.cast(buf, ctypes.c_void_p), 64, ctypes.byref(n)) == boa.E_FORMAT


def test_streaming_host_only_entry_points(boa):
    """boa_stream_bound and boa_stream_decompressed_size work on host memory only (Fig. 2 shards)."""
    import struct
    import zlib
    lib = boa.lib()
    # 10 bytes in chunks of 4, groups of 2 chunks: shards of 8 and 2 bytes
    assert boa.stream_bound(10, 4, 2) == boa.compress_bound(8, 4) + boa.compress_bound(2, 4)
    assert boa.stream_bound(16, 4, 2) == 2 * boa.compress_bound(8, 4) and boa.stream_bound(0, 4, 2) == 0
    # two hand-assembled shards (BOA1 header, first bytes, sizes, CRC, payload): 5 bytes in one chunk, then 1 byte
    def shard(n, payload):
        head = struct.pack("<4sIQIIIIQ", b"BOA1", 1, n, 8, n, 1, 16, 0x1234) + b"A\0\0\0" + struct.pack("<I", len(payload))
        return head + struct.pack("<I", zlib.crc32(head) & 0xFFFFFFFF) + payload
    blob = shard(5, b"\x01\x02\x03\x04\x05\x06") + shard(1, b"\0\0\0\0")
    buf = ctypes.create_string_buffer(blob, len(blob))
    n, ns = ctypes.c_size_t(), ctypes.c_size_t()
    assert lib.boa_stream_decompressed_size(ctypes.cast(buf, ctypes.c_void_p), len(blob), ctypes.byref(n), ctypes.byref(ns)) == 0
    assert (n.value, ns.value) == (6, 2)
    assert lib.boa_stream_decompressed_size(ctypes.cast(buf, ctypes.c_void_p), len(blob) - 1, ctypes.byref(n), ctypes.byref(ns)) == boa.E_FORMAT
    assert lib.boa_stream_decompressed_size(None, 0, ctypes.byref(n), ctypes.byref(ns)) == 0 and n.value == 0 and ns.value == 0
    assert lib.boa_stream_compress(None, None, 0, 0, 0, None, None, None, None, None) == boa.E_ARG


def test_model_load_rejects_bad_blobs_before_touching_the_gpu(boa):
    with pytest.raises(boa.BoaError) as e:
        boa.Model(b"NOPE" + b"\0" * 100)
    assert e.value.code == boa.E_FORMAT
    from paper_2511_11337_b200 import synth
    blob = bytearray(synth.make_weights(synth.ModelShape(1, 64, dt_rank=4), 0))
    blob[20] = 8  # d_state = 8: not what the kernels are built for
    with pytest.raises(boa.BoaError) as e:
        boa.Model(bytes(blob))
    assert e.value.code == boa.E_UNSUPPORTED


def test_product_package_never_imports_the_oracle():
    pkg = os.path.join(ROOT, "paper_2511_11337_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert not re.search(r"^\s*(from|import)\s+oracle\b", txt, flags=re.M), f
                assert not re.search(r'#include\s*[<"][^>"]*oracle', txt), f
