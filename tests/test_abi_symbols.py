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
