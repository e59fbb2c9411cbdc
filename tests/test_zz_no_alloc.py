"""The allocation-free entry point boa_rc_encode_packed_noalloc (include/boa.h): its scratch is a static device array,
not a cudaMalloc'ed workspace.  Checked against the existing path (boa_debug_rc_encode: per-stream rows + sizes, packed
here with numpy) bit for bit - integer work, so the bar is equality - on two calls in a row that share the array, the
second smaller than the first so that anything stale from the first would show.  Collected last on purpose (file name):
the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def _tables(g, S, T):
    """Valid tables: C[0] = 0, C[256] = 2^16, every frequency >= 1 (random, some rows sharply peaked)."""
    w = g.random((S, T, 256)) ** 8
    w[:, ::3, 255] += 40.0                                         # long runs of a likely symbol: carries, pending 0xFF
    f = 1 + np.floor(w / w.sum(-1, keepdims=True) * (65536 - 256)).astype(np.int64)
    f[..., 0] += 65536 - f.sum(-1)
    C = np.zeros((S, T, 257), np.int64)
    C[..., 1:] = np.cumsum(f, -1)
    assert (C[..., 256] == 65536).all() and (np.diff(C, axis=-1) >= 1).all()
    return C.astype(np.int32)


def _case(boa, seed, S, T):
    g = np.random.default_rng(seed)
    C = _tables(g, S, T)
    syms = np.where(g.random((S, T)) < 0.6, 255, g.integers(0, 256, (S, T))).astype(np.uint8)
    d_C, d_s = torch.from_numpy(C).cuda(), torch.from_numpy(syms).cuda()
    cap = 2 * T + 16
    rows, sizes = boa.debug_rc_encode(d_C, d_s, cap)               # the existing path
    rows, sizes = rows.cpu().numpy(), sizes.cpu().numpy()
    want = b"".join(rows[i, : sizes[i]].tobytes() for i in range(S))
    return d_C, d_s, sizes, want


def _run(boa, d_C, d_s, payload_cap):
    S = d_s.shape[0]
    payload = torch.full((payload_cap,), 0xEE, dtype=torch.uint8, device="cuda")
    sizes = torch.full((S,), -1, dtype=torch.int32, device="cuda")
    status = torch.full((2,), -1, dtype=torch.int64, device="cuda")
    boa.rc_encode_packed_noalloc(d_C, d_s, payload, sizes, status)  # asynchronous
    torch.cuda.synchronize()
    return payload.cpu().numpy(), sizes.cpu().numpy(), status.cpu().numpy()


def test_no_alloc_entry_point_matches_the_existing_path_on_two_calls_in_a_row(boa):
    for seed, S, T in [(11, 300, 257), (12, 37, 64)]:              # > 1 warp-scan block of streams, then a smaller call
        d_C, d_s, want_sizes, want = _case(boa, seed, S, T)
        payload, sizes, status = _run(boa, d_C, d_s, len(want) + 5)
        assert np.array_equal(sizes, want_sizes), (S, T)
        assert int(status[0]) == len(want) and int(status[1]) == 0, status
        assert payload[: len(want)].tobytes() == want, (S, T)
        assert (payload[len(want):] == 0xEE).all()                 # nothing written beyond the packed payload


def test_no_alloc_entry_point_limits_and_errors(boa):
    assert boa.noalloc_scratch_bytes() == 4 << 20
    T = 8192
    n_max = boa.noalloc_max_streams(T)
    assert 0 < n_max < 65536 and 256 + 8 * n_max + n_max * (2 * T + 8) <= 4 << 20
    d_C = torch.zeros((1, 1, 257), dtype=torch.int32, device="cuda")
    d_s = torch.zeros((n_max + 1, T), dtype=torch.uint8, device="cuda")
    out = torch.zeros(64, dtype=torch.uint8, device="cuda")
    sizes = torch.zeros(n_max + 1, dtype=torch.int32, device="cuda")
    status = torch.zeros(2, dtype=torch.int64, device="cuda")
    with pytest.raises(boa.BoaError) as e:                         # beyond the static scratch: refused before any launch
        boa.rc_encode_packed_noalloc(d_C, d_s, out, sizes, status)
    assert e.value.code == boa.E_CAPACITY and "static scratch" in str(e.value)
    with pytest.raises(boa.BoaError) as e:                         # a host pointer would need a staging allocation
        boa.rc_encode_packed_noalloc(d_C, d_s[:1, :1].contiguous(), out, sizes.cpu(), status)
    assert e.value.code == boa.E_ARG
    # payload capacity too small: reported in the status word, nothing written beyond the capacity
    d_C, d_s, want_sizes, want = _case(boa, 13, 9, 50)
    payload, sizes, status = _run(boa, d_C, d_s, len(want) - 1)
    assert int(status[1]) & 1 and int(status[0]) == len(want) and np.array_equal(sizes, want_sizes)
    keep = len(want) - int(want_sizes[-1])
    assert payload[:keep].tobytes() == want[:keep]
