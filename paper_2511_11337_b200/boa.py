"""Thin binding over the C ABI of include/boa.h (libboa.so).  Argument marshalling only: every step
of the path runs inside the library's CUDA kernels.  Buffers are torch tensors (uint8; CUDA tensors
are used in place, CPU tensors are passed as host pointers and staged by the library).

There is no CPU fallback: importing works anywhere (the symbol table is checked), but every call
that computes raises BoaError(BOA_E_CUDA) without a usable sm_100 device.
"""
from __future__ import annotations

import ctypes as C
import os

import torch

from . import build as _build

OK = 0
E_ARG, E_FORMAT, E_CRC, E_MODEL_MISMATCH, E_CAPACITY, E_CORRUPT, E_CUDA, E_NOMEM, E_UNSUPPORTED = range(-1, -10, -1)
K_NAMES = ("embed", "inproj", "convx", "scan", "outproj", "head", "coder", "finish", "ffn1", "ffn2", "lnorm",
           "chain_in_x", "chain_out_in_x", "chain_out_head")
K_COUNT = len(K_NAMES)

EXPORTS = ("boa_model_load", "boa_model_free", "boa_model_fingerprint", "boa_compress_bound", "boa_compress",
           "boa_decompressed_size", "boa_decompress", "boa_compress_shard", "boa_container_index_bytes", "boa_container_assemble",
           "boa_decompress_shard", "boa_stream_bound", "boa_stream_compress",
           "boa_stream_decompressed_size", "boa_stream_decompress", "boa_fx_model_load", "boa_fx_model_free",
           "boa_fx_model_fingerprint", "boa_fx_compress", "boa_fx_decompress", "boa_fx_last_launches", "boa_fx_debug_step_dump",
           "boa_strerror", "boa_last_cuda_error", "boa_set_profiling", "boa_get_profile",
           "boa_debug_set_slab", "boa_debug_set_chain", "boa_debug_set_persist", "boa_debug_set_pair_tiles", "boa_debug_set_max_wave", "boa_debug_gemm", "boa_debug_step_dump", "boa_debug_quantise", "boa_debug_rc_encode", "boa_debug_rc_decode",
           "boa_noalloc_scratch_bytes", "boa_noalloc_max_streams", "boa_rc_encode_packed_noalloc")


class Profile(C.Structure):
    _fields_ = [("launches_total", C.c_uint64), ("steps", C.c_uint64), ("streams", C.c_uint64),
                ("sampled_launches", C.c_uint64 * K_COUNT), ("sampled_ms", C.c_double * K_COUNT),
                ("total_ms", C.c_double)]


class BoaError(RuntimeError):
    def __init__(self, code: int, what: str):
        detail = lib().boa_last_cuda_error().decode() if code == E_CUDA else ""
        super().__init__(f"{what}: {strerror(code)} ({code})" + (f" [{detail}]" if detail else ""))
        self.code = code


_lib = None


def lib() -> C.CDLL:
    """Load libboa.so (building it with nvcc if missing or stale).  Fails loudly if it cannot."""
    global _lib
    if _lib is not None:
        return _lib
    path = _build.LIB
    if _build.is_stale():
        have_nvcc = os.path.exists(os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc"))
        if have_nvcc or not os.path.exists(path):
            path = _build.build_library()   # raises if nvcc is missing or fails: no silent fallback
    l = C.CDLL(path)
    vp, sz, u8p = C.c_void_p, C.c_size_t, C.c_void_p
    l.boa_model_load.argtypes = [vp, sz, C.POINTER(vp)]
    l.boa_model_load.restype = C.c_int
    l.boa_model_free.argtypes = [vp]
    l.boa_model_free.restype = None
    l.boa_model_fingerprint.argtypes = [vp]
    l.boa_model_fingerprint.restype = C.c_uint64
    l.boa_compress_bound.argtypes = [sz, sz]
    l.boa_compress_bound.restype = sz
    l.boa_compress.argtypes = [vp, u8p, sz, sz, u8p, C.POINTER(sz), vp]
    l.boa_compress.restype = C.c_int
    l.boa_decompressed_size.argtypes = [u8p, sz, C.POINTER(sz)]
    l.boa_decompressed_size.restype = C.c_int
    l.boa_decompress.argtypes = [vp, u8p, sz, u8p, C.POINTER(sz), vp]
    l.boa_decompress.restype = C.c_int
    l.boa_compress_shard.argtypes = [vp, u8p, sz, sz, u8p, C.POINTER(sz), vp, vp, vp]
    l.boa_compress_shard.restype = C.c_int
    l.boa_container_index_bytes.argtypes = [sz, sz]
    l.boa_container_index_bytes.restype = sz
    l.boa_container_assemble.argtypes = [C.c_uint64, sz, sz, sz, vp, vp, vp, vp, vp, u8p, C.POINTER(sz), vp, vp]
    l.boa_container_assemble.restype = C.c_int
    l.boa_decompress_shard.argtypes = [vp, u8p, sz, sz, sz, u8p, C.POINTER(sz), vp]
    l.boa_decompress_shard.restype = C.c_int
    l.boa_stream_bound.argtypes = [sz, sz, sz]
    l.boa_stream_bound.restype = sz
    l.boa_stream_compress.argtypes = [vp, u8p, sz, sz, sz, u8p, C.POINTER(sz), vp, C.POINTER(sz), vp]
    l.boa_stream_compress.restype = C.c_int
    l.boa_stream_decompressed_size.argtypes = [u8p, sz, C.POINTER(sz), C.POINTER(sz)]
    l.boa_stream_decompressed_size.restype = C.c_int
    l.boa_stream_decompress.argtypes = [vp, u8p, sz, u8p, C.POINTER(sz), vp]
    l.boa_stream_decompress.restype = C.c_int
    l.boa_fx_model_load.argtypes = [vp, sz, C.POINTER(vp)]
    l.boa_fx_model_load.restype = C.c_int
    l.boa_fx_model_free.argtypes = [vp]
    l.boa_fx_model_free.restype = None
    l.boa_fx_model_fingerprint.argtypes = [vp]
    l.boa_fx_model_fingerprint.restype = C.c_uint64
    l.boa_fx_compress.argtypes = [vp, u8p, sz, sz, u8p, C.POINTER(sz), vp]
    l.boa_fx_compress.restype = C.c_int
    l.boa_fx_decompress.argtypes = [vp, u8p, sz, u8p, C.POINTER(sz), vp]
    l.boa_fx_decompress.restype = C.c_int
    l.boa_fx_last_launches.argtypes = [vp]
    l.boa_fx_last_launches.restype = C.c_uint64
    l.boa_fx_debug_step_dump.argtypes = [vp, u8p, sz, sz, sz, vp, vp, vp]
    l.boa_fx_debug_step_dump.restype = C.c_int
    l.boa_strerror.argtypes = [C.c_int]
    l.boa_strerror.restype = C.c_char_p
    l.boa_last_cuda_error.argtypes = []
    l.boa_last_cuda_error.restype = C.c_char_p
    l.boa_set_profiling.argtypes = [vp, C.c_int]
    l.boa_set_profiling.restype = C.c_int
    l.boa_get_profile.argtypes = [vp, C.POINTER(Profile)]
    l.boa_get_profile.restype = C.c_int
    l.boa_debug_set_slab.argtypes = [vp, C.c_int]
    l.boa_debug_set_slab.restype = C.c_int
    l.boa_debug_set_chain.argtypes = [vp, C.c_int]
    l.boa_debug_set_chain.restype = C.c_int
    l.boa_debug_set_persist.argtypes = [vp, sz, C.c_int]
    l.boa_debug_set_persist.restype = C.c_int
    l.boa_debug_set_pair_tiles.argtypes = [vp, C.c_int]
    l.boa_debug_set_pair_tiles.restype = C.c_int
    l.boa_debug_set_max_wave.argtypes = [vp, sz]
    l.boa_debug_set_max_wave.restype = C.c_int
    l.boa_debug_gemm.argtypes = [vp, sz, sz, vp, sz, C.c_int, C.c_int, vp, vp]
    l.boa_debug_gemm.restype = C.c_int
    l.boa_debug_step_dump.argtypes = [vp, u8p, sz, sz, sz, vp, vp, vp, vp]
    l.boa_debug_step_dump.restype = C.c_int
    l.boa_debug_quantise.argtypes = [vp, sz, vp, vp]
    l.boa_debug_quantise.restype = C.c_int
    l.boa_debug_rc_encode.argtypes = [vp, u8p, sz, sz, u8p, sz, vp, vp]
    l.boa_debug_rc_encode.restype = C.c_int
    l.boa_debug_rc_decode.argtypes = [vp, u8p, sz, vp, sz, sz, u8p, vp]
    l.boa_debug_rc_decode.restype = C.c_int
    l.boa_noalloc_scratch_bytes.argtypes = []
    l.boa_noalloc_scratch_bytes.restype = sz
    l.boa_noalloc_max_streams.argtypes = [sz]
    l.boa_noalloc_max_streams.restype = sz
    l.boa_rc_encode_packed_noalloc.argtypes = [vp, u8p, sz, sz, u8p, sz, vp, vp, vp]
    l.boa_rc_encode_packed_noalloc.restype = C.c_int
    _lib = l
    return l


def strerror(code: int) -> str:
    return lib().boa_strerror(code).decode()


def _check(code: int, what: str):
    if code != OK:
        raise BoaError(code, what)


def _ptr(t: torch.Tensor | None) -> int | None:
    if t is None:
        return None
    assert t.is_contiguous()
    return t.data_ptr() if t.numel() else None


def _stream(device=None) -> int:
    return torch.cuda.current_stream(device).cuda_stream if torch.cuda.is_available() else 0


def as_u8(data, device=None, pin: bool = False) -> torch.Tensor:
    """bytes / numpy / tensor -> contiguous uint8 tensor (on `device` if given)."""
    if isinstance(data, torch.Tensor):
        t = data
    else:
        t = torch.frombuffer(bytearray(data), dtype=torch.uint8) if len(data) else torch.empty(0, dtype=torch.uint8)
    t = t.contiguous().view(torch.uint8) if t.dtype != torch.uint8 else t.contiguous()
    if device is not None:
        t = t.to(device)
    elif pin and torch.cuda.is_available():
        t = t.pin_memory()
    return t


class Model:
    """boa_model handle.  `weights` is a BOAW blob (bytes)."""

    def __init__(self, weights: bytes):
        self._h = C.c_void_p()
        buf = (C.c_char * len(weights)).from_buffer_copy(weights)
        _check(lib().boa_model_load(C.cast(buf, C.c_void_p), len(weights), C.byref(self._h)), "boa_model_load")

    def close(self):
        if self._h:
            lib().boa_model_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def fingerprint(self) -> int:
        return lib().boa_model_fingerprint(self._h)

    def set_profiling(self, sample_every: int):
        _check(lib().boa_set_profiling(self._h, sample_every), "boa_set_profiling")

    def profile(self) -> dict:
        p = Profile()
        _check(lib().boa_get_profile(self._h, C.byref(p)), "boa_get_profile")
        return {"launches_total": p.launches_total, "steps": p.steps, "streams": p.streams, "total_ms": p.total_ms,
                "sampled_launches": {K_NAMES[k]: p.sampled_launches[k] for k in range(K_COUNT)},
                "sampled_ms": {K_NAMES[k]: p.sampled_ms[k] for k in range(K_COUNT)}}

    # -- the product calls ---------------------------------------------------------------------------
    def compress_into(self, src: torch.Tensor, chunk_bytes: int, dst: torch.Tensor) -> int:
        """boa_compress: src, dst uint8 tensors (each CUDA or CPU).  Returns bytes written."""
        n = C.c_size_t(dst.numel())
        _check(lib().boa_compress(self._h, _ptr(src), src.numel(), chunk_bytes, _ptr(dst), C.byref(n), _stream()),
               "boa_compress")
        return n.value

    def decompress_into(self, src: torch.Tensor, dst: torch.Tensor) -> int:
        n = C.c_size_t(dst.numel())
        _check(lib().boa_decompress(self._h, _ptr(src), src.numel(), _ptr(dst) or 0, C.byref(n), _stream()),
               "boa_decompress")
        return n.value

    def compress(self, data, chunk_bytes: int, device="cuda") -> torch.Tensor:
        src = as_u8(data, device)
        dst = torch.empty(compress_bound(src.numel(), chunk_bytes), dtype=torch.uint8, device=src.device)
        return dst[: self.compress_into(src, chunk_bytes, dst)]

    def decompress(self, blob, device="cuda") -> torch.Tensor:
        src = as_u8(blob, device)
        dst = torch.empty(decompressed_size(src), dtype=torch.uint8, device=src.device)
        self.decompress_into(src, dst)
        return dst

    # -- one container from several GPUs ---------------------------------------------------
    def compress_shard(self, src: torch.Tensor, chunk_bytes: int, payload: torch.Tensor):
        """boa_compress_shard: src = the bytes of a contiguous chunk range (CUDA or CPU), payload = uint8 buffer (CUDA or
        CPU).  Returns (payload bytes written, sizes [chunks] int32 CPU tensor, first [chunks] uint8 CPU tensor)."""
        nc = -(-src.numel() // chunk_bytes) if src.numel() else 0
        sizes = torch.zeros(max(nc, 1), dtype=torch.int32)
        first = torch.zeros(max(nc, 1), dtype=torch.uint8)
        n = C.c_size_t(payload.numel())
        _check(lib().boa_compress_shard(self._h, _ptr(src), src.numel(), chunk_bytes, _ptr(payload) or 0, C.byref(n),
                                        sizes.data_ptr(), first.data_ptr(), _stream()), "boa_compress_shard")
        return n.value, sizes[:nc], first[:nc]

    def container_assemble(self, n: int, chunk_bytes: int, parts, out: torch.Tensor, payloads=None):
        return container_assemble(self.fingerprint, n, chunk_bytes, parts, out, payloads)

    def decompress_shard(self, src: torch.Tensor, first_chunk: int, n_chunks: int, dst: torch.Tensor) -> int:
        n = C.c_size_t(dst.numel())
        _check(lib().boa_decompress_shard(self._h, _ptr(src), src.numel(), first_chunk, n_chunks, _ptr(dst) or 0, C.byref(n),
                                          _stream()), "boa_decompress_shard")
        return n.value

    # -- streaming front end (Fig. 2): host buffers in, concatenated shards out --------------------------
    def stream_compress(self, data, chunk_bytes: int, group_chunks: int):
        """boa_stream_compress: returns (CPU uint8 tensor of the concatenated shards, list of shard lengths)."""
        src = as_u8(data)
        dst = torch.empty(stream_bound(src.numel(), chunk_bytes, group_chunks), dtype=torch.uint8)
        groups = -(-src.numel() // (chunk_bytes * group_chunks)) if src.numel() else 0
        lens = (C.c_uint64 * max(groups, 1))()
        n, ns = C.c_size_t(dst.numel()), C.c_size_t(groups)
        _check(lib().boa_stream_compress(self._h, _ptr(src), src.numel(), chunk_bytes, group_chunks, _ptr(dst), C.byref(n),
                                         C.cast(lens, C.c_void_p), C.byref(ns), _stream()), "boa_stream_compress")
        return dst[: n.value], [int(lens[i]) for i in range(ns.value)]

    def stream_decompress(self, blob) -> torch.Tensor:
        src = as_u8(blob)
        total, ns = C.c_size_t(0), C.c_size_t(0)
        _check(lib().boa_stream_decompressed_size(_ptr(src), src.numel(), C.byref(total), C.byref(ns)),
               "boa_stream_decompressed_size")
        dst = torch.empty(total.value, dtype=torch.uint8)
        n = C.c_size_t(dst.numel())
        _check(lib().boa_stream_decompress(self._h, _ptr(src), src.numel(), _ptr(dst) or 0, C.byref(n), _stream()),
               "boa_stream_decompress")
        return dst

    # -- test-only -----------------------------------------------------------------------------------
    def debug_set_slab(self, enabled: bool):
        _check(lib().boa_debug_set_slab(self._h, 1 if enabled else 0), "boa_debug_set_slab")

    def debug_set_chain(self, enabled: bool):
        _check(lib().boa_debug_set_chain(self._h, 1 if enabled else 0), "boa_debug_set_chain")

    def debug_set_persist(self, max_streams: int, cluster_ctas: int = 0):
        _check(lib().boa_debug_set_persist(self._h, max_streams, cluster_ctas), "boa_debug_set_persist")

    def debug_set_pair_tiles(self, min_row_tiles: int):
        _check(lib().boa_debug_set_pair_tiles(self._h, min_row_tiles), "boa_debug_set_pair_tiles")

    def debug_set_max_wave(self, streams: int):
        _check(lib().boa_debug_set_max_wave(self._h, streams), "boa_debug_set_max_wave")

    def debug_step_dump(self, data, chunk_bytes: int, n_steps: int, want=("logits", "probs", "cdf"), device="cuda"):
        src = as_u8(data, device)
        rows = (src.numel() // chunk_bytes) * n_steps
        out = {}
        if "logits" in want:
            out["logits"] = torch.empty((rows, 256), dtype=torch.float32, device=device)
        if "probs" in want:
            out["probs"] = torch.empty((rows, 256), dtype=torch.float32, device=device)
        if "cdf" in want:
            out["cdf"] = torch.empty((rows, 257), dtype=torch.int32, device=device)
        _check(lib().boa_debug_step_dump(self._h, _ptr(src), src.numel(), chunk_bytes, n_steps, _ptr(out.get("logits")),
                                         _ptr(out.get("probs")), _ptr(out.get("cdf")), _stream()), "boa_debug_step_dump")
        b = src.numel() // chunk_bytes
        return {k: v.view(b, n_steps, -1) for k, v in out.items()}


def stream_bound(n: int, chunk_bytes: int, group_chunks: int) -> int:
    return lib().boa_stream_bound(n, chunk_bytes, group_chunks)


class FxModel:
    """boa_fx_model handle: FX1, the deterministic fixed-point pipeline.  `weights` is a BOAW blob."""

    def __init__(self, weights: bytes):
        self._h = C.c_void_p()
        buf = (C.c_char * len(weights)).from_buffer_copy(weights)
        _check(lib().boa_fx_model_load(C.cast(buf, C.c_void_p), len(weights), C.byref(self._h)), "boa_fx_model_load")

    def close(self):
        if self._h:
            lib().boa_fx_model_free(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def fingerprint(self) -> int:
        return lib().boa_fx_model_fingerprint(self._h)

    @property
    def last_launches(self) -> int:
        return lib().boa_fx_last_launches(self._h)

    def compress_into(self, src: torch.Tensor, chunk_bytes: int, dst: torch.Tensor) -> int:
        n = C.c_size_t(dst.numel())
        _check(lib().boa_fx_compress(self._h, _ptr(src), src.numel(), chunk_bytes, _ptr(dst), C.byref(n), _stream()), "boa_fx_compress")
        return n.value

    def decompress_into(self, src: torch.Tensor, dst: torch.Tensor) -> int:
        n = C.c_size_t(dst.numel())
        _check(lib().boa_fx_decompress(self._h, _ptr(src), src.numel(), _ptr(dst) or 0, C.byref(n), _stream()), "boa_fx_decompress")
        return n.value

    def compress(self, data, chunk_bytes: int, device="cuda") -> torch.Tensor:
        src = as_u8(data, device)
        dst = torch.empty(compress_bound(src.numel(), chunk_bytes), dtype=torch.uint8, device=src.device)
        return dst[: self.compress_into(src, chunk_bytes, dst)]

    def decompress(self, blob, device="cuda") -> torch.Tensor:
        src = as_u8(blob, device)
        dst = torch.empty(decompressed_size(src), dtype=torch.uint8, device=src.device)
        self.decompress_into(src, dst)
        return dst

    def debug_step_dump(self, data, chunk_bytes: int, n_steps: int, device="cuda"):
        src = as_u8(data, device)
        b = src.numel() // chunk_bytes
        logits = torch.empty((b * n_steps, 256), dtype=torch.int32, device=device)
        cdf = torch.empty((b * n_steps, 257), dtype=torch.int32, device=device)
        _check(lib().boa_fx_debug_step_dump(self._h, _ptr(src), src.numel(), chunk_bytes, n_steps, _ptr(logits), _ptr(cdf), _stream()),
               "boa_fx_debug_step_dump")
        return {"logits": logits.view(b, n_steps, 256), "cdf": cdf.view(b, n_steps, 257)}


def container_assemble(fingerprint: int, n: int, chunk_bytes: int, parts, out: torch.Tensor, payloads=None):
    """boa_container_assemble: parts = [(sizes int32 CPU tensor, first uint8 CPU tensor), ...] in chunk order;
    payloads = matching list of uint8 tensors (CUDA or CPU) or None (index only).  Returns (bytes written, offsets).
    Host-only when every tensor is a CPU tensor (no GPU needed)."""
    k = len(parts)
    sizes = [p[0].contiguous() for p in parts]
    first = [p[1].contiguous() for p in parts]
    counts = (C.c_size_t * max(k, 1))(*[int(z.numel()) for z in sizes])
    fp = (C.c_void_p * max(k, 1))(*[f.data_ptr() if f.numel() else None for f in first])
    zp = (C.c_void_p * max(k, 1))(*[z.data_ptr() if z.numel() else None for z in sizes])
    offs = (C.c_uint64 * (k + 1))()
    pp = pl = None
    if payloads is not None:
        pp = (C.c_void_p * max(k, 1))(*[_ptr(p) for p in payloads])
        pl = (C.c_size_t * max(k, 1))(*[int(p.numel()) for p in payloads])
    ln = C.c_size_t(out.numel())
    _check(lib().boa_container_assemble(fingerprint, n, chunk_bytes, k, C.cast(counts, C.c_void_p), C.cast(fp, C.c_void_p),
                                        C.cast(zp, C.c_void_p), C.cast(pp, C.c_void_p) if pp is not None else None,
                                        C.cast(pl, C.c_void_p) if pl is not None else None, _ptr(out), C.byref(ln),
                                        C.cast(offs, C.c_void_p), _stream() if out.is_cuda else 0), "boa_container_assemble")
    return ln.value, [int(o) for o in offs]


def container_index_bytes(n: int, chunk_bytes: int) -> int:
    return lib().boa_container_index_bytes(n, chunk_bytes)


def compress_bound(n: int, chunk_bytes: int) -> int:
    return lib().boa_compress_bound(n, chunk_bytes)


def decompressed_size(blob: torch.Tensor) -> int:
    n = C.c_size_t(0)
    _check(lib().boa_decompressed_size(_ptr(blob) or 0, blob.numel(), C.byref(n)), "boa_decompressed_size")
    return n.value


def debug_gemm(a: torch.Tensor, w: torch.Tensor, weight_pieces: int, grid_ctas: int = 0) -> torch.Tensor:
    """a [M,K] fp32 (CUDA or CPU), w [N,K] fp32 CPU -> a @ w.T [M,N] fp32 on a's device, by the tensor-core kernel."""
    a = a.contiguous()
    w = w.contiguous().cpu()
    c = torch.empty((a.shape[0], w.shape[0]), dtype=torch.float32, device=a.device)
    _check(lib().boa_debug_gemm(_ptr(a), a.shape[0], a.shape[1], _ptr(w), w.shape[0], weight_pieces, grid_ctas, _ptr(c),
                                _stream()), "boa_debug_gemm")
    return c


def debug_quantise(logits: torch.Tensor) -> torch.Tensor:
    """logits [rows,256] fp32 (CUDA or CPU) -> cdf [rows,257] int32 on the same device."""
    logits = logits.contiguous()
    cdf = torch.empty((logits.shape[0], 257), dtype=torch.int32, device=logits.device)
    _check(lib().boa_debug_quantise(_ptr(logits), logits.shape[0], _ptr(cdf), _stream()), "boa_debug_quantise")
    return cdf


def debug_rc_encode(cdf: torch.Tensor, syms: torch.Tensor, cap: int):
    """cdf [S,len,257] int32, syms [S,len] uint8 -> (out [S,cap] uint8, sizes [S] int32)."""
    s, ln = syms.shape
    out = torch.zeros((s, cap), dtype=torch.uint8, device=syms.device)
    sizes = torch.zeros(s, dtype=torch.int32, device=syms.device)
    _check(lib().boa_debug_rc_encode(_ptr(cdf.contiguous()), _ptr(syms.contiguous()), s, ln, _ptr(out), cap, _ptr(sizes),
                                     _stream()), "boa_debug_rc_encode")
    return out, sizes


def debug_rc_decode(cdf: torch.Tensor, payload: torch.Tensor, sizes: torch.Tensor, length: int) -> torch.Tensor:
    s, cap = payload.shape
    syms = torch.zeros((s, length), dtype=torch.uint8, device=payload.device)
    _check(lib().boa_debug_rc_decode(_ptr(cdf.contiguous()), _ptr(payload.contiguous()), cap, _ptr(sizes.contiguous()),
                                     s, length, _ptr(syms), _stream()), "boa_debug_rc_decode")
    return syms


def noalloc_scratch_bytes() -> int:
    return lib().boa_noalloc_scratch_bytes()


def noalloc_max_streams(length: int) -> int:
    return lib().boa_noalloc_max_streams(length)


def rc_encode_packed_noalloc(cdf: torch.Tensor, syms: torch.Tensor, payload: torch.Tensor, sizes: torch.Tensor,
                             status: torch.Tensor) -> None:
    """The allocation-free entry point (include/boa.h): cdf [S,len,257] int32, syms [S,len] uint8 -> payload (packed),
    sizes [S] int32, status [2] int64, all CUDA tensors the CALLER provides.  Asynchronous on torch's current stream."""
    s, ln = syms.shape
    code = lib().boa_rc_encode_packed_noalloc(_ptr(cdf), _ptr(syms), s, ln, _ptr(payload), payload.numel(), _ptr(sizes),
                                              _ptr(status), _stream())
    if code == E_CAPACITY:
        raise BoaError(code, "boa_rc_encode_packed_noalloc: " + lib().boa_last_cuda_error().decode())
    _check(code, "boa_rc_encode_packed_noalloc")
