"""Seeded synthetic inputs: model weights (BOAW blobs) and byte workloads.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds
none of the method's arithmetic (no model step, no quantiser, no coder): only
random initialisation, the BOAW serialisation, and the byte generators for the
five BASELINE.json configs (recipes: SURVEY.md §8(d); readings #12-#14 in
DESIGN.md).  It needs numpy only.

The paper's CERN files (PAPER.md "Dataset") and trained weights are
not available; these generators stand in for them (HEP-like float32 columns for
ATLAS / bundled CMS, fixed-width zero-padded records for the padded CMS file).
"""
from __future__ import annotations

import struct
from dataclasses import dataclass

import numpy as np

BOAW_MAGIC = b"BOAW"
BOAW_VERSION = 1
BOAW_HEADER_BYTES = 64
DTYPE_FP32 = 0
DTYPE_BF16 = 1
FLAG_TIED_HEAD = 1   # head = Emb^T (north_star's block); clear = a separate head matrix after the layers
FLAG_FFN = 2         # every layer is followed by u <- LayerNorm(FFN(u)) (Alg. 1 l.4)


@dataclass(frozen=True)
class ModelShape:
    n_layer: int
    d_model: int
    d_state: int = 16
    d_conv: int = 4
    expand: int = 2
    dt_rank: int = 0  # 0 -> ceil(d_model / 16)
    d_ff: int = 0     # > 0: the paper's block (Alg. 1 l.4): FFN of this hidden width + LayerNorm after every mixer
    tied: bool = True # False: untied head matrix [256, D]

    @property
    def d_inner(self) -> int:
        return self.expand * self.d_model

    @property
    def rank(self) -> int:
        return self.dt_rank if self.dt_rank else -(-self.d_model // 16)

    def state_bytes_per_stream(self) -> int:
        """fp32 SSM state + conv window per stream (SURVEY §8(a) size table)."""
        e = self.d_inner
        return self.n_layer * (4 * e * self.d_state + 4 * e * (self.d_conv - 1))

    def mac_per_byte(self) -> int:
        d, e, r, n = self.d_model, self.d_inner, self.rank, self.d_state
        return self.n_layer * (d * 2 * e + e * (r + 2 * n) + r * e + e * d + 2 * d * self.d_ff) + 256 * d

    @property
    def flags(self) -> int:
        return (FLAG_TIED_HEAD if self.tied else 0) | (FLAG_FFN if self.d_ff else 0)


def _to_bf16_bits(a32: np.ndarray) -> np.ndarray:
    """Round fp32 to bf16 (round-to-nearest-even), returned as uint16 bit patterns."""
    u = np.ascontiguousarray(a32, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = (u + 0x7FFF + ((u >> 16) & 1)) >> 16
    return r.astype(np.uint16)


def bf16_bits_to_f32(bits: np.ndarray) -> np.ndarray:
    return (bits.astype(np.uint32) << 16).view(np.float32)


def _pad16(b: bytes) -> bytes:
    return b + b"\0" * ((-len(b)) % 16)


def tensor_order(shape: ModelShape):
    """(name, dims, is_matrix) in blob order.  Matrices are stored as bf16 when dtype=1."""
    d, e, n, k, r = shape.d_model, shape.d_inner, shape.d_state, shape.d_conv, shape.rank
    out = [("emb", (256, d), True)]
    for l in range(shape.n_layer):
        p = f"l{l}."
        out += [
            (p + "norm_w", (d,), False),
            (p + "w_in", (2 * e, d), True),
            (p + "conv_w", (e, k), False),
            (p + "conv_b", (e,), False),
            (p + "w_x", (r + 2 * n, e), True),
            (p + "w_dt", (e, r), True),
            (p + "b_dt", (e,), False),
            (p + "a_log", (e, n), False),
            (p + "d_skip", (e,), False),
            (p + "w_out", (d, e), True),
        ]
        if shape.d_ff:
            f = shape.d_ff
            out += [
                (p + "ffn_w1", (f, d), True),
                (p + "ffn_b1", (f,), False),
                (p + "ffn_w2", (d, f), True),
                (p + "ffn_b2", (d,), False),
                (p + "ln_w", (d,), False),
                (p + "ln_b", (d,), False),
            ]
    if not shape.tied:
        out.append(("head", (256, d), True))
    return out


def make_weights(shape: ModelShape, seed: int, dtype: int = DTYPE_FP32,
                 std: float = 0.02, emb_std: float | None = None, ffn_std: float | None = None) -> bytes:
    """Random-init BOAW blob.  Draw order = blob order, fp64 draws -> fp32 (-> bf16 for matrices).

    All matrices incl. emb and conv_w ~ N(0, std^2); norm_w = 1; conv_b = 0; d_skip = 1;
    a_log[e][n] = log(n+1); b_dt = softplus^-1(dt), dt = exp(U(log 1e-3, log 1e-1)).
    `emb_std` (e.g. 0.25) gives the "sharp" variant used to stress the quantiser and coder.
    FFN variant (shape.d_ff > 0): ffn_w1, ffn_w2 ~ N(0, ffn_std^2) (default std); the FFN biases and ln_b
    ~ N(0, std^2) and ln_w = 1 + N(0, std^2), so that a dropped bias or affine term changes the result;
    untied head ~ N(0, emb_std^2).
    """
    g = np.random.Generator(np.random.PCG64(seed))
    emb_std = std if emb_std is None else emb_std
    hdr = struct.pack("<4s10I", BOAW_MAGIC, BOAW_VERSION, dtype, shape.n_layer, shape.d_model,
                      shape.d_state, shape.d_conv, shape.expand, shape.rank, shape.flags, shape.d_ff)
    parts = [hdr + b"\0" * (BOAW_HEADER_BYTES - len(hdr))]
    for name, dims, is_mat in tensor_order(shape):
        base = name.split(".")[-1]
        if base == "emb" or base == "head":
            a = g.normal(0.0, emb_std, dims)
        elif base in ("w_in", "w_x", "w_dt", "w_out", "conv_w"):
            a = g.normal(0.0, std, dims)
        elif base in ("ffn_w1", "ffn_w2"):
            a = g.normal(0.0, ffn_std if ffn_std is not None else std, dims)
        elif base in ("ffn_b1", "ffn_b2", "ln_b"):
            a = g.normal(0.0, std, dims)
        elif base == "ln_w":
            a = 1.0 + g.normal(0.0, std, dims)
        elif base == "norm_w" or base == "d_skip":
            a = np.ones(dims)
        elif base == "conv_b":
            a = np.zeros(dims)
        elif base == "b_dt":
            dt = np.exp(g.uniform(np.log(1e-3), np.log(1e-1), dims))
            a = dt + np.log(-np.expm1(-dt))
        elif base == "a_log":
            a = np.broadcast_to(np.log(np.arange(1, dims[1] + 1, dtype=np.float64)), dims)
        else:  # pragma: no cover
            raise AssertionError(name)
        a32 = np.ascontiguousarray(a, dtype=np.float32)
        if is_mat and dtype == DTYPE_BF16:
            parts.append(_pad16(_to_bf16_bits(a32).tobytes()))
        else:
            parts.append(_pad16(a32.tobytes()))
    return b"".join(parts)


def parse_header(blob: bytes):
    magic, ver, dtype, nl, d, n, k, ex, r, flags, d_ff = struct.unpack_from("<4s10I", blob, 0)
    if magic != BOAW_MAGIC or ver != BOAW_VERSION:
        raise ValueError("not a BOAW v1 blob")
    return ModelShape(nl, d, n, k, ex, r, d_ff if flags & FLAG_FFN else 0, bool(flags & FLAG_TIED_HEAD)), dtype, flags


# --------------------------------------------------------------------------- byte workloads

def markov_bytes(n: int, seed: int) -> bytes:
    """cfg 1: order-1 Markov source, each of the 256 rows ~ Dirichlet(0.1)."""
    g = np.random.Generator(np.random.PCG64(seed))
    P = g.dirichlet(np.full(256, 0.1), size=256)
    s = int(g.integers(256))
    u = g.random(n)
    cdf = np.cumsum(P, axis=1)
    out = np.empty(n, dtype=np.uint8)
    for i in range(n):
        s = min(int(np.searchsorted(cdf[s], u[i], side="right")), 255)
        out[i] = s
    return out.tobytes()


def kinematics_bytes(n: int, seed: int) -> bytes:
    """cfg 2 / 4: 20-byte records of 5 little-endian float32 (pt, eta, phi, mass, charge)."""
    g = np.random.Generator(np.random.PCG64(seed))
    n_rec = -(-n // 20)
    pt = g.exponential(30.0, n_rec)
    eta = np.clip(g.normal(0.0, 1.5, n_rec), -4.5, 4.5)
    phi = g.uniform(-np.pi, np.pi, n_rec)
    mass = np.abs(g.normal(0.1, 0.05, n_rec))
    charge = g.choice(np.array([-1.0, 1.0]), n_rec)
    rec = np.stack([pt, eta, phi, mass, charge], axis=1).astype("<f4")
    return rec.tobytes()[:n]


def records_bytes(n: int, seed: int) -> bytes:
    """cfg 3: 48-byte records: 8 constant bytes, 4 int32 counters, 4 float32 from a 16-value
    Zipf(1.2)-weighted set quantised to 1e-2, 8 zero bytes."""
    g = np.random.Generator(np.random.PCG64(seed))
    n_rec = -(-n // 48)
    header = g.integers(256, size=8).astype(np.uint8)
    values = np.round(np.sort(g.uniform(0.0, 100.0, 16)), 2)
    w = 1.0 / np.arange(1, 17) ** 1.2
    w /= w.sum()
    idx = g.choice(16, size=(n_rec, 4), p=w)
    rec = np.zeros((n_rec, 48), dtype=np.uint8)
    rec[:, 0:8] = header
    r = np.arange(n_rec, dtype=np.int64)
    bases = (0, 10**6, 10**7, 10**8)
    steps = (1, 1, 2, 3)
    ctr = np.stack([b + r * s for b, s in zip(bases, steps)], axis=1).astype("<i4")
    rec[:, 8:24] = ctr.view(np.uint8).reshape(n_rec, 16)
    rec[:, 24:40] = values[idx].astype("<f4").view(np.uint8).reshape(n_rec, 16)
    return rec.tobytes()[:n]


def mix_bytes(n: int, seed: int, chunk: int = 65536) -> bytes:
    """cfg 5: chunks alternate kinematics (even ids) and records (odd ids)."""
    half = -(-n // 2)
    a = np.frombuffer(kinematics_bytes(half + chunk, seed), dtype=np.uint8)
    b = np.frombuffer(records_bytes(half + chunk, seed + 1), dtype=np.uint8)
    n_chunks = -(-n // chunk)
    out = np.empty(n_chunks * chunk, dtype=np.uint8)
    view = out.reshape(n_chunks, chunk)
    ne, no = (n_chunks + 1) // 2, n_chunks // 2
    view[0::2] = a[: ne * chunk].reshape(ne, chunk)
    view[1::2] = b[: no * chunk].reshape(no, chunk)
    return out.tobytes()[:n]


@dataclass(frozen=True)
class Config:
    name: str
    shape: ModelShape
    weight_dtype: int
    model_seed: int
    data_seed: int
    n_bytes: int
    chunk_bytes: int
    generator: str

    def weights(self, **kw) -> bytes:
        return make_weights(self.shape, self.model_seed, self.weight_dtype, **kw)

    def data(self, n: int | None = None) -> bytes:
        n = self.n_bytes if n is None else n
        fn = {"markov": markov_bytes, "kinematics": kinematics_bytes,
              "records": records_bytes, "mix": mix_bytes}[self.generator]
        return fn(n, self.data_seed)


MiB = 1 << 20
CONFIGS = {
    # BASELINE.json configs[0..4]; seeds per DESIGN.md reading #14
    1: Config("cfg1_tiny_markov", ModelShape(1, 64, dt_rank=4), DTYPE_FP32, 0, 1001, 64 * 1024, 4096, "markov"),
    2: Config("cfg2_kinematics_64MiB", ModelShape(2, 256, dt_rank=16), DTYPE_FP32, 1, 1002, 64 * MiB, 16384, "kinematics"),
    3: Config("cfg3_records_256MiB", ModelShape(2, 256, dt_rank=16), DTYPE_FP32, 1, 1003, 256 * MiB, 16384, "records"),
    4: Config("cfg4_kinematics_1GiB", ModelShape(4, 256, dt_rank=16), DTYPE_BF16, 2, 1004, 1024 * MiB, 16384, "kinematics"),
    5: Config("cfg5_mix_512MiB", ModelShape(8, 512, dt_rank=32), DTYPE_BF16, 3, 1005, 512 * MiB, 65536, "mix"),
    # not a BASELINE.json config: the paper's own block (d_m = 256, n_l = 1, FFN +
    # LayerNorm after the mixer, untied head, ~4.4 MB of fp32 weights) on the input of config 2
    6: Config("next2_paper_block_64MiB", ModelShape(1, 256, dt_rank=16, d_ff=1024, tied=False), DTYPE_FP32, 4, 1002,
              64 * MiB, 16384, "kinematics"),
}
