"""O1 — the byte-level autoregressive Mamba-1 step function, fp64 (oracle; test infrastructure).

Follows PAPER.md step by step:
  * step function / stream state   P:68-76, eq. 4-5   (S_{t+1}, l_{t+1}) = Phi(S_t, s_t)
  * forward pass                    P:134-148, Alg. 1  embed -> blocks -> head
  * discretisation A_bar=exp(dA)    P:361, eq. 16
  * recurrence h=A_bar h + B_bar x  P:367-369, eq. 18-19
  * selection d=softplus(W x + b)   P:375-380, eq. 20-22
Readings: block = pre-RMSNorm -> mixer -> residual, no FFN (#1); no final norm (#2);
B_bar = d*B (#3); no bias on B_t, C_t (#4); eps=1e-5, stable softplus, SiLU=x*sigmoid(x) (#10);
conv tap K-1 multiplies the current input (#11).
The paper's own block (blobs with FLAG_FFN): after the mixer and its residual,
u <- LayerNorm(FFN(u)) as Alg. 1 l.4 writes it - no residual around the FFN;
FFN(u) = W2 GELU(W1 u + b1) + b2 with GELU(v) = v Phi(v) (erf form); LayerNorm over the D features with the
biased variance, eps = 1e-5, affine (ln_w, ln_b); head untied when FLAG_TIED_HEAD is clear (#23).

Streams are independent; every function below takes a leading "stream" axis S and
treats the S rows independently — that axis is the only vectorisation.
"""
from __future__ import annotations

import struct
from dataclasses import dataclass, field

import numpy as np

EPS = 1e-5


@dataclass
class Layer:
    norm_w: np.ndarray   # [D]
    w_in: np.ndarray     # [2E, D]
    conv_w: np.ndarray   # [E, K]
    conv_b: np.ndarray   # [E]
    w_x: np.ndarray      # [R+2N, E]
    w_dt: np.ndarray     # [E, R]
    b_dt: np.ndarray     # [E]
    a_log: np.ndarray    # [E, N]
    d_skip: np.ndarray   # [E]
    w_out: np.ndarray    # [D, E]
    # the paper's block only (FLAG_FFN), else None
    ffn_w1: np.ndarray = None   # [F, D]
    ffn_b1: np.ndarray = None   # [F]
    ffn_w2: np.ndarray = None   # [D, F]
    ffn_b2: np.ndarray = None   # [D]
    ln_w: np.ndarray = None     # [D]
    ln_b: np.ndarray = None     # [D]


@dataclass
class Weights:
    n_layer: int
    d_model: int
    d_state: int
    d_conv: int
    expand: int
    dt_rank: int
    emb: np.ndarray                      # [256, D]  (also the tied head)
    layers: list = field(default_factory=list)
    blob_crc: int = 0
    d_ff: int = 0                        # > 0: FFN + LayerNorm after every mixer
    head: np.ndarray = None              # [256, D] untied head, None = tied (Emb)

    @property
    def d_inner(self) -> int:
        return self.expand * self.d_model


def load_weights(blob: bytes) -> Weights:
    """Parse a BOAW v1 blob; stored fp32 / bf16 values are widened to fp64 exactly."""
    import zlib
    magic, ver, dtype, nl, d, n, k, ex, r, flags, f = struct.unpack_from("<4s10I", blob, 0)
    if magic != b"BOAW" or ver != 1:
        raise ValueError("not a BOAW v1 blob")
    if flags & ~3 or bool(flags & 2) != (f > 0):
        raise ValueError("bad BOAW flags")
    e = ex * d
    off = 64

    def take(shape, is_matrix):
        nonlocal off
        cnt = int(np.prod(shape))
        if is_matrix and dtype == 1:
            raw = np.frombuffer(blob, dtype="<u2", count=cnt, offset=off)
            arr = (raw.astype(np.uint32) << 16).view(np.float32).astype(np.float64)
            nbytes = 2 * cnt
        else:
            arr = np.frombuffer(blob, dtype="<f4", count=cnt, offset=off).astype(np.float64)
            nbytes = 4 * cnt
        off += nbytes + ((-nbytes) % 16)
        return arr.reshape(shape)

    w = Weights(nl, d, n, k, ex, r, emb=take((256, d), True), blob_crc=zlib.crc32(blob) & 0xFFFFFFFF)
    w.d_ff = f
    for _ in range(nl):
        ly = Layer(
            norm_w=take((d,), False), w_in=take((2 * e, d), True), conv_w=take((e, k), False),
            conv_b=take((e,), False), w_x=take((r + 2 * n, e), True), w_dt=take((e, r), True),
            b_dt=take((e,), False), a_log=take((e, n), False), d_skip=take((e,), False),
            w_out=take((d, e), True))
        if f:
            ly.ffn_w1 = take((f, d), True)
            ly.ffn_b1 = take((f,), False)
            ly.ffn_w2 = take((d, f), True)
            ly.ffn_b2 = take((d,), False)
            ly.ln_w = take((d,), False)
            ly.ln_b = take((d,), False)
        w.layers.append(ly)
    if not (flags & 1):
        w.head = take((256, d), True)
    if off != len(blob):
        raise ValueError("BOAW blob has trailing or missing bytes")
    return w


def sigmoid(x):
    return 1.0 / (1.0 + np.exp(-x))


def silu(x):
    return x * sigmoid(x)


def softplus(v):
    """log(1+exp(v)) in the overflow-free form max(v,0)+log1p(exp(-|v|))  (eq. 20)."""
    return np.maximum(v, 0.0) + np.log1p(np.exp(-np.abs(v)))


def rmsnorm(u, w):
    return u * (1.0 / np.sqrt(np.mean(u * u, axis=-1, keepdims=True) + EPS)) * w


_erf = np.vectorize(__import__("math").erf, otypes=[np.float64])


def gelu(v):
    """GELU(v) = v Phi(v) = v (1 + erf(v / sqrt 2)) / 2, Phi the standard normal CDF (reading #23)."""
    return 0.5 * v * (1.0 + _erf(v / np.sqrt(2.0)))


def layernorm(v, w, b):
    """(v - mean) / sqrt(var + eps) * w + b over the last axis, var = the biased variance (reading #23)."""
    mu = np.mean(v, axis=-1, keepdims=True)
    var = np.mean((v - mu) * (v - mu), axis=-1, keepdims=True)
    return (v - mu) / np.sqrt(var + EPS) * w + b


def ffn(u, ly):
    """Alg. 1 l.4's FFN: W2 GELU(W1 u + b1) + b2 (reading #23)."""
    return gelu(u @ ly.ffn_w1.T + ly.ffn_b1) @ ly.ffn_w2.T + ly.ffn_b2


@dataclass
class State:
    """Stream cache S_t: per layer the last K-1 conv inputs and the SSM state h."""
    win: list   # per layer [S, K-1, E]   win[:, j] = x_{t-(K-1)+j}
    h: list     # per layer [S, E, N]


def init_state(w: Weights, n_streams: int) -> State:
    e = w.d_inner
    return State(win=[np.zeros((n_streams, w.d_conv - 1, e)) for _ in range(w.n_layer)],
                 h=[np.zeros((n_streams, e, w.d_state)) for _ in range(w.n_layer)])


def conv_step(win, x, conv_w, conv_b):
    """Causal depthwise conv, one step.  win [S,K-1,E] = (x_{t-3},x_{t-2},x_{t-1}); x [S,E] = x_t.
    xc_e = b_e + sum_k w[e][k] * (x_{t-3}, x_{t-2}, x_{t-1}, x_t)[k];  returns (xc, new window)."""
    k = conv_w.shape[1]
    xc = conv_b + conv_w[:, k - 1] * x
    for j in range(k - 1):
        xc = xc + conv_w[:, j] * win[:, j, :]
    new_win = np.concatenate([win[:, 1:, :], x[:, None, :]], axis=1)
    return xc, new_win


def ssm_step(h, xs, delta, bv, cv, a, d_skip):
    """eq. 16, 18, 19 with B_bar = delta*B:  h <- exp(delta*A) h + (delta*B) xs ;  y = C.h + D xs.
    h [S,E,N], xs [S,E], delta [S,E], bv/cv [S,N], a [E,N] (negative), d_skip [E]."""
    a_bar = np.exp(delta[:, :, None] * a[None, :, :])
    h = a_bar * h + (delta[:, :, None] * bv[:, None, :]) * xs[:, :, None]
    y = np.sum(cv[:, None, :] * h, axis=2) + d_skip * xs
    return h, y


def step(w: Weights, st: State, sym: np.ndarray):
    """Phi_theta (eq. 5): previous bytes `sym` [S] (uint8) + state -> logits [S,256]; state is updated in place."""
    n, r = w.d_state, w.dt_rank
    e = w.d_inner
    u = w.emb[sym.astype(np.int64)]                       # Alg. 1 line 1 (ByteEmbed)
    for l, ly in enumerate(w.layers):                      # Alg. 1 lines 2-3
        rr = rmsnorm(u, ly.norm_w)
        xz = rr @ ly.w_in.T
        x, z = xz[:, :e], xz[:, e:]
        xc, st.win[l] = conv_step(st.win[l], x, ly.conv_w, ly.conv_b)
        xs = silu(xc)
        dbc = xs @ ly.w_x.T                                # eq. 21-22 (and the low-rank delta input)
        dlt, bv, cv = dbc[:, :r], dbc[:, r:r + n], dbc[:, r + n:]
        delta = softplus(dlt @ ly.w_dt.T + ly.b_dt)        # eq. 20
        a = -np.exp(ly.a_log)
        st.h[l], y = ssm_step(st.h[l], xs, delta, bv, cv, a, ly.d_skip)
        y = y * silu(z)
        u = u + y @ ly.w_out.T
        if w.d_ff:
            u = layernorm(ffn(u, ly), ly.ln_w, ly.ln_b)   # Alg. 1 line 4
    head = w.emb if w.head is None else w.head
    return u @ head.T                                      # Alg. 1 line 5


def logits_for_chunks(w: Weights, chunks: np.ndarray) -> np.ndarray:
    """chunks [S, T] uint8 (equal length).  Returns logits [S, T-1, 256]: row t predicts byte t+1
    from bytes 0..t (byte 0 is stored raw, the last byte is never fed to the model)."""
    s, t = chunks.shape
    st = init_state(w, s)
    out = np.empty((s, max(t - 1, 0), 256))
    for i in range(t - 1):
        out[:, i, :] = step(w, st, chunks[:, i])
    return out
