"""O2 — softmax (eq. 6) and the strictly positive integer histogram / CDF (eq. 7).
Oracle; test infrastructure.

The paper fixes only the properties of the table (f_t(a) >= 1, sum f_t = M = 2^B, identical on both
sides) and not the rounding rule.  The rule used here is DESIGN.md reading #5:

    m    = max_a l[a]                                        (the logits are fp32 numbers)
    e[a] = EXP(l[a] - m)   in (0, 1]                         (EXP: the fp32 routine below)
    g[a] = min(floor(e[a] * 2^23), 2^23)                     integer, the arg-max gets exactly 2^23
    G[a] = sum_{x<a} g[x],  T = G[256]                       integer prefix sums (order-free)
    C[a] = a + floor(G[a] * (2^16 - 256) / T)                64-bit integers;  f[a] = C[a+1] - C[a]

A floating-point value decides an integer here (floor(e*2^23)), so both sides must take that decision
in the same precision, and that precision is the kernel's: fp32.  EXP is therefore a *specified*
fp32 algorithm — every operation an individually rounded IEEE-754 binary32 multiply / add / subtract
(no fused multiply-add), so numpy float32 and a GPU's __fmul_rn/__fadd_rn give the same bits:

    t = d * LOG2E ;  t < -64 -> 0 ;  n = rint(t) ;  r = t - n  (exact) ;
    p = c6 ; p = p*r + c5 ; ... ; p = p*r + c0  (c0 = 1) ;  EXP = p * 2^n  (exact)

Reading #17: a NaN logit or a non-finite maximum gives the uniform table (f = 256 everywhere).
"""
from __future__ import annotations

import numpy as np

FREQ_BITS = 16
M = 1 << FREQ_BITS
G_ONE = 1 << 23

_f32 = np.float32
LOG2E = np.array(0x3FB8AA3B, dtype=np.uint32).view(np.float32)
# degree-6 polynomial for 2^r on [-1/2, 1/2], c0 = 1 exactly (max rel. error 1.0e-7 incl. fp32 rounding)
EXP2_COEF = np.array([0x3F800000, 0x3F317218, 0x3E75FDEE, 0x3D63576B, 0x3C1D9662, 0x3AAFA26E, 0x39212C6C],
                     dtype=np.uint32).view(np.float32)


def softmax(logits: np.ndarray) -> np.ndarray:
    """eq. 6 in fp64 (max subtracted: mathematically identical)."""
    l = np.asarray(logits, dtype=np.float64)
    ex = np.exp(l - np.max(l, axis=-1, keepdims=True))
    return ex / np.sum(ex, axis=-1, keepdims=True)


def exp_f32_spec(d: np.ndarray) -> np.ndarray:
    """EXP(d) for fp32 d <= 0, operation by operation in binary32."""
    d = np.asarray(d, dtype=_f32)
    with np.errstate(invalid="ignore", over="ignore"):
        t = (d * LOG2E).astype(_f32)
        dead = ~(t >= _f32(-64.0))            # also true for NaN / -inf
        t = np.where(dead, _f32(0.0), t)
        n = np.rint(t).astype(_f32)
        r = (t - n).astype(_f32)
        p = np.full_like(r, EXP2_COEF[6])
        for j in range(5, -1, -1):
            p = (p * r).astype(_f32)
            p = (p + EXP2_COEF[j]).astype(_f32)
        e = np.ldexp(p, n.astype(np.int32)).astype(_f32)
    return np.where(dead, _f32(0.0), e)


def quantise(logits_f32: np.ndarray) -> np.ndarray:
    """fp32 logits [..., 256] -> integer CDF C [..., 257] (int64), C[0] = 0, C[256] = 2^16, f >= 1."""
    l = np.asarray(logits_f32, dtype=_f32)
    assert l.shape[-1] == 256
    m = np.max(l, axis=-1, keepdims=True)                      # NaN propagates through np.max
    bad = ~np.isfinite(m[..., 0])
    with np.errstate(invalid="ignore"):
        d = (l - m).astype(_f32)
    e = exp_f32_spec(d)
    g = np.minimum(np.floor(e.astype(np.float64) * G_ONE), G_ONE).astype(np.int64)   # e*2^23 is exact
    G = np.zeros(l.shape[:-1] + (257,), dtype=np.int64)
    np.cumsum(g, axis=-1, out=G[..., 1:])
    T = G[..., 256:257]
    T = np.where(T == 0, 1, T)                                  # only reachable on `bad` rows
    a = np.arange(257, dtype=np.int64)
    C = a + (G * (M - 256)) // T
    C[bad] = a * 256
    return C


def find_symbol(C: np.ndarray, x: int) -> int:
    """The unique s with C[s] <= x < C[s+1]."""
    return int(np.searchsorted(C, x, side="right")) - 1
