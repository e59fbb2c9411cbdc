"""O3 — the range coder (eq. 8-13), exact Python integers.  Oracle; test infrastructure.

Encoder (eq. 8-9), with M = 2^freq_bits:
    L <- L + floor(R * C(s) / M) ;   R <- floor(R * (C(s+1) - C(s)) / M)
Renormalisation (eq. 10-11): the paper shifts out the top unit (byte) of L once it is
fixed and rescales L, R by 2^8 on a w-bit ring.  As printed the rule has no bound on R when L and
L+R-1 straddle a byte boundary; reading #6 is the classical carry-propagating form of the
same rule: shift whenever R < 2^(w-8); a byte that may still receive a carry is held back (`cache`
plus a run of `pending` 0xFF units) and written only when it is final — "emits bytes as soon as
they are fixed".  First unit encoded is first decoded (queue order).

Decoder (eq. 12-13), reading #7: it keeps V = C - L (code value relative to the base)
instead of C and L separately — algebraically identical, no carries on the decode side:
    x = floor(((V + 1) * M - 1) / R)  in [0, M) ;  s: C(s) <= x < C(s+1) ;
    V <- V - floor(R * C(s) / M) ;  R <- floor(R * f(s) / M) ;  on refill V <- (V << 8) + b.

`unit_bits` / `n_units` exist so tests can run the *same* code at toy widths (2-4-bit units on an
8-16-bit ring), where carries through long pending runs happen constantly.  The product format is
unit_bits = 8, n_units = 4 (w = 32), freq_bits = 16 (reading #5/#6); flush = n_units + 1 shifts (#9).
"""
from __future__ import annotations


class RangeEncoder:
    def __init__(self, unit_bits: int = 8, n_units: int = 4, freq_bits: int = 16):
        self.u = unit_bits
        self.w = unit_bits * n_units
        self.n_units = n_units
        self.fb = freq_bits
        assert self.w - self.u >= freq_bits, "range must keep freq_bits of resolution after renormalisation"
        self.unit_mask = (1 << unit_bits) - 1
        self.low = 0                       # w+1 bits: bit w is the carry
        self.range = (1 << self.w) - 1
        self.cache = 0
        self.pending = 0
        self.started = False
        self.out = []                      # list of units (bytes when unit_bits == 8)

    def _shift_low(self):
        w, u = self.w, self.u
        carry = self.low >> w
        if (self.low & ((1 << w) - 1)) < (self.unit_mask << (w - u)) or carry == 1:
            if self.started:
                self.out.append((self.cache + carry) & self.unit_mask)
            self.out.extend([(self.unit_mask + carry) & self.unit_mask] * self.pending)
            self.pending = 0
            self.started = True
            self.cache = (self.low >> (w - u)) & self.unit_mask
        else:
            self.pending += 1
        self.low = (self.low & ((1 << (w - u)) - 1)) << u

    def encode(self, c_lo: int, c_hi: int):
        """Code the symbol whose cumulative interval is [c_lo, c_hi) out of M."""
        assert 0 <= c_lo < c_hi <= (1 << self.fb)
        self.low += (self.range * c_lo) >> self.fb            # eq. 8
        self.range = (self.range * (c_hi - c_lo)) >> self.fb  # eq. 9
        while self.range < (1 << (self.w - self.u)):          # eq. 10-11 (reading #6)
            self._shift_low()
            self.range <<= self.u

    def finish(self):
        for _ in range(self.n_units + 1):
            self._shift_low()
        return bytes(self.out) if self.u == 8 else list(self.out)


class RangeDecoder:
    def __init__(self, data, unit_bits: int = 8, n_units: int = 4, freq_bits: int = 16):
        self.u = unit_bits
        self.w = unit_bits * n_units
        self.fb = freq_bits
        self.data = data
        self.pos = 0
        self.range = (1 << self.w) - 1
        self.v = 0
        for _ in range(n_units):
            self.v = (self.v << self.u) | self._next()

    def _next(self):
        if self.pos >= len(self.data):
            raise EOFError("range decoder ran past the end of its stream")
        b = self.data[self.pos]
        self.pos += 1
        return b

    def target(self) -> int:
        """eq. 12."""
        return (((self.v + 1) << self.fb) - 1) // self.range

    def consume(self, c_lo: int, c_hi: int):
        self.v -= (self.range * c_lo) >> self.fb
        self.range = (self.range * (c_hi - c_lo)) >> self.fb
        while self.range < (1 << (self.w - self.u)):
            self.v = (self.v << self.u) | self._next()        # eq. 13
            self.range <<= self.u


def encode_stream(cdfs, symbols) -> bytes:
    """cdfs[t] = C_t (257 ints), symbols[t] = s_t.  Returns the payload of one stream."""
    enc = RangeEncoder()
    for C, s in zip(cdfs, symbols):
        enc.encode(int(C[s]), int(C[s + 1]))
    return enc.finish()


def decode_stream(cdfs, payload: bytes):
    """Inverse of encode_stream given the same tables.  Returns (symbols, bytes consumed)."""
    import bisect
    dec = RangeDecoder(payload)
    out = []
    for C in cdfs:
        C = [int(v) for v in C]
        x = dec.target()
        s = bisect.bisect_right(C, x) - 1
        dec.consume(C[s], C[s + 1])
        out.append(s)
    return out, dec.pos
