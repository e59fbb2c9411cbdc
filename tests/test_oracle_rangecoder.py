"""Pins for oracle/rangecoder.py (O3): the eq. 12 inverse identity by brute force, a big-integer
definition of the code value, toy-width fuzzing of the carry logic, exact and entropy code lengths,
and the survey-derived byte vectors."""
import os

import numpy as np
import pytest

from oracle.rangecoder import RangeDecoder, RangeEncoder, decode_stream, encode_stream

HERE = os.path.dirname(__file__)


def rng(seed=0):
    return np.random.Generator(np.random.PCG64(seed))


def random_cdf(g, nsym, M, peaky):
    w = g.gamma(0.05 if peaky else 1.0, 1.0, nsym) + 1e-12
    f = np.maximum(1, np.floor(w / w.sum() * (M - nsym)).astype(np.int64))
    f[np.argmax(f)] += M - f.sum()
    assert f.min() >= 1 and f.sum() == M
    return np.concatenate([[0], np.cumsum(f)])


def test_eq12_is_the_inverse_of_eq8_brute_force():
    # V >= floor(R*C/M)  <=>  floor(((V+1)*M-1)/R) >= C    for every R in [2^6,2^8), C in [0,M], V < R, M = 2^4
    M = 16
    for R in range(64, 256):
        for V in range(R):
            x = ((V + 1) * M - 1) // R
            assert 0 <= x < M
            for C in range(M + 1):
                assert (V >= (R * C) // M) == (x >= C)


def big_integer_code(cdfs, syms, unit_bits, n_units, fb):
    """The plain definition: keep the whole base L as one unbounded integer (no cache / pending /
    carry machinery); the emitted units are its digits."""
    w = unit_bits * n_units
    low, rng_, shifts = 0, (1 << w) - 1, 0
    for C, s in zip(cdfs, syms):
        low += (rng_ * int(C[s])) >> fb
        rng_ = (rng_ * int(C[s + 1] - C[s])) >> fb
        while rng_ < (1 << (w - unit_bits)):
            low <<= unit_bits
            rng_ <<= unit_bits
            shifts += 1
    n_out = shifts + n_units
    digits = [(low >> (unit_bits * (n_out - 1 - i))) & ((1 << unit_bits) - 1) for i in range(n_out)]
    assert low >> (unit_bits * n_out) == 0
    return digits


@pytest.mark.parametrize("unit_bits,n_units,fb", [(2, 4, 4), (3, 4, 6), (4, 4, 8), (2, 8, 8), (8, 4, 16)])
def test_fuzz_against_big_integer_definition_and_round_trip(unit_bits, n_units, fb):
    g = rng(unit_bits * 100 + n_units)
    M = 1 << fb
    nsym = min(256, M // 2)
    carries = longest = 0
    n_seq = 300 if unit_bits == 8 else 1500
    for it in range(n_seq):
        T = int(g.integers(0, 60))
        cdfs = [random_cdf(g, nsym, M, peaky=(it % 2 == 0)) for _ in range(T)]
        # bias towards the last symbol of the table: drives low towards all-ones units (pending runs)
        syms = [int(nsym - 1) if g.random() < 0.6 else int(g.integers(nsym)) for _ in range(T)]
        enc = RangeEncoder(unit_bits, n_units, fb)
        for C, s in zip(cdfs, syms):
            before = enc.pending
            enc.encode(int(C[s]), int(C[s + 1]))
            longest = max(longest, enc.pending)
            if before and enc.low >> enc.w:
                carries += 1
        out = list(enc.finish())
        assert out == big_integer_code(cdfs, syms, unit_bits, n_units, fb)
        dec = RangeDecoder(out, unit_bits, n_units, fb)
        for C, s in zip(cdfs, syms):
            x = dec.target()
            assert C[s] <= x < C[s + 1]
            dec.consume(int(C[s]), int(C[s + 1]))
        assert dec.pos == len(out)                      # decoder consumes exactly what was produced
    if unit_bits < 8:
        assert longest >= 3                              # the pending path was really exercised


def test_uniform_table_costs_exactly_n_plus_4_bytes():
    C = np.arange(257) * 256
    for n in (0, 1, 2, 1000):
        syms = rng(n).integers(0, 256, n)
        out = encode_stream([C] * n, syms)
        assert len(out) == n + 4
        back, used = decode_stream([C] * n, out)
        assert back == list(syms) and used == len(out)


def test_iid_code_length_matches_cross_entropy():
    # eq. 1: bytes ~= sum_t -log256 q(s_t); and within 0.1 % of n*H(P,Q) in the log256 form
    g = rng(11)
    C = random_cdf(g, 256, 1 << 16, peaky=False)
    qd = np.diff(C) / 65536.0
    p = g.dirichlet(np.full(256, 0.7))
    n = 1 << 19
    syms = g.choice(256, size=n, p=p)
    enc = RangeEncoder()
    lo, hi = C[:-1].tolist(), C[1:].tolist()
    for s in syms.tolist():
        enc.encode(lo[s], hi[s])
    nbytes = len(enc.finish())
    ideal = float(np.sum(-np.log(qd[syms])) / np.log(256))
    assert 0 < nbytes - ideal < 5 + n * 2e-5            # coder overhead: flush + range truncation (<= 2^-8 bit/symbol)
    H_pq = float(-(p * np.log(qd)).sum() / np.log(256))
    sigma = np.sqrt(max(float((p * (np.log(qd) / np.log(256)) ** 2).sum()) - H_pq ** 2, 0) / n)
    assert abs(nbytes / (n * H_pq) - 1) < 1e-3 + 4 * sigma / H_pq   # sampling noise of the source itself


def test_skewed_32bit_fuzz_round_trip_with_carries():
    g = rng(12)
    carries = 0
    for it in range(40):
        T = 400
        cdfs = [random_cdf(g, 256, 1 << 16, peaky=True) for _ in range(T)]
        syms = [255 if g.random() < 0.5 else int(g.integers(256)) for _ in range(T)]
        enc = RangeEncoder()
        for C, s in zip(cdfs, syms):
            enc.encode(int(C[s]), int(C[s + 1]))
            carries += enc.low >> 32
        out = enc.finish()
        back, used = decode_stream(cdfs, out)
        assert back == syms and used == len(out)
    assert carries > 0


def _table(name):
    f = np.ones(256, dtype=np.int64)
    if name == "uniform":
        f[:] = 256
    elif name == "peak0":
        f[0] = 65281
    elif name == "peak255":
        f[255] = 65281
    return np.concatenate([[0], np.cumsum(f)])


def test_survey_byte_vectors():
    n = 0
    for line in open(os.path.join(HERE, "golden", "rc_vectors.txt")):
        if line.startswith("#") or not line.strip():
            continue
        tname, syms, payload = [s.strip() for s in line.split(";")]
        if "x" in syms:
            b, c = syms.split("x")
            seq = [int(b, 16)] * int(c)
        else:
            seq = [int(t, 16) for t in syms.split()]
        C = _table(tname)
        assert encode_stream([C] * len(seq), seq).hex(" ") == payload, line
        n += 1
    assert n == 6
