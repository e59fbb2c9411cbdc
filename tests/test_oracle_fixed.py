"""Pins for oracle/fixed.py — the deterministic fixed-point pipeline FX1 (PAPER "Portability",
P:259-277).  The module is a specification in exact integers, so the pins are of three kinds:
(a) every primitive against exact rational / 50-digit arithmetic done another way (fractions, decimal - the tables are
generated with mpmath), brute force at small widths; (b) the vectorised step against a scalar re-statement in plain
Python integers, bit for bit; (c) what the pipeline is for: tables with the required invariants, a lossless round trip,
and a measured, asserted distance to the fp64 oracle's probabilities."""
import math
from decimal import Decimal, getcontext
from fractions import Fraction

import numpy as np

from oracle import codec, container, fixed as fx, model, quantise
from paper_2511_11337_b200 import synth


def rng(seed=0):
    return np.random.Generator(np.random.PCG64(seed))


def _round_half_even(fr: Fraction) -> int:
    fl = math.floor(fr)
    d = fr - fl
    return fl + (1 if (d > Fraction(1, 2) or (d == Fraction(1, 2) and fl % 2 == 1)) else 0)


def test_rounding_shift_and_division_brute_force():
    for k in range(1, 6):
        vals = np.arange(-80, 81, dtype=np.int64)
        got = fx.rne(vals, k)
        for v, g in zip(vals, got):
            want = _round_half_even(Fraction(int(v), 1 << k))
            assert int(g) == want == fx.rne(int(v), k), (v, k)
    assert fx.rne(5, 0) == 5 and fx.rne(5, -3) == 40 and list(fx.rne(np.array([3, -3]), -2)) == [12, -12]
    for d in range(1, 12):
        n = np.arange(-60, 61, dtype=np.int64)
        got = fx.rdiv(n, np.full_like(n, d))
        for a, g in zip(n, got):
            assert int(g) == _round_half_even(Fraction(int(a), d)) == fx.rdiv(int(a), d), (a, d)
    assert fx.sat(2 ** 31) == 2 ** 31 - 1 and fx.sat(-2 ** 31 - 5) == -2 ** 31 and list(fx.sat(np.array([2 ** 40, -2 ** 40, 7]))) == [2 ** 31 - 1, -2 ** 31, 7]
    assert fx.qmul(3 << 20, 5 << 19) == 15 << 19 and fx.qmul(2 ** 31 - 1, 2 ** 31 - 1) == 2 ** 31 - 1      # saturates


def test_isqrt_and_bitlen_exact():
    xs = np.concatenate([np.arange(0, 5000), rng(1).integers(0, 2 ** 62, 20000), [2 ** 62 - 1, 2 ** 58, (2 ** 29) ** 2 - 1, (2 ** 29) ** 2]]).astype(np.int64)
    y = fx.isqrt(xs)
    for a, b in zip(xs, y):
        assert int(b) == math.isqrt(int(a))
    m = np.array([0, 1, 2, 3, 4, 127, 128, 2 ** 30, 2 ** 31 - 1], np.int64)
    assert list(fx.bitlen(m)) == [int(v).bit_length() for v in m]


def test_tables_against_decimal_arithmetic():
    """EXP2_TAB / LOG1P_TAB (generated with mpmath) recomputed with the decimal module at 50 digits."""
    getcontext().prec = 50
    ln2 = Decimal(2).ln()
    assert len(fx.EXP2_TAB) == len(fx.LOG1P_TAB) == 257
    for i in range(257):
        e = (Decimal(2) ** 30) * (-(Decimal(i) / 256) * ln2).exp()
        l = (Decimal(2) ** 30) * (1 + Decimal(i) / 256).ln()
        assert int(fx.EXP2_TAB[i]) == int(e.to_integral_value(rounding="ROUND_HALF_EVEN")), i
        assert int(fx.LOG1P_TAB[i]) == int(l.to_integral_value(rounding="ROUND_HALF_EVEN")), i
    assert fx.EXP2_TAB[0] == 2 ** 30 and fx.EXP2_TAB[256] == 2 ** 29 and fx.LOG1P_TAB[0] == 0
    assert fx.LOG2E_Q30 == int((Decimal(2) ** 30 / ln2).to_integral_value(rounding="ROUND_HALF_EVEN"))
    assert fx.EPS_Q40 == round(1e-5 * 2 ** 40) and fx.TABLE_CRC == 0x6B76FB0D      # the CRC an implementation checks its copy with


def test_integer_transcendentals_against_fp64():
    g = rng(2)
    t = np.concatenate([[0, 1, fx.ONE - 1, fx.ONE, 31 * fx.ONE, 40 * fx.ONE], g.integers(0, 34 * fx.ONE, 20000)]).astype(np.int64)
    e2 = fx.exp2_neg(t)
    assert e2[0] == 2 ** 30 and np.all(e2[4:6] == [0, 0]) and np.all((e2 >= 0) & (e2 <= 2 ** 30))
    assert np.max(np.abs(e2 / 2.0 ** 30 - np.exp2(-t / fx.ONE))) < 1.0e-6               # 256-interval linear interpolation: <= 9.2e-7
    assert all(int(fx.exp2_neg(int(v))) == int(w) for v, w in zip(t[:200], e2[:200]))   # scalar path == array path
    o = np.argsort(t)
    assert np.all(np.diff(e2[o]) <= 0)                                                  # monotone
    x = g.integers(-30 * fx.ONE, 30 * fx.ONE, 20000).astype(np.int64)
    s = fx.sigmoid(x)
    assert np.all(s + fx.sigmoid(-x) == 2 ** 30)                                        # exact complement
    assert np.max(np.abs(s / 2.0 ** 30 - 1 / (1 + np.exp(-x / fx.ONE)))) < 2e-6
    xr = x / fx.ONE
    assert np.max(np.abs(fx.silu(x) / fx.ONE - xr / (1 + np.exp(-xr)))) < 2e-5
    sp = fx.softplus(x)
    ref = np.maximum(xr, 0) + np.log1p(np.exp(-np.abs(xr)))
    assert np.max(np.abs(sp / fx.ONE - ref)) < 2e-5 and np.all(sp >= 0) and np.all(np.diff(sp[np.argsort(x)]) >= 0)
    for v in (0, 5, -5, 12345678, -87654321):
        assert int(fx.sigmoid(np.array([v]))[0]) == fx.sigmoid(v) and int(fx.softplus(np.array([v]))[0]) == fx.softplus(v)
        assert int(fx.silu(np.array([v]))[0]) == fx.silu(v)


def test_int8_rows_and_the_integer_gemm_in_exact_rationals():
    g = rng(3)
    w = (g.normal(0, 0.05, (9, 40)) * np.exp(g.normal(0, 3, (9, 1)))).astype(np.float32)
    w[4] = 0.0
    w[5, :] = 0.0; w[5, 3] = 127.0 / 64                                                 # max * 2^6 = 127 exactly: s = 6
    q, s = fx.quantise_weight_rows(w)
    assert s[4] == 0 and np.all(q[4] == 0) and s[5] == 6 and q[5, 3] == 127
    for r in range(9):
        if r == 4:
            continue
        m = np.abs(w[r].astype(np.float64)).max()
        assert m * 2.0 ** s[r] <= 127 < m * 2.0 ** (s[r] + 1) and np.abs(q[r]).max() >= 64
        assert np.abs(q[r] / 2.0 ** s[r] - w[r]).max() <= 2.0 ** (-s[r] - 1) + 1e-18
    a = g.integers(-3 * fx.ONE, 3 * fx.ONE, (7, 40)).astype(np.int64)
    a[2] = 0
    a[3, 0] = 2 ** 31 - 1                                                               # a row at full scale: k = 24
    qa, k = fx.quantise_rows(a)
    assert k[2] == 0 and np.all(qa[2] == 0) and k[3] == 24 and np.abs(qa).max() <= 127
    for i in range(7):
        if i != 2:
            assert 64 <= np.abs(qa[i]).max() <= 127
    out = fx.gemm_q(a, q, s)
    for i in range(7):
        for r in range(9):
            acc = sum(int(x) * int(y) for x, y in zip(qa[i], q[r]))
            want = _round_half_even(Fraction(acc) * Fraction(2) ** int(k[i] - s[r]))    # acc * 2^(k-F) * 2^-s in units of 2^-F
            assert int(out[i, r]) == max(-2 ** 31, min(2 ** 31 - 1, want)), (i, r)
    # and it is a faithful product: against fp64 on the dequantised operands within the int8 step sizes
    ref = (a / fx.ONE) @ w.astype(np.float64).T
    tol = np.abs(a / fx.ONE).sum(1)[:, None] * (2.0 ** (-s - 1))[None, :] + np.abs(w).sum(1)[None, :] * (2.0 ** (k - fx.F - 1))[:, None]
    live = np.abs(ref) < 2000
    assert np.all(np.abs(out / fx.ONE - ref)[live] <= tol[live] + 2.0 ** -19)


def test_integer_rmsnorm_against_fp64_and_its_scale_invariance():
    g = rng(4)
    D = 256
    w = fx.to_q(1.0 + g.normal(0, 0.1, D))
    u = fx.to_q(g.normal(0, 1.0, (6, D)) * np.array([1e-3, 0.1, 1.0, 30.0, 300.0, 0.0])[:, None])
    sd = int(fx.isqrt(D << 40))
    assert abs(sd / 2 ** 20 - math.sqrt(D)) < 2 ** -19
    r = fx.rmsnorm(u, w, sd)
    uf = u / fx.ONE
    ref = uf / np.sqrt((uf * uf).mean(1, keepdims=True) + 1e-5) * (w / fx.ONE)
    assert np.all(r[5] == 0) and np.max(np.abs(r / fx.ONE - ref)[1:5]) < 3e-5
    assert np.max(np.abs(r / fx.ONE - ref)[0]) < 1e-3            # |u| ~ 1e-3: 10 significant bits left of a Q value
    # multiplying a row by 2^j only changes the exponent e; t and S are the same integers, and so is the result up to eps
    big = fx.rmsnorm(u[2:3] * 8, w, sd)
    assert np.max(np.abs(big - r[2:3])) <= 16                     # eps = 1e-5 against a mean square of ~1 and of ~64:
                                                                   # a relative 5e-6 of values up to ~3.5 = 3.7e6 units


def _tiny(layers=2, emb_std=0.25):
    shape = synth.ModelShape(layers, 64, dt_rank=4)
    blob = synth.make_weights(shape, 21, emb_std=emb_std)
    w = model.load_weights(blob)
    return w, fx.quantise_model(w)


def test_vectorised_step_equals_the_scalar_specification():
    w, q = _tiny()
    data = np.frombuffer(synth.CONFIGS[1].data(3 * 12), np.uint8).reshape(3, 12)
    st = fx.init_state(q, 3)
    ss = [[{"win": [[0, 0, 0] for _ in range(q.d_inner)], "h": [[0] * q.d_state for _ in range(q.d_inner)]} for _ in q.layers] for _ in range(3)]
    for t in range(11):
        lv = fx.step(q, st, data[:, t])
        assert lv.dtype == np.int64 and np.all((lv >= -2 ** 31) & (lv < 2 ** 31))
        for i in range(3):
            assert [int(v) for v in lv[i]] == fx.scalar_step(q, ss[i], int(data[i, t])), (t, i)
    # a stream's result does not depend on its neighbours: stepping stream 1 alone gives the same integers
    st1 = fx.init_state(q, 1)
    for t in range(11):
        l1 = fx.step(q, st1, data[1:2, t])
    assert np.array_equal(l1[0], lv[1])


def test_tables_invariants_and_closed_forms():
    z = np.zeros((1, 256), np.int64)
    assert np.all(np.diff(fx.table(z)) == 256)                                          # uniform logits
    one = np.full((1, 256), -60 * fx.ONE, np.int64); one[0, 17] = 3 * fx.ONE
    f = np.diff(fx.table(one))[0]
    assert f[17] == 65281 and f.sum() == 65536 and np.all(np.delete(f, 17) == 1)        # one-hot
    two = one.copy(); two[0, 200] = 3 * fx.ONE
    f = np.diff(fx.table(two))[0]
    assert f[17] == f[200] == 32641
    l = rng(5).integers(-8 * fx.ONE, 8 * fx.ONE, (500, 256)).astype(np.int64)
    C = fx.table(l)
    f = np.diff(C, axis=-1)
    assert np.all(C[:, 0] == 0) and np.all(C[:, 256] == 65536) and f.min() >= 1
    p = fx.probabilities(l)
    assert np.max(np.abs(f / 65536.0 - (1 + 65280 * p) / 65536.0)) < 2.5e-5            # eq. 7: the table is the softmax + the floor


def test_distance_to_the_fp64_oracle_and_lossless_round_trip():
    """What INT8 rows cost: |p_FX1 - p_fp64| on the configured (near-uniform) and on a sharp weight set, asserted with
    margin and printed; the containers round-trip bit-exactly and differ from the fp64 oracle's only by that cost."""
    cfg = synth.CONFIGS[1]
    data = cfg.data(4 * 48 + 11)
    for emb_std, bound, size_tol in ((None, 5e-6, 0.002), (0.25, 2e-2, 0.02)):
        blob = cfg.weights() if emb_std is None else cfg.weights(emb_std=emb_std)
        w = model.load_weights(blob)
        q = fx.quantise_model(w)
        chunks = np.frombuffer(data[: 4 * 48], np.uint8).reshape(4, 48)
        st, stf = fx.init_state(q, 4), model.init_state(w, 4)
        worst = 0.0
        for t in range(47):
            pq = fx.probabilities(fx.step(q, st, chunks[:, t]))
            pf = quantise.softmax(model.step(w, stf, chunks[:, t]))
            worst = max(worst, float(np.abs(pq - pf).max()))
        blob_fx = fx.compress(q, data, 48)
        assert fx.decompress(q, blob_fx) == data
        ref = codec.compress(w, data, 48)
        print(f"[FX1] emb_std={emb_std}: max |p_FX1 - p_fp64| = {worst:.3e}; container {len(blob_fx)} B vs fp64 oracle {len(ref)} B")
        assert worst <= bound and abs(len(blob_fx) - len(ref)) <= size_tol * len(ref)
        # the arithmetic word keeps the two kinds of container apart
        try:
            container.unpack(blob_fx, codec.fingerprint(w))
            raise AssertionError("an FX1 container was accepted as an fp64-oracle container")
        except container.FormatError:
            pass
