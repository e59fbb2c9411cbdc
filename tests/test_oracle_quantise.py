"""Pins for oracle/quantise.py (O2): library exp / softmax, closed-form tables, invariants,
brute-force symbol search, and the division-free search identity the decoder may rely on."""
import numpy as np
import torch

from oracle import quantise as q


def rng(seed=0):
    return np.random.Generator(np.random.PCG64(seed))


def test_softmax_against_torch():
    l = rng(1).normal(0, 4, (50, 256))
    np.testing.assert_allclose(q.softmax(l), torch.softmax(torch.tensor(l), -1).numpy(), rtol=1e-13)
    assert np.allclose(q.softmax(l).sum(-1), 1.0, atol=1e-14)


def test_exp_spec_against_fp64_exp():
    d = -np.abs(rng(2).normal(0, 8, 200000)).astype(np.float32)
    d[:5] = [0.0, -1e-8, -44.0, -44.5, -np.inf]
    e = q.exp_f32_spec(d)
    assert e.dtype == np.float32 and e[0] == 1.0 and e[4] == 0.0
    ref = np.exp(d.astype(np.float64))
    live = d * q.LOG2E >= -64
    # 1e-7 polynomial + fp32 rounding of t = d*log2(e) (half an ulp of |t|, i.e. <= 6e-8 * |d| relative)
    assert np.all(np.abs(e[live] - ref[live]) / ref[live] < 2.5e-7 + 1.3e-7 * np.abs(d[live]))
    assert np.max(np.abs(e[live] - ref[live])) < 1.5e-7                 # absolute: what the table sees
    assert np.all(e[~live] == 0.0) and np.all(ref[~live] < 2.0 ** -64)
    assert np.all(e <= 1.0)
    # monotone in d up to fp32 rounding: sort and check no large inversions
    o = np.argsort(d)
    assert np.all(np.diff(e[o].astype(np.float64)) >= -3e-7 * e[o][1:])


def test_closed_form_tables():
    f = np.diff(q.quantise(np.zeros(256, np.float32)))
    assert np.all(f == 256)                                   # uniform logits
    f = np.diff(q.quantise(np.full(256, -3.25, np.float32)))
    assert np.all(f == 256)                                   # shift invariance of softmax
    l = np.full(256, -1000.0, np.float32); l[77] = 5.0
    f = np.diff(q.quantise(l))
    assert f[77] == 65281 and np.all(np.delete(f, 77) == 1)   # one-hot: 65536 - 255
    l[200] = 5.0
    f = np.diff(q.quantise(l))
    assert f[77] == 32641 and f[200] == 32641 and f.sum() == 65536   # two-way tie: (65536-254)/2
    # p = (1/2, 1/4, 1/4, 0...) : exact powers of two survive the fp32 exp exactly
    l = np.full(256, -np.inf, np.float32); l[:3] = np.log(np.array([0.5, 0.25, 0.25])).astype(np.float32)
    f = np.diff(q.quantise(l))
    assert abs(int(f[0]) - (1 + 65280 // 2)) <= 1 and abs(int(f[1]) - (1 + 65280 // 4)) <= 1 and f.sum() == 65536


def test_invariants_and_closeness_to_softmax():
    g = rng(3)
    for scale in (0.02, 1.0, 6.0, 40.0):
        l = (g.normal(0, scale, (3000, 256))).astype(np.float32)
        C = q.quantise(l)
        f = np.diff(C, axis=-1)
        assert np.all(C[:, 0] == 0) and np.all(C[:, 256] == 65536) and f.min() >= 1
        # eq. 7 meaning: f/M is the softmax up to the +1 floor and integer rounding
        p = q.softmax(l.astype(np.float64))
        # error budget: +-1 from the two floors of C, 2^-23 per g (256 of them enter T), 3e-7 from EXP
        assert np.all(np.abs(f - (1 + 65280 * p)) <= 1.0 + 65280 * (2.0 ** -23 + p * (257 * 2.0 ** -23 + 3e-7)))
        # order preserving up to one count
        i = np.argsort(l, axis=-1)
        fs = np.take_along_axis(f, i, -1)
        assert np.all(np.diff(fs, axis=-1) >= -1)


def test_non_finite_rule():
    l = rng(4).normal(0, 1, (4, 256)).astype(np.float32)
    l[0, 3] = np.nan; l[1, 9] = np.inf; l[2, :] = -np.inf
    C = q.quantise(l)
    for r in (0, 1, 2):
        assert np.all(np.diff(C[r]) == 256)
    assert not np.all(np.diff(C[3]) == 256) and C[3, 256] == 65536
    l2 = rng(5).normal(0, 1, 256).astype(np.float32); l2[17] = -np.inf       # a -inf logit is legal
    f = np.diff(q.quantise(l2))
    assert f[17] == 1 and f.sum() == 65536


def test_find_symbol_brute_force_and_division_free_identity():
    g = rng(6)
    l = (g.normal(0, 5, (40, 256))).astype(np.float32)
    C = q.quantise(l)
    # rebuild g, G, T the way the rule states, independently of quantise()'s internals
    e = np.exp((l - l.max(-1, keepdims=True)).astype(np.float64))
    for r in range(40):
        xs = np.concatenate([g.integers(0, 65536, 300), C[r, :-1], C[r, 1:] - 1])
        for x in xs:
            s = q.find_symbol(C[r], int(x))
            assert C[r, s] <= x < C[r, s + 1]
            brute = max(a for a in range(256) if C[r, a] <= x)
            assert s == brute
    # C[a] <= x  <=>  a <= x  and  G[a]*65280 < (x-a+1)*T      (floor(n/T) <= y  <=>  n < (y+1) T)
    gq = np.minimum(np.floor(q.exp_f32_spec((l - l.max(-1, keepdims=True)).astype(np.float32)).astype(np.float64) * 2 ** 23), 2 ** 23).astype(np.int64)
    G = np.concatenate([np.zeros((40, 1), np.int64), np.cumsum(gq, -1)], -1)
    T = G[:, -1]
    assert np.max(np.abs(gq / 2.0 ** 23 - e)) < 1e-6
    for r in range(40):
        for x in np.concatenate([g.integers(0, 65536, 200), C[r, 1:-1], C[r, 1:-1] - 1]):
            x = int(x)
            for a in range(0, 257, 7):
                lhs = C[r, a] <= x
                rhs = a <= x and int(G[r, a]) * 65280 < (x - a + 1) * int(T[r])
                assert lhs == rhs


def test_exp2_coefficients_in_exact_arithmetic():
    """Pins EXP2_COEF independently of both transcriptions of the EXP recipe (oracle/quantise.py, coder_kernels.cuh):
    the seven binary32 constants, evaluated as EXACT rationals (no fp32 rounding anywhere), against 2^r at 50 digits
    on a dense grid of r in [-1/2, 1/2].  A wrong hex digit in c0..c4 breaks the bound; c0 = 1 makes EXP(0) = 1 exact
    (the arg-max gets g = 2^23, R#5); c1 is the binary32 nearest to ln 2; and the whole polynomial stays within 2e-8
    (relative) of the continuous least-squares fit of 2^r with c0 fixed, which is how such a table is regenerated."""
    from fractions import Fraction
    import mpmath as mp
    mp.mp.dps = 50
    c = [Fraction(float(v)) for v in q.EXP2_COEF]               # binary32 -> exact rational
    assert len(c) == 7 and c[0] == 1
    ln2 = mp.log(2)
    c1 = np.float32(float(ln2))
    assert q.EXP2_COEF[1] == c1 and abs(mp.mpf(float(c1)) - ln2) <= mp.mpf(2) ** -25   # nearest binary32 to ln 2
    assert q.LOG2E == np.float32(float(1 / ln2))

    def poly(r):
        p = c[6]
        for j in range(5, -1, -1):
            p = p * r + c[j]
        return p

    worst = mp.mpf(0)
    for i in range(-4096, 4097):
        p = poly(Fraction(i, 8192))
        rel = abs(mp.mpf(p.numerator) / mp.mpf(p.denominator) / mp.power(2, mp.mpf(i) / 8192) - 1)
        worst = max(worst, rel)
    assert worst <= mp.mpf("1.6e-8"), worst                     # documented: 1.0e-7 incl. the fp32 rounding of Horner
    # independent derivation: least squares of (sum_{k>=1} c_k r^k - (2^r - 1)) * 2^-r over [-1/2, 1/2] (c0 = 1 fixed)
    ks = range(1, 7)
    A, b = mp.matrix(6, 6), mp.matrix(6, 1)
    for a_, ka in enumerate(ks):
        for b_, kb in enumerate(ks):
            A[a_, b_] = mp.quad(lambda x: 4 ** (-x) * x ** (ka + kb), [-0.5, 0.5])
        b[a_] = mp.quad(lambda x: 4 ** (-x) * x ** ka * (2 ** x - 1), [-0.5, 0.5])
    fit = mp.lu_solve(A, b)
    for i in range(-64, 65):
        r = mp.mpf(i) / 128
        d = sum((mp.mpf(float(q.EXP2_COEF[k])) - fit[k - 1]) * r ** k for k in ks)
        assert abs(d) <= mp.mpf("2e-8"), (i, d)
    # sensitivity: the bound does notice a single wrong hex digit (16 ulp) in c2
    bad = list(c)
    bad[2] = Fraction(float(np.array(0x3E75FDFE, np.uint32).view(np.float32)))
    pb = bad[6]
    for j in range(5, -1, -1):
        pb = pb * Fraction(1, 2) + bad[j]
    assert abs(mp.mpf(pb.numerator) / mp.mpf(pb.denominator) / mp.sqrt(2) - 1) > mp.mpf("1.6e-8")
