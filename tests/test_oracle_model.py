"""Pins for oracle/model.py (O1) against things other than itself: torch library routines, direct
sums, an unrolled brute force, a closed form, and an independent sequence-mode implementation."""
import numpy as np
import pytest
import torch
import torch.nn.functional as F

from oracle import model
from paper_2511_11337_b200 import synth


def rng(seed=0):
    return np.random.Generator(np.random.PCG64(seed))


def test_elementwise_against_torch_fp64():
    x = rng(1).normal(0, 3, 1000)
    x[:4] = [0.0, 40.0, -40.0, 800.0]
    t = torch.tensor(x, dtype=torch.float64)
    np.testing.assert_allclose(model.silu(x), F.silu(t).numpy(), rtol=1e-14, atol=1e-300)
    np.testing.assert_allclose(model.softplus(x[:3]), F.softplus(t[:3], threshold=1e9).numpy(), rtol=1e-14)
    np.testing.assert_allclose(model.softplus(x[4:]), F.softplus(t[4:], threshold=1e9).numpy(), rtol=1e-14)
    np.testing.assert_allclose(model.sigmoid(x), torch.sigmoid(t).numpy(), rtol=1e-14, atol=1e-300)
    assert model.softplus(np.array([800.0]))[0] == 800.0 and np.isfinite(model.softplus(np.array([-800.0]))[0])


def test_rmsnorm_against_torch():
    g = rng(2)
    u, w = g.normal(0, 2, (5, 64)), g.normal(1, 0.1, 64)
    ref = F.rms_norm(torch.tensor(u), (64,), torch.tensor(w), eps=1e-5).numpy()
    np.testing.assert_allclose(model.rmsnorm(u, w), ref, rtol=1e-13)


def test_conv_step_against_conv1d_and_direct_sum():
    g = rng(3)
    S, E, K, T = 3, 8, 4, 11
    x = g.normal(0, 1, (S, T, E))
    cw, cb = g.normal(0, 1, (E, K)), g.normal(0, 1, E)
    win = np.zeros((S, K - 1, E))
    got = np.empty((S, T, E))
    for t in range(T):
        got[:, t], win = model.conv_step(win, x[:, t], cw, cb)
    # library routine: causal depthwise conv = conv1d(padding=K-1, groups=E) cropped to T
    ref = F.conv1d(torch.tensor(x).transpose(1, 2), torch.tensor(cw)[:, None, :], torch.tensor(cb),
                   padding=K - 1, groups=E)[:, :, :T].transpose(1, 2).numpy()
    np.testing.assert_allclose(got, ref, rtol=1e-13, atol=1e-14)
    # direct sum with explicit indices: tap k multiplies x_{t-(K-1)+k}
    for t in (0, 2, 7):
        for e in (0, 5):
            acc = cb[e]
            for k in range(K):
                j = t - (K - 1) + k
                if j >= 0:
                    acc += cw[e, k] * x[1, j, e]
            assert abs(acc - got[1, t, e]) < 1e-13
    # the window holds the last K-1 inputs, oldest first
    np.testing.assert_array_equal(win, x[:, T - (K - 1):, :])


def test_ssm_step_against_unrolled_brute_force():
    g = rng(4)
    S, E, N, T = 2, 3, 4, 7
    a = -np.exp(g.normal(0, 0.5, (E, N)))
    d_skip = g.normal(0, 1, E)
    delta = np.exp(g.normal(-1, 0.5, (T, S, E)))
    bv, cv, xs = g.normal(0, 1, (T, S, N)), g.normal(0, 1, (T, S, N)), g.normal(0, 1, (T, S, E))
    h = np.zeros((S, E, N))
    ys = []
    for t in range(T):
        h, y = model.ssm_step(h, xs[t], delta[t], bv[t], cv[t], a, d_skip)
        ys.append(y)
    # h_T = sum_j (prod_{i>j} exp(delta_i A)) delta_j B_j x_j     (eq. 18 unrolled)
    for s in range(S):
        for e in range(E):
            for n in range(N):
                tot = 0.0
                for j in range(T):
                    prod = 1.0
                    for i in range(j + 1, T):
                        prod *= np.exp(delta[i, s, e] * a[e, n])
                    tot += prod * delta[j, s, e] * bv[j, s, n] * xs[j, s, e]
                assert abs(tot - h[s, e, n]) < 1e-12
            # y_T = C_T . h_T + D x_T   (eq. 19)
            assert abs(np.dot(cv[T - 1, s], h[s, e]) + d_skip[e] * xs[T - 1, s, e] - ys[-1][s, e]) < 1e-12


def test_ssm_step_closed_form_constant_input():
    # constant delta, B, x = 1:  h_T = delta*B*(1 - a^T)/(1 - a),  a = exp(delta*A)   (geometric series)
    E, N, T = 2, 3, 25
    a_mat = -np.array([[1.0, 2.0, 3.0], [0.5, 1.5, 16.0]])
    delta = np.full((1, E), 0.07)
    bv = np.array([[0.3, -1.1, 2.0]])
    cv = np.zeros((1, N))
    xs = np.ones((1, E))
    h = np.zeros((1, E, N))
    for _ in range(T):
        h, _y = model.ssm_step(h, xs, delta, bv, cv, a_mat, np.zeros(E))
    abar = np.exp(0.07 * a_mat)
    ref = 0.07 * bv[0][None, :] * (1 - abar ** T) / (1 - abar)
    np.testing.assert_allclose(h[0], ref, rtol=1e-12)


def _sequence_mode_logits(blob, chunks):
    """Independent implementation: whole sequence at once in torch fp64 — matmuls batched over time,
    conv by F.conv1d, the recurrence through its closed-form sum with cumulative log-decays."""
    shape, dtype, _ = synth.parse_header(blob)
    D, E, N, K, R = shape.d_model, shape.d_inner, shape.d_state, shape.d_conv, shape.rank
    off = 64
    tens = {}
    for name, dims, is_mat in synth.tensor_order(shape):
        cnt = int(np.prod(dims))
        if is_mat and dtype == synth.DTYPE_BF16:
            a = synth.bf16_bits_to_f32(np.frombuffer(blob, "<u2", cnt, off)).astype(np.float64)
            off += 2 * cnt + (-2 * cnt) % 16
        else:
            a = np.frombuffer(blob, "<f4", cnt, off).astype(np.float64)
            off += 4 * cnt + (-4 * cnt) % 16
        tens[name] = torch.tensor(a.reshape(dims))
    x_in = torch.tensor(chunks[:, :-1].astype(np.int64))
    S, T = x_in.shape
    u = tens["emb"][x_in]                                             # [S,T,D]
    for l in range(shape.n_layer):
        p = f"l{l}."
        r = F.rms_norm(u, (D,), tens[p + "norm_w"], eps=1e-5)
        xz = torch.einsum("std,fd->stf", r, tens[p + "w_in"])
        x, z = xz[..., :E], xz[..., E:]
        xc = F.conv1d(x.transpose(1, 2), tens[p + "conv_w"][:, None, :], tens[p + "conv_b"],
                      padding=K - 1, groups=E)[:, :, :T].transpose(1, 2)
        xs = F.silu(xc)
        dbc = torch.einsum("ste,fe->stf", xs, tens[p + "w_x"])
        dl, bv, cv = dbc[..., :R], dbc[..., R:R + N], dbc[..., R + N:]
        delta = F.softplus(torch.einsum("str,er->ste", dl, tens[p + "w_dt"]) + tens[p + "b_dt"], threshold=1e9)
        A = -torch.exp(tens[p + "a_log"])                             # [E,N]
        logdec = delta[..., None] * A                                 # [S,T,E,N], log of per-step decay
        cum = torch.cumsum(logdec, dim=1)                             # sum_{i<=t}
        inp = delta[..., None] * bv[:, :, None, :] * xs[..., None]    # [S,T,E,N]
        # h_t = sum_{j<=t} exp(cum_t - cum_j) inp_j
        w8 = torch.exp(cum[:, :, None] - cum[:, None, :])             # [S,T(t),T(j),E,N]
        mask = torch.tril(torch.ones(T, T, dtype=torch.float64))[None, :, :, None, None]
        h = torch.sum(w8 * mask * inp[:, None], dim=2)                # [S,T,E,N]
        y = torch.einsum("sten,stn->ste", h, cv) + tens[p + "d_skip"] * xs
        y = y * F.silu(z)
        u = u + torch.einsum("ste,de->std", y, tens[p + "w_out"])
        if shape.d_ff:                                                # Alg. 1 l.4 with library routines
            hid = F.gelu(F.linear(u, tens[p + "ffn_w1"], tens[p + "ffn_b1"]))
            u = F.layer_norm(F.linear(hid, tens[p + "ffn_w2"], tens[p + "ffn_b2"]), (D,),
                             tens[p + "ln_w"], tens[p + "ln_b"], eps=1e-5)
    return torch.einsum("std,vd->stv", u, tens["emb" if shape.tied else "head"]).numpy()


@pytest.mark.parametrize("dtype,emb_std", [(synth.DTYPE_FP32, None), (synth.DTYPE_BF16, 0.25)])
def test_step_mode_against_sequence_mode(dtype, emb_std):
    shape = synth.ModelShape(2, 32, dt_rank=2)
    blob = synth.make_weights(shape, 7, dtype, std=0.2, emb_std=emb_std)
    chunks = rng(5).integers(0, 256, (3, 20), dtype=np.uint8)
    got = model.logits_for_chunks(model.load_weights(blob), chunks)
    ref = _sequence_mode_logits(blob, chunks)
    assert np.max(np.abs(ref)) > 0.05          # non-trivial logits
    np.testing.assert_allclose(got, ref, rtol=1e-10, atol=1e-11)


@pytest.mark.parametrize("tied", [True, False])
def test_paper_block_step_mode_against_sequence_mode(tied):
    # FFN + LayerNorm after every mixer (Alg. 1 l.4), tied and untied head
    shape = synth.ModelShape(2, 32, dt_rank=2, d_ff=96, tied=tied)
    blob = synth.make_weights(shape, 11, synth.DTYPE_FP32, std=0.2, emb_std=0.3)
    chunks = rng(6).integers(0, 256, (3, 17), dtype=np.uint8)
    w = model.load_weights(blob)
    got = model.logits_for_chunks(w, chunks)
    ref = _sequence_mode_logits(blob, chunks)
    assert np.max(np.abs(ref)) > 0.05
    np.testing.assert_allclose(got, ref, rtol=1e-10, atol=1e-11)
    # the block is not the north_star block in disguise: dropping the FFN flag's tensors changes the logits
    plain = synth.make_weights(synth.ModelShape(2, 32, dt_rank=2), 11, synth.DTYPE_FP32, std=0.2, emb_std=0.3)
    other = model.logits_for_chunks(model.load_weights(plain), chunks)
    assert np.max(np.abs(other - got)) > 1e-3


def test_gelu_against_library_and_identities():
    from scipy.stats import norm
    x = rng(8).normal(0, 2.5, 500)
    x[:3] = [0.0, 30.0, -30.0]
    # (the erf form cancels in the far negative tail: absolute, not relative, agreement there)
    np.testing.assert_allclose(model.gelu(x), x * norm.cdf(x), rtol=1e-12, atol=1e-15)         # v Phi(v)
    np.testing.assert_allclose(model.gelu(x), F.gelu(torch.tensor(x)).numpy(), rtol=1e-12, atol=1e-15)
    np.testing.assert_allclose(model.gelu(x) - model.gelu(-x), x, rtol=1e-12, atol=1e-15)      # Phi(v) + Phi(-v) = 1
    assert model.gelu(np.array([0.0]))[0] == 0.0 and model.gelu(np.array([30.0]))[0] == 30.0
    assert abs(model.gelu(np.array([1.0]))[0] - 0.8413447460685429) < 1e-15                   # Phi(1)


def test_layernorm_against_torch_and_invariants():
    g = rng(9)
    v, w, b = g.normal(3, 2, (5, 48)), g.normal(1, 0.2, 48), g.normal(0, 0.3, 48)
    ref = F.layer_norm(torch.tensor(v), (48,), torch.tensor(w), torch.tensor(b), eps=1e-5).numpy()
    np.testing.assert_allclose(model.layernorm(v, w, b), ref, rtol=1e-12, atol=1e-14)
    plain = model.layernorm(v, np.ones(48), np.zeros(48))
    np.testing.assert_allclose(plain.mean(axis=1), 0.0, atol=1e-14)
    var = v.var(axis=1)                                                   # biased
    np.testing.assert_allclose(plain.var(axis=1), var / (var + 1e-5), rtol=1e-12)
    # invariant to a shift of the input, scales out a positive factor (up to eps)
    np.testing.assert_allclose(model.layernorm(v + 7.0, w, b), model.layernorm(v, w, b), rtol=1e-9, atol=1e-12)


def test_ffn_against_direct_sum():
    import math
    g = rng(10)
    D, Fh = 6, 10
    ly = model.Layer(*[None] * 10)
    ly.ffn_w1, ly.ffn_b1 = g.normal(0, 1, (Fh, D)), g.normal(0, 1, Fh)
    ly.ffn_w2, ly.ffn_b2 = g.normal(0, 1, (D, Fh)), g.normal(0, 1, D)
    u = g.normal(0, 1, (2, D))
    got = model.ffn(u, ly)
    for s in range(2):
        for d in range(D):
            acc = ly.ffn_b2[d]
            for j in range(Fh):
                pre = ly.ffn_b1[j] + sum(ly.ffn_w1[j, k] * u[s, k] for k in range(D))
                acc += ly.ffn_w2[d, j] * 0.5 * pre * (1.0 + math.erf(pre / math.sqrt(2.0)))
            assert abs(acc - got[s, d]) < 1e-12


def test_load_weights_slots_paper_block():
    shape = synth.ModelShape(1, 16, dt_rank=1, d_ff=24, tied=False)
    D, E, N, K, R, Fh = 16, 32, 16, 4, 1, 24
    total = sum(int(np.prod(d)) for _, d, _ in synth.tensor_order(shape))
    import struct
    hdr = struct.pack("<4s10I", b"BOAW", 1, 0, 1, D, N, K, 2, R, 2, Fh).ljust(64, b"\0")
    w = model.load_weights(hdr + np.arange(total, dtype="<f4").tobytes())
    ly = w.layers[0]
    off = 256 * D + D + 2 * E * D + E * K + E + (R + 2 * N) * E + E * R + E + E * N + E + D * E
    for arr, shp in [(ly.ffn_w1, (Fh, D)), (ly.ffn_b1, (Fh,)), (ly.ffn_w2, (D, Fh)), (ly.ffn_b2, (D,)),
                     (ly.ln_w, (D,)), (ly.ln_b, (D,)), (w.head, (256, D))]:
        assert arr.shape == shp and arr.reshape(-1)[0] == off and arr.reshape(-1)[-1] == off + arr.size - 1
        off += arr.size
    assert off == total
    # flag and width must agree
    bad = struct.pack("<4s10I", b"BOAW", 1, 0, 1, D, N, K, 2, R, 2, 0).ljust(64, b"\0")
    with pytest.raises(ValueError):
        model.load_weights(bad + np.arange(total, dtype="<f4").tobytes())


def test_load_weights_slots():
    # a hand-built blob whose k-th stored value is k: every tensor must land in its documented slot
    shape = synth.ModelShape(1, 16, dt_rank=1)
    D, E, N, K, R = 16, 32, 16, 4, 1
    total = sum(int(np.prod(d)) for _, d, _ in synth.tensor_order(shape))
    import struct
    hdr = struct.pack("<4s9I", b"BOAW", 1, 0, 1, D, N, K, 2, R, 1).ljust(64, b"\0")
    blob = hdr + np.arange(total, dtype="<f4").tobytes()
    w = model.load_weights(blob)
    assert w.emb.shape == (256, D) and w.emb[1, 0] == D
    off = 256 * D
    ly = w.layers[0]
    for arr, shp in [(ly.norm_w, (D,)), (ly.w_in, (2 * E, D)), (ly.conv_w, (E, K)), (ly.conv_b, (E,)),
                     (ly.w_x, (R + 2 * N, E)), (ly.w_dt, (E, R)), (ly.b_dt, (E,)), (ly.a_log, (E, N)),
                     (ly.d_skip, (E,)), (ly.w_out, (D, E))]:
        assert arr.shape == shp and arr.reshape(-1)[0] == off and arr.reshape(-1)[-1] == off + arr.size - 1
        off += arr.size
    with pytest.raises(ValueError):
        model.load_weights(blob + b"\0" * 16)


def test_bf16_weights_are_widened_exactly():
    shape = synth.ModelShape(1, 16, dt_rank=1)
    blob = synth.make_weights(shape, 3, synth.DTYPE_BF16)
    w = model.load_weights(blob)
    bits = w.emb.astype(np.float32).view(np.uint32)
    assert np.all(bits & 0xFFFF == 0) and np.all(w.emb == w.emb.astype(np.float32))
    assert np.std(w.emb) == pytest.approx(0.02, rel=0.1)
