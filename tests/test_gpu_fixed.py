"""GPU parity of FX1, the deterministic fixed-point pipeline, against its
exact-integer oracle (oracle/fixed.py).  Integer arithmetic has one correct answer, so the bar is equality: the load-time
quantisation, the logits of every step (int32, Q12.20), the tables, and whole containers byte for byte - the GPU decodes
what the oracle encoded and the oracle decodes what the GPU encoded."""
import numpy as np
import pytest
import torch

from oracle import container, fixed as fx, model
from paper_2511_11337_b200 import synth

pytestmark = pytest.mark.gpu


def _np(t):
    return t.detach().cpu().numpy()


def _cases():
    s1 = synth.CONFIGS[1]
    return {
        "cfg1": s1.weights(),
        "cfg1_sharp": s1.weights(emb_std=0.25),
        "d128_l2_bf16_sharp": synth.make_weights(synth.ModelShape(2, 128, dt_rank=8), 7, synth.DTYPE_BF16, emb_std=0.25),
        "d192_l1_sharp": synth.make_weights(synth.ModelShape(1, 192), 5, emb_std=0.25),          # dt_rank 12, J = 44
        "cfg2_shape_sharp": synth.make_weights(synth.CONFIGS[2].shape, 1, emb_std=0.25),
        "cfg5_shape_l2_sharp": synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25),
        "wide_scales": synth.make_weights(synth.ModelShape(1, 64, dt_rank=4), 31, std=0.5, emb_std=2.0),   # saturation is reached
        # the widest model FX1 accepts: K = 2048 = 16 k-blocks (the contraction's 8-stage ring is refilled), dt_rank 64
        "d1024_r64_bf16_sharp": synth.make_weights(synth.ModelShape(1, 1024, dt_rank=64), 11, synth.DTYPE_BF16, emb_std=0.25),
    }


@pytest.fixture(scope="module", params=list(_cases()))
def case(request, boa):
    blob = _cases()[request.param]
    return request.param, boa.FxModel(blob), fx.quantise_model(model.load_weights(blob))


def test_logits_and_tables_bit_exact(case):
    name, gm, q = case
    S, T = 5, 40
    data = np.frombuffer(synth.CONFIGS[1].data(S * T), np.uint8).reshape(S, T)
    d = gm.debug_step_dump(data.tobytes(), T, T - 1)
    st = fx.init_state(q, S)
    for t in range(T - 1):
        want = fx.step(q, st, data[:, t])
        got = _np(d["logits"][:, t]).astype(np.int64)
        assert np.array_equal(got, want), (name, t, int(np.abs(got - want).max()))
        assert np.array_equal(_np(d["cdf"][:, t]).astype(np.int64), fx.table(want)), (name, t)


def test_containers_byte_identical_both_ways(case, boa):
    name, gm, q = case
    chunk = 48
    data = synth.CONFIGS[1].data(6 * chunk + 17)                  # ragged last chunk
    want = fx.compress(q, data, chunk)
    got = _np(gm.compress(data, chunk)).tobytes()
    assert got == want, name                                       # same bytes incl. the 'FX01' fingerprint and the index CRC
    assert gm.fingerprint == fx.fingerprint(q)
    assert _np(gm.decompress(torch.frombuffer(bytearray(want), dtype=torch.uint8).cuda())).tobytes() == data
    assert fx.decompress(q, got) == data
    # host pointers
    assert _np(gm.compress(data, chunk, device="cpu")).tobytes() == want


def test_fx_edges_errors_and_batch_independence(boa):
    cfg = synth.CONFIGS[1]
    blob = cfg.weights(emb_std=0.25)
    gm = boa.FxModel(blob)
    assert gm.compress(b"", 64).numel() == 44 and gm.decompress(gm.compress(b"", 64)).numel() == 0
    for n, chunk in [(1, 64), (5, 1), (300, 2), (1000, 7)]:
        data = cfg.data(n)
        assert _np(gm.decompress(gm.compress(data, chunk))).tobytes() == data, (n, chunk)
    data = cfg.data(140 * 30)                                      # 140 streams: more than one 128-row tile of the contraction
    _, _, _, _, pa = container.unpack(_np(gm.compress(data, 30)).tobytes())
    for i in (0, 63, 64, 127, 128, 139):
        _, _, _, _, ps = container.unpack(_np(gm.compress(data[i * 30:(i + 1) * 30], 30)).tobytes())
        assert ps[0] == pa[i], i
    # an FX1 container and a floating-point model reject each other
    fm = boa.Model(blob)
    comp = gm.compress(cfg.data(500), 100)
    with pytest.raises(boa.BoaError) as e:
        fm.decompress(comp)
    assert e.value.code == boa.E_MODEL_MISMATCH
    with pytest.raises(boa.BoaError) as e:
        gm.decompress(fm.compress(cfg.data(500), 100))
    assert e.value.code == boa.E_MODEL_MISMATCH
    with pytest.raises(boa.BoaError) as e:                         # the paper's block is outside FX1
        boa.FxModel(synth.make_weights(synth.ModelShape(1, 64, dt_rank=4, d_ff=64), 1))
    assert e.value.code == boa.E_UNSUPPORTED


def test_fx_round_trip_at_scale(boa):
    """4,096 streams x 200 bytes of the config-2 input through the cfg2-shaped model: byte-exact round trip, and a sampled
    stream's payload equals the oracle's."""
    cfg = synth.CONFIGS[2]
    blob = cfg.weights()
    gm = boa.FxModel(blob)
    B, T = 4096, 200
    data = cfg.data(B * T)
    src = torch.frombuffer(bytearray(data), dtype=torch.uint8).cuda()
    comp = gm.compress(src, T)
    assert torch.equal(gm.decompress(comp), src)
    q = fx.quantise_model(model.load_weights(blob))
    _, _, _, _, pays = container.unpack(_np(comp).tobytes(), gm.fingerprint)
    for i in (0, 4095):
        _, _, _, _, p1 = container.unpack(fx.compress(q, data[i * T:(i + 1) * T][:60], 60))
        # (the first 60 bytes of the stream alone: the oracle is slow; the GPU payload of that prefix must be the same bytes)
        _, _, _, _, g1 = container.unpack(_np(gm.compress(data[i * T:(i + 1) * T][:60], 60)).tobytes())
        assert g1[0] == p1[0], i
    assert len(pays) == B


def test_fx_more_chunks_than_one_wave(boa):
    """70,001 chunks of 3 bytes: more than the 65,536 streams a wave steps together, so the second wave starts at a stream
    offset inside the input, the size index and the payload.  Byte-exact round trip, and chunks on both sides of the wave
    boundary code to the bytes they get when compressed alone (a stream does not depend on its neighbours)."""
    cfg = synth.CONFIGS[1]
    gm = boa.FxModel(cfg.weights(emb_std=0.25))
    chunk, nc = 3, 70001
    data = cfg.data(nc * chunk - 1)                                # ragged last chunk (2 bytes)
    comp = gm.compress(data, chunk)
    assert _np(gm.decompress(comp)).tobytes() == data
    _, _, _, _, pa = container.unpack(_np(comp).tobytes())
    assert len(pa) == nc
    for i in (0, 65535, 65536, 70000):
        _, _, _, _, ps = container.unpack(_np(gm.compress(data[i * chunk:(i + 1) * chunk], chunk)).tobytes())
        assert ps[0] == pa[i], i
