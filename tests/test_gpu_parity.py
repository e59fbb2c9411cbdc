"""GPU parity tests (run on the B200 box with -m gpu): the CUDA path, called through the C ABI, against the
CPU oracle on the same seeded inputs.  The four checks of BASELINE.json's north_star plus the table rule:

  1. range coder bit-exact with the oracle's, given the oracle's frequency tables
  2. probabilities within max-abs 1e-5 of the oracle's (fp64)
  3. compressed size within 0.5 % of the oracle's
  4. GPU compress -> GPU decompress byte-exact on every input
  5. integer tables bit-exact with the oracle's rule applied to the same fp32 logits (a float decides an
     integer there, so both sides take the decision in fp32 by the same specified EXP, R#5)
"""
import numpy as np
import pytest
import torch

from oracle import codec, container, model, quantise, rangecoder
from paper_2511_11337_b200 import synth

pytestmark = pytest.mark.gpu

PROB_TOL = 1e-5      # north_star: "probabilities must be within max-abs 1e-5 of the oracle's"
SIZE_TOL = 0.005     # north_star: "compressed size must be within 0.5% of the oracle's"


def _np(t):
    return t.detach().cpu().numpy()


def _cases():
    s1 = synth.CONFIGS[1]
    s2 = synth.CONFIGS[2]
    small2 = synth.ModelShape(2, 128, dt_rank=8)
    return {
        "cfg1": (s1.weights(), s1),
        "cfg1_sharp": (s1.weights(emb_std=0.25), s1),
        "d128_l2_bf16_sharp": (synth.make_weights(small2, 7, synth.DTYPE_BF16, emb_std=0.25), s1),
        "cfg2_shape_sharp": (synth.make_weights(s2.shape, 1, emb_std=0.25), s2),
        # E = 384: three 128-channel scan slices, dt_rank 12 (W_dt row in shared memory), ragged x_proj tile
        "d192_l1_sharp": (synth.make_weights(synth.ModelShape(1, 192), 5, emb_std=0.25), s1),
        # the cfg4 / cfg5 model shapes (bf16 matrices): 4 layers at D = 256; D = 512, dt_rank 32, four scan slices
        "cfg4_shape_sharp": (synth.make_weights(synth.CONFIGS[4].shape, 2, synth.DTYPE_BF16, emb_std=0.25), s2),
        "cfg5_shape_l2_sharp": (synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25), s2),
        # SURVEY 8(f) NEXT-2, the paper's own block (Alg. 1 l.4): FFN + LayerNorm after every mixer.  The paper's
        # shape (1 layer, D = 256, hidden 1024, untied head, fp32), and two layers with bf16 matrices, a tied head and
        # a hidden width that is not a power of two
        "paper_block_sharp": (synth.make_weights(synth.CONFIGS[6].shape, 4, emb_std=0.25, ffn_std=0.1), s2),
        "paper_block_l2_d128_bf16_sharp": (synth.make_weights(synth.ModelShape(2, 128, dt_rank=8, d_ff=320), 9, synth.DTYPE_BF16,
                                                              emb_std=0.25, ffn_std=0.1), s1),
        # the ends of k_layernorm's lane map: D = 64 (half a warp holds the row) and D = 512 (four float4 per lane)
        "paper_block_d64_sharp": (synth.make_weights(synth.ModelShape(1, 64, dt_rank=4, d_ff=64, tied=False), 12,
                                                     emb_std=0.25, ffn_std=0.1), s1),
        "paper_block_d512_bf16_sharp": (synth.make_weights(synth.ModelShape(1, 512, dt_rank=32, d_ff=128), 13, synth.DTYPE_BF16,
                                                           emb_std=0.25, ffn_std=0.1), s2),
    }


@pytest.fixture(scope="module", params=list(_cases()))
def case(request, boa):
    blob, cfg = _cases()[request.param]
    return request.param, blob, cfg, boa.Model(blob), model.load_weights(blob)


# ---------------------------------------------------------------------------------------------- check 5
def test_quantiser_bit_exact_on_given_logits(boa):
    g = np.random.Generator(np.random.PCG64(11))
    rows = []
    rows.append(g.normal(0, 0.02, (300, 256)))                    # near-uniform regime of the configured weights
    rows.append(g.normal(0, 3.0, (300, 256)))                     # sharp
    rows.append(g.normal(0, 30.0, (300, 256)))                    # f = 1 floor everywhere but a few symbols
    rows.append(np.zeros((1, 256)))                               # uniform -> f = 256
    one = np.full((1, 256), -100.0); one[0, 17] = 5.0             # one-hot -> 65281 + 255 ones
    tie = np.full((1, 256), -100.0); tie[0, [3, 200]] = 1.0       # two-way tie -> 32641 each
    bad = np.zeros((3, 256)); bad[0, 5] = np.nan; bad[1, 9] = np.inf; bad[2, :] = -np.inf
    neg = np.zeros((1, 256)); neg[0, 100] = -np.inf               # -inf below a finite max is legal
    logits = np.concatenate(rows + [one, tie, bad, neg]).astype(np.float32)
    want = quantise.quantise(logits)
    got = _np(boa.debug_quantise(torch.from_numpy(logits).cuda())).astype(np.int64)
    assert np.array_equal(got, want)
    f = np.diff(got, axis=1)
    assert f.min() >= 1 and np.all(got[:, 0] == 0) and np.all(got[:, 256] == 65536)
    assert np.all(f[900] == 256) and f[901, 17] == 65281 and f[902, 3] == f[902, 200] == 32641
    assert np.all(f[903:906] == 256)


# ------------------------------------------------------------------- the tensor-core contraction kernel alone
def _to_bf16(x):
    u = np.ascontiguousarray(x, np.float32).view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32)


@pytest.mark.parametrize("pieces,grid_ctas", [(3, 0), (3, 3), (1, 0), (1, 2)])
@pytest.mark.parametrize("M,N,K", [(300, 48, 512), (128, 256, 64), (1, 64, 256), (517, 320, 1024)])
def test_tensor_core_gemm_against_fp64(boa, pieces, grid_ctas, M, N, K):
    """C = A W^T by tcgen05 on bf16 pieces (tc_gemm.cuh) against numpy fp64 matmul: every product is kept to
    ~2^-24, so the error is bounded by a few ulp of sum_k |a||w| (several tiles, ragged M, padded N; grid_ctas > 0
    makes each persistent CTA walk over several tiles, i.e. both TMEM accumulator buffers and the stage ring wrap)."""
    g = np.random.Generator(np.random.PCG64(M * 7 + N * 3 + K + pieces))
    a = (g.normal(0, 1.0, (M, K)) * np.exp(g.normal(0, 2.0, (M, 1)))).astype(np.float32)   # rows of very different scale
    w = g.normal(0, 0.05, (N, K)).astype(np.float32)
    if pieces == 1:
        w = _to_bf16(w)                                             # a bf16 blob: one exact piece
    want = a.astype(np.float64) @ w.astype(np.float64).T
    scale = np.abs(a).astype(np.float64) @ np.abs(w).astype(np.float64).T
    got = _np(boa.debug_gemm(torch.from_numpy(a).cuda(), torch.from_numpy(w), pieces, grid_ctas)).astype(np.float64)
    err = np.abs(got - want) / scale
    assert err.max() <= 2.0 ** -20, (err.max(), np.unravel_index(err.argmax(), err.shape))
    # and from host pointers
    got_h = _np(boa.debug_gemm(torch.from_numpy(a), torch.from_numpy(w), pieces, grid_ctas))
    assert np.array_equal(got_h.astype(np.float64), got)


@pytest.mark.parametrize("pieces", [3, 1])
@pytest.mark.parametrize("M,N,K", [(300, 48, 512), (128, 256, 64), (1, 64, 256), (517, 320, 1024), (700, 192, 128), (2100, 1024, 256)])
def test_cta_pair_gemm_returns_the_bits_of_the_single_cta_gemm(boa, pieces, M, N, K):
    """The step path multiplies with CTA-pair tiles (tc_gemm2.cuh: tcgen05 cta_group::2, 256 x 128), the encode-side time
    slabs with single-CTA tiles (tc_gemm.cuh: 128 x 64).  Both issue, per output element, the same piece products into
    the same accumulator classes in the same order, so they must agree bit for bit (the decoder steps, the encoder
    runs slabs) - for odd numbers of row tiles and of 64-column weight tiles (a pair with a missing half), one tile per
    pair and several tiles per pair (accumulator and stage rings wrap), and against numpy fp64."""
    g = np.random.Generator(np.random.PCG64(M * 5 + N * 11 + K + pieces))
    a = (g.normal(0, 1.0, (M, K)) * np.exp(g.normal(0, 2.0, (M, 1)))).astype(np.float32)
    w = g.normal(0, 0.05, (N, K)).astype(np.float32)
    if pieces == 1:
        w = _to_bf16(w)
    ad, wt = torch.from_numpy(a).cuda(), torch.from_numpy(w)
    single = _np(boa.debug_gemm(ad, wt, pieces, 0))
    for grid in (-1, -2, -6):
        pair = _np(boa.debug_gemm(ad, wt, pieces, grid))
        assert np.array_equal(pair.view(np.uint32), single.view(np.uint32)), (grid, np.abs(pair - single).max())
    want = a.astype(np.float64) @ w.astype(np.float64).T
    scale = np.abs(a).astype(np.float64) @ np.abs(w).astype(np.float64).T
    assert (np.abs(single - want) / scale).max() <= 2.0 ** -20


@pytest.mark.parametrize("shape", ["cfg1", "d192_l1", "cfg2", "cfg5_l2_bf16", "paper_block_d64", "paper_block_l2_d128_bf16"])
def test_pair_tiles_and_single_tiles_write_the_same_container(boa, shape):
    """The whole step path with CTA-pair tiles forced on (every contraction incl. the conv epilogue of in_proj, the
    residual epilogue and the FFN) against single-CTA tiles: same container bytes, and either decodes the other's.
    D = 64 / 192 give contractions with an odd number of 64-column weight tiles (a pair whose second half is missing),
    300 streams an odd number of row tiles."""
    s1 = synth.CONFIGS[1]
    blob = {"cfg1": lambda: s1.weights(emb_std=0.25),
            "d192_l1": lambda: synth.make_weights(synth.ModelShape(1, 192), 5, emb_std=0.25),
            "cfg2": lambda: synth.make_weights(synth.CONFIGS[2].shape, 1, emb_std=0.25),
            "cfg5_l2_bf16": lambda: synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25),
            "paper_block_d64": lambda: synth.make_weights(synth.ModelShape(1, 64, dt_rank=4, d_ff=64, tied=False), 12, emb_std=0.25, ffn_std=0.1),
            "paper_block_l2_d128_bf16": lambda: synth.make_weights(synth.ModelShape(2, 128, dt_rank=8, d_ff=320), 9, synth.DTYPE_BF16,
                                                                   emb_std=0.25, ffn_std=0.1)}[shape]()
    gm = boa.Model(blob)
    for n, chunk in [(300 * 23, 23), (5 * 50 + 7, 50), (1, 40)]:
        data = s1.data(n)
        gm.debug_set_slab(False)                                   # encode with the step kernels, like the decoder
        try:
            gm.debug_set_pair_tiles(1 << 30)
            single = gm.compress(data, chunk)
            gm.debug_set_pair_tiles(0)
            pair = gm.compress(data, chunk)
            assert torch.equal(single, pair), (shape, n, chunk)
            assert _np(gm.decompress(single)).tobytes() == data    # pair-tile decoder, single-tile encoder
            gm.debug_set_slab(True)
            assert torch.equal(gm.compress(data, chunk), pair)     # time slabs (single-CTA tiles) == pair-tile steps
            gm.debug_set_pair_tiles(1 << 30)
            assert _np(gm.decompress(pair)).tobytes() == data      # single-tile decoder, pair-tile encoder
        finally:
            gm.debug_set_slab(True)
            gm.debug_set_pair_tiles(2 ** 31 - 1)


@pytest.mark.parametrize("shape", ["cfg1", "d192_l1", "cfg2", "cfg4_bf16", "cfg5_l2_bf16"])
def test_chained_contractions_write_the_bytes_of_one_kernel_per_contraction(boa, shape):
    """The step path chains the dependent contractions between two scans inside one launch (tc::k_gemm_chain: in_proj ->
    x_proj | out_proj -> in_proj -> x_proj | out_proj -> head; row-tile counters order the work items; 2L + 2 launches per
    step instead of 4L + 2).  Against one kernel per contraction: same container, each decodes the other's; 1 ... 700
    streams (several row tiles per CTA and fewer work items than CTAs), 1 to 4 layers, fp32 and bf16 blobs."""
    s1 = synth.CONFIGS[1]
    blob = {"cfg1": lambda: s1.weights(emb_std=0.25),
            "d192_l1": lambda: synth.make_weights(synth.ModelShape(1, 192), 5, emb_std=0.25),
            "cfg2": lambda: synth.make_weights(synth.CONFIGS[2].shape, 1, emb_std=0.25),
            "cfg4_bf16": lambda: synth.make_weights(synth.CONFIGS[4].shape, 2, synth.DTYPE_BF16, emb_std=0.25),
            "cfg5_l2_bf16": lambda: synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25)}[shape]()
    gm = boa.Model(blob)
    gm.debug_set_slab(False)                                       # encode with the step path, like the decoder
    try:
        for n, chunk in [(1 * 37, 37), (5 * 41 + 13, 41), (130 * 23, 23), (700 * 19 + 5, 19)]:
            data = s1.data(n)
            gm.debug_set_chain(False)
            plain = gm.compress(data, chunk)
            n_plain = plain_launches(gm)
            gm.debug_set_chain(True)
            chained = gm.compress(data, chunk)
            assert torch.equal(plain, chained), (shape, n, chunk)
            assert plain_launches(gm) < n_plain                      # fewer launches for the same bytes
            assert _np(gm.decompress(plain)).tobytes() == data     # chained decoder
            gm.debug_set_chain(False)
            assert _np(gm.decompress(chained)).tobytes() == data   # one kernel per contraction
    finally:
        gm.debug_set_slab(True)
        gm.debug_set_chain(False)


def plain_launches(gm):
    return gm.profile()["launches_total"]


@pytest.mark.parametrize("shape", ["cfg1", "d192_l1", "cfg2", "cfg4_bf16", "cfg5_l2_bf16"])
def test_persistent_step_kernel_writes_the_bytes_of_the_graph_path(boa, shape):
    """north_star's persistent decode-step kernel (step_persist.cuh: one launch steps a small wave for all of its bytes,
    a cluster of CTAs per row tile, cluster barriers between the phases) against the graph of one kernel per phase: same
    container when encoding step by step, and each decodes the other's - for 1, 5, 64, 130 (two row tiles) and 300
    streams, clusters of 8, 4 and 1 CTAs (fewer CTAs than scan slices), ragged tails, 1 to 4 layers."""
    s1 = synth.CONFIGS[1]
    blob = {"cfg1": lambda: s1.weights(emb_std=0.25),
            "d192_l1": lambda: synth.make_weights(synth.ModelShape(1, 192), 5, emb_std=0.25),
            "cfg2": lambda: synth.make_weights(synth.CONFIGS[2].shape, 1, emb_std=0.25),
            "cfg4_bf16": lambda: synth.make_weights(synth.CONFIGS[4].shape, 2, synth.DTYPE_BF16, emb_std=0.25),
            "cfg5_l2_bf16": lambda: synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25)}[shape]()
    gm = boa.Model(blob)
    gm.debug_set_slab(False)                                       # encode with the step path, like the decoder
    try:
        for n, chunk, cluster in [(1 * 37, 37, 8), (5 * 41 + 13, 41, 8), (64 * 29, 29, 4), (130 * 23, 23, 8), (300 * 19 + 5, 19, 1), (9, 40, 8)]:
            data = s1.data(n)
            gm.debug_set_persist(0)
            graph = gm.compress(data, chunk)
            gm.debug_set_persist(1 << 20, cluster)
            pers = gm.compress(data, chunk)
            assert torch.equal(graph, pers), (shape, n, chunk, cluster)
            assert _np(gm.decompress(graph)).tobytes() == data     # persistent decoder
            gm.debug_set_persist(0)
            assert _np(gm.decompress(pers)).tobytes() == data      # graph decoder
    finally:
        gm.debug_set_slab(True)
        gm.debug_set_persist(0, 8)


# ---------------------------------------------------------------------------------------------- check 1
@pytest.mark.parametrize("kind", ["uniform", "peaked", "random"])
def test_range_coder_bit_exact_given_oracle_tables(boa, kind):
    g = np.random.Generator(np.random.PCG64(5))
    S, T = 37, 700                                                 # > one block of 64 coder threads, ragged
    if kind == "uniform":
        logits = np.zeros((S, T, 256), np.float32)
    elif kind == "peaked":                                         # long runs of f=65281 symbols, then rare ones:
        logits = np.full((S, T, 256), -50.0, np.float32)           # exercises pending-0xFF runs and carries
        logits[:, :, 255] = 0.0
    else:
        logits = g.normal(0, 4.0, (S, T, 256)).astype(np.float32)
    C = quantise.quantise(logits)                                  # the ORACLE's tables
    syms = g.integers(0, 256, (S, T)).astype(np.uint8)
    if kind == "peaked":
        syms = np.where(g.random((S, T)) < 0.97, 255, syms).astype(np.uint8)
    want = [rangecoder.encode_stream(C[i], syms[i].astype(np.int64)) for i in range(S)]
    cap = 2 * T + 16
    out, sizes = boa.debug_rc_encode(torch.from_numpy(C.astype(np.int32)).cuda(), torch.from_numpy(syms).cuda(), cap)
    out, sizes = _np(out), _np(sizes)
    for i in range(S):
        assert sizes[i] == len(want[i]) and out[i, : sizes[i]].tobytes() == want[i], (kind, i)
    # and the GPU decoder inverts the ORACLE's encoder
    pay = np.zeros((S, cap), np.uint8)
    for i in range(S):
        pay[i, : len(want[i])] = np.frombuffer(want[i], np.uint8)
    dec = boa.debug_rc_decode(torch.from_numpy(C.astype(np.int32)).cuda(), torch.from_numpy(pay).cuda(),
                              torch.from_numpy(np.array([len(w) for w in want], np.int32)).cuda(), T)
    assert np.array_equal(_np(dec), syms)
    if kind == "uniform":
        assert all(len(w) == T + 4 for w in want)                 # uniform table: exactly n + 4 bytes


def test_range_coder_golden_vectors(boa):
    import os
    path = os.path.join(os.path.dirname(__file__), "golden", "rc_vectors.txt")
    tables = {"uniform": np.arange(257) * 256,
              "peak0": np.concatenate([[0], 65281 + np.arange(256)]),
              "peak255": np.concatenate([np.arange(256), [65536]])}
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        tname, s, pay = [x.strip() for x in line.split(";")]
        if "x" in s:
            b, cnt = s.split("x")
            syms = [int(b, 16)] * int(cnt)
        else:
            syms = [int(x, 16) for x in s.split()]
        C = np.tile(tables[tname].astype(np.int32), (1, len(syms), 1))
        out, sizes = boa.debug_rc_encode(torch.from_numpy(C).cuda(), torch.tensor([syms], dtype=torch.uint8).cuda(),
                                         2 * len(syms) + 16)
        assert _np(out)[0, : int(sizes[0])].tobytes() == bytes(int(x, 16) for x in pay.split()), line


# ---------------------------------------------------------------------------------------- checks 2 and 5
def test_probabilities_and_tables_against_oracle(case, boa):
    name, blob, cfg, gm, w = case
    S, T = 5, 96                                                   # 5 streams: a ragged 128-row tile
    data = np.frombuffer(cfg.data(S * T), np.uint8).reshape(S, T)
    d = gm.debug_step_dump(data.tobytes(), T, T - 1)
    logits64 = model.logits_for_chunks(w, data)
    p_ref = quantise.softmax(logits64)
    p_gpu = _np(d["probs"]).astype(np.float64)
    err = np.abs(p_gpu - p_ref).max()
    print(f"[parity] {name}: max |p_gpu - p_oracle| = {err:.3e} (bar {PROB_TOL:g}), max p = {p_ref.max():.3f}, "
          f"max |logit err| = {np.abs(_np(d['logits']) - logits64).max():.3e}")
    assert err <= PROB_TOL, name
    assert np.abs(_np(d["logits"]) - logits64).max() <= 2e-4 * max(1.0, np.abs(logits64).max())
    # tables: the oracle's rule on the GPU's own fp32 logits must give the GPU's tables, bit for bit
    assert np.array_equal(_np(d["cdf"]).astype(np.int64), quantise.quantise(_np(d["logits"])))
    if "sharp" in name:
        assert p_ref.max() > 0.05                                   # the sharp sets are actually sharp


# ---------------------------------------------------------------------------------------- checks 3 and 4
def test_round_trip_and_size_against_oracle(case, boa):
    name, blob, cfg, gm, w = case
    chunk = 160
    data = cfg.data(7 * chunk + 33)                                # ragged last chunk
    comp = gm.compress(data, chunk)
    assert _np(gm.decompress(comp)).tobytes() == data
    ref = codec.compress(w, data, chunk)
    assert abs(len(comp) - len(ref)) <= SIZE_TOL * len(ref), (name, len(comp), len(ref))
    # container structure: parse with the oracle's reader, GPU fingerprint
    n, cb, last, first, payloads = container.unpack(_np(comp).tobytes(), gm.fingerprint)
    assert (n, cb, last) == (len(data), chunk, 33) and first == bytes(data[i * chunk] for i in range(8))
    # eq. 1: each GPU payload is within (0,5) bytes of the ideal code length under the GPU's own tables
    full = np.frombuffer(data[: 7 * chunk], np.uint8).reshape(7, chunk)
    C = _np(gm.debug_step_dump(full.tobytes(), chunk, chunk - 1, want=("cdf",))["cdf"]).astype(np.int64)
    for i in range(7):
        assert 0 < len(payloads[i]) - codec.ideal_bytes(C[i], full[i, 1:]) < 5


def test_host_pointers_and_device_pointers_agree(case, boa):
    name, blob, cfg, gm, w = case
    data = cfg.data(3000)
    a = gm.compress(data, 500, device="cuda")
    b = gm.compress(data, 500, device="cpu")                       # host buffers, staged by the library
    assert b.device.type == "cpu" and _np(a).tobytes() == _np(b).tobytes()
    assert _np(gm.decompress(b, device="cpu")).tobytes() == data


# ------------------------------------------------- SURVEY 8(d) parity subset: checks 2, 3, 5 on the configs' real inputs
def _parity_subset(cfg, length=2048, n_ids=8):
    """8 chunk ids (first, last, 6 seeded) x the first 2048 bytes of each, from the config's full input."""
    data = np.frombuffer(cfg.data(), np.uint8)
    nc = len(data) // cfg.chunk_bytes
    g = np.random.Generator(np.random.PCG64(cfg.data_seed))
    ids = [0, nc - 1] + sorted(int(x) for x in g.choice(np.arange(1, nc - 1), n_ids - 2, replace=False))
    return ids, np.stack([data[i * cfg.chunk_bytes: i * cfg.chunk_bytes + length] for i in ids])


@pytest.mark.parametrize("name", ["cfg2", "cfg2_sharp", "cfg3_sharp", "cfg4_sharp", "cfg5_sharp", "paper_block_sharp"])
def test_parity_subset_of_the_configured_inputs(boa, name):
    """SURVEY 8(d) "Oracle timing": 8 chunks x the first 2,048 bytes of BASELINE.json configs[1..4]'s own inputs
    (chunk_bytes = 2048) through the configs' own model shapes: probabilities within 1e-5 over all 2,047 steps (the
    state is far from its zero start by then), tables bit-exact on the GPU's logits, container size within 0.5 % of
    the oracle's (16 KB: 80-byte resolution), eq. 1 per stream, byte-exact round trip."""
    cfgno = {"cfg2": 2, "cfg2_sharp": 2, "cfg3_sharp": 3, "cfg4_sharp": 4, "cfg5_sharp": 5, "paper_block_sharp": 6}[name]
    cfg = synth.CONFIGS[cfgno]
    kw = {} if name == "cfg2" else ({"emb_std": 0.25, "ffn_std": 0.1} if cfgno == 6 else {"emb_std": 0.25})
    blob = cfg.weights(**kw)
    gm, w = boa.Model(blob), model.load_weights(blob)
    T = 2048
    ids, chunks = _parity_subset(cfg, T)
    raw = chunks.tobytes()
    d = gm.debug_step_dump(raw, T, T - 1)
    logits64 = model.logits_for_chunks(w, chunks)                  # the oracle's model, once
    p_ref = quantise.softmax(logits64)
    err = np.abs(_np(d["probs"]).astype(np.float64) - p_ref).max()
    C_gpu = _np(d["cdf"]).astype(np.int64)
    assert np.array_equal(C_gpu.reshape(-1, 257), quantise.quantise(_np(d["logits"]).reshape(-1, 256)))      # check 5
    comp = gm.compress(raw, T)
    assert _np(gm.decompress(comp)).tobytes() == raw                                                       # check 4
    # the oracle's container size from its own tables and coder (codec.compress restated on the logits above)
    C_ref = quantise.quantise(logits64.astype(np.float32))
    ref_size = container.index_bytes(len(ids)) + sum(len(rangecoder.encode_stream(C_ref[i], chunks[i, 1:].astype(np.int64)))
                                                     for i in range(len(ids)))
    _, _, _, _, payloads = container.unpack(_np(comp).tobytes(), gm.fingerprint)
    gaps = [len(payloads[i]) - codec.ideal_bytes(C_gpu[i], chunks[i, 1:]) for i in range(len(ids))]
    print(f"[parity] {name} subset chunks {ids}: max |p_gpu - p_oracle| = {err:.3e}, max p = {p_ref.max():.3f}, "
          f"size {comp.numel()} B vs oracle {ref_size} B ({abs(comp.numel() - ref_size) / ref_size:.2e}), "
          f"bits/byte {8 * comp.numel() / len(raw):.3f}, eq. 1 gaps {min(gaps):.2f}..{max(gaps):.2f} B")
    assert err <= PROB_TOL                                                                                  # check 2
    assert abs(comp.numel() - ref_size) <= SIZE_TOL * ref_size                                              # check 3
    assert all(0 < g < 5 for g in gaps)
    # check 1 on the product path itself (time-slab coder, 16-byte staged stores, device-side compaction): every payload is,
    # byte for byte, what the ORACLE's range coder writes for the GPU's own tables
    for i in range(len(ids)):
        assert payloads[i] == rangecoder.encode_stream(C_gpu[i], chunks[i, 1:].astype(np.int64)), (name, ids[i])


# ---------------------------------------------------------------------------------------------- edges
def test_edge_cases(boa):
    cfg = synth.CONFIGS[1]
    gm = boa.Model(cfg.weights())
    empty = gm.compress(b"", 4096)
    assert empty.numel() == 44 and gm.decompress(empty).numel() == 0
    for n, chunk in [(1, 4096), (5, 1), (4096, 4096), (4097, 4096), (1000, 7), (300, 2)]:
        data = cfg.data(n)
        comp = gm.compress(data, chunk)
        assert comp.numel() <= boa.compress_bound(n, chunk)
        assert _np(gm.decompress(comp)).tobytes() == data, (n, chunk)
    # 1-byte chunks code zero symbols: payload = 4 flush bytes each
    comp = _np(gm.compress(cfg.data(5), 1)).tobytes()
    assert len(comp) == container.index_bytes(5) + 5 * 4


def test_fingerprint_is_stable_and_follows_weights_and_arithmetic(boa):
    """The fingerprint = (generation ^ CRC of the probe logits) << 32 | CRC(blob): the same for two handles of one blob,
    different in BOTH halves for another blob (other weights give other probe logits), and what containers carry."""
    cfg = synth.CONFIGS[1]
    a1, a2, b = boa.Model(cfg.weights()), boa.Model(cfg.weights()), boa.Model(cfg.weights(emb_std=0.25))
    assert a1.fingerprint == a2.fingerprint
    assert (a1.fingerprint >> 32) != (b.fingerprint >> 32) and (a1.fingerprint & 0xFFFFFFFF) != (b.fingerprint & 0xFFFFFFFF)
    import zlib
    assert (a1.fingerprint & 0xFFFFFFFF) == (zlib.crc32(cfg.weights()) & 0xFFFFFFFF)
    comp = _np(a1.compress(cfg.data(300), 100)).tobytes()
    assert int.from_bytes(comp[32:40], "little") == a1.fingerprint
    assert _np(a2.decompress(torch.frombuffer(bytearray(comp), dtype=torch.uint8).cuda())).tobytes() == cfg.data(300)


def test_errors(boa):
    cfg = synth.CONFIGS[1]
    gm = boa.Model(cfg.weights())
    other = boa.Model(cfg.weights(emb_std=0.25))
    data = cfg.data(2000)
    comp = gm.compress(data, 250)
    dst = torch.empty(2000, dtype=torch.uint8, device="cuda")

    def code(fn):
        with pytest.raises(boa.BoaError) as e:
            fn()
        return e.value.code

    assert code(lambda: other.decompress(comp)) == boa.E_MODEL_MISMATCH
    bad = comp.clone(); bad[45] ^= 1                               # index byte -> CRC
    assert code(lambda: gm.decompress_into(bad, dst)) == boa.E_CRC
    bad = comp.clone(); bad[0] = 0
    assert code(lambda: gm.decompress_into(bad, dst)) == boa.E_FORMAT
    assert code(lambda: gm.decompress_into(comp[:-3], dst)) == boa.E_FORMAT
    assert code(lambda: gm.decompress_into(comp, dst[:100])) == boa.E_CAPACITY
    small = torch.empty(60, dtype=torch.uint8, device="cuda")
    assert code(lambda: gm.compress_into(torch.zeros(2000, dtype=torch.uint8, device="cuda"), 250, small)) == boa.E_CAPACITY
    # BOAW header: the FFN flag and the hidden width must agree; unknown flag bits are refused
    import struct
    blob = bytearray(synth.make_weights(synth.ModelShape(1, 64, dt_rank=4, d_ff=64), 1))
    for flags, d_ff in [(1, 64), (3, 0), (7, 64)]:
        bad_blob = bytearray(blob); struct.pack_into("<2I", bad_blob, 36, flags, d_ff)
        assert code(lambda: boa.Model(bytes(bad_blob))) == boa.E_FORMAT
    # payload corruption: either detected (BOA_E_CORRUPT) or decodes to different bytes, never a crash
    bad = comp.clone(); bad[-40:] = 0xFF
    try:
        out = gm.decompress(bad)
        assert _np(out).tobytes() != data
    except boa.BoaError as e:
        assert e.code == boa.E_CORRUPT


@pytest.mark.parametrize("shape", ["cfg1", "cfg4", "cfg5_l2"])
def test_result_independent_of_batch_and_position(boa, shape):
    """P:116 lock-step determinism, strengthened: a chunk's payload does not depend on which other chunks are
    stepped with it, so any B reproduces the same tables - and so does any split of the chunks into waves (the wave
    size comes from the free device memory at run time, so encoder and decoder may step different B)."""
    cfg = synth.CONFIGS[1]
    blob = {"cfg1": lambda: cfg.weights(emb_std=0.25),
            "cfg4": lambda: synth.make_weights(synth.CONFIGS[4].shape, 2, synth.DTYPE_BF16, emb_std=0.25),
            "cfg5_l2": lambda: synth.make_weights(synth.ModelShape(2, 512, dt_rank=32), 3, synth.DTYPE_BF16, emb_std=0.25)}[shape]()
    gm = boa.Model(blob)
    chunk = 200 if shape == "cfg1" else 60
    data = cfg.data(140 * chunk)                                   # 140 streams: two 128-row tensor-core tiles
    whole = _np(gm.compress(data, chunk)).tobytes()
    _, _, _, _, pa = container.unpack(whole)
    for i in (0, 9, 127, 128, 139):
        solo = gm.compress(data[i * chunk:(i + 1) * chunk], chunk)
        _, _, _, _, ps = container.unpack(_np(solo).tobytes())
        assert ps[0] == pa[i], i
    # forced wave splits: 140 chunks in waves of 33 (ragged last wave) and of 128; same container, and a decoder that
    # steps other waves than the encoder did still inverts it
    for wave in (33, 128):
        gm.debug_set_max_wave(wave)
        try:
            assert _np(gm.compress(data, chunk)).tobytes() == whole, wave
            assert _np(gm.decompress(torch.frombuffer(bytearray(whole), dtype=torch.uint8).cuda())).tobytes() == data
        finally:
            gm.debug_set_max_wave(0)


def test_more_chunks_than_one_wave(boa):
    """More than 65,536 chunks run in waves of streams; 2-byte chunks code one symbol each."""
    cfg = synth.CONFIGS[1]
    gm = boa.Model(cfg.weights(emb_std=0.25))
    data = cfg.data(2 * 70001 + 1)
    comp = gm.compress(data, 2)
    assert _np(gm.decompress(comp)).tobytes() == data


@pytest.mark.parametrize("config", [2, 6])
def test_full_size_in_the_bench_configuration(boa, config):
    """BASELINE.json configs[1] at full size, exactly as bench.py runs it (64 MiB, 4096 chunks x 16 KiB, B = 4096 streams
    per step): byte-exact round trip of the whole input, and - on sampled streams the oracle can compute one by one -
    probabilities within 1e-5 and tables bit-exact for the first steps of the same full-width launch.  Config 6 is the
    paper's own block on the same input, as `bench.py --config 6` runs it."""
    cfg = synth.CONFIGS[config]
    blob = cfg.weights()
    gm = boa.Model(blob)
    w = model.load_weights(blob)
    data = cfg.data()
    src = torch.frombuffer(bytearray(data), dtype=torch.uint8).cuda()
    comp = gm.compress(src, cfg.chunk_bytes)
    back = gm.decompress(comp)
    assert torch.equal(back, src)
    B, T = len(data) // cfg.chunk_bytes, 25
    d = gm.debug_step_dump(src, cfg.chunk_bytes, T - 1, want=("logits", "probs", "cdf"))
    buf = np.frombuffer(data, np.uint8).reshape(B, cfg.chunk_bytes)
    ids = [0, 127, 128, 1777, B - 1]                                # tile edges, middle, last stream
    ref = quantise.softmax(model.logits_for_chunks(w, buf[ids, :T]))
    got = _np(d["probs"][ids]).astype(np.float64)
    err = np.abs(got - ref).max()
    print(f"[parity] {cfg.name} full size, streams {ids}: max |p_gpu - p_oracle| = {err:.3e}")
    assert err <= PROB_TOL
    lg = _np(d["logits"][ids])
    assert np.array_equal(_np(d["cdf"][ids]).astype(np.int64).reshape(-1, 257), quantise.quantise(lg.reshape(-1, 256)))
    # eq. 1 on sampled streams, WHOLE chunks (16,383 coded symbols each): the payload the full-size run wrote
    # for stream i is within (0, 5) bytes of the ideal code length sum_t -log256(f_t(s_t)/2^16) under the GPU's own
    # tables.  The tables of every step of those streams come from a second, small dump run on the same bytes (the
    # result for a stream does not depend on which streams are stepped with it, P:116 - checked here as well: the small
    # run writes the very payloads of the full-size run).
    _, _, _, _, payloads = container.unpack(_np(comp).tobytes(), gm.fingerprint)
    assert len(payloads) == B and all(len(p) >= 4 for p in payloads)
    sel = [0, 128, B - 1]
    sub = np.ascontiguousarray(buf[sel])
    _, _, _, _, pay_sub = container.unpack(_np(gm.compress(sub.tobytes(), cfg.chunk_bytes)).tobytes(), gm.fingerprint)
    C = _np(gm.debug_step_dump(sub.tobytes(), cfg.chunk_bytes, cfg.chunk_bytes - 1, want=("cdf",))["cdf"]).astype(np.int64)
    for j, i in enumerate(sel):
        assert pay_sub[j] == payloads[i], i
        gap = len(payloads[i]) - codec.ideal_bytes(C[j], sub[j, 1:])
        print(f"[parity] {cfg.name} stream {i}: payload {len(payloads[i])} B, ideal + {gap:.3f} B")
        assert 0 < gap < 5, (i, gap)
    # the time-slab encoder and the step encoder write the same container at full size (the decoder always steps)
    gm.debug_set_slab(False)
    try:
        assert torch.equal(gm.compress(src, cfg.chunk_bytes), comp)
    finally:
        gm.debug_set_slab(True)


def test_maximum_wave_65536_streams_cfg4_model(boa):
    """The largest wave the library steps together (65,536 streams, SURVEY 8(d) cfg4 sweep end point) on the cfg4 model
    (4 layers, D = 256, bf16 matrices): 512 row tiles per contraction, 10 GB of stream state.  Byte-exact round trip of
    every stream, and sampled streams against the oracle (probabilities 1e-5, tables bit-exact)."""
    cfg = synth.CONFIGS[4]
    blob = synth.make_weights(cfg.shape, cfg.model_seed, synth.DTYPE_BF16, emb_std=0.25)
    gm = boa.Model(blob)
    w = model.load_weights(blob)
    B, T = 65536, 24
    data = synth.CONFIGS[2].data(B * T)
    src = torch.frombuffer(bytearray(data), dtype=torch.uint8).cuda()
    comp = gm.compress(src, T)
    assert torch.equal(gm.decompress(comp), src)
    d = gm.debug_step_dump(src, T, T - 1, want=("logits", "probs", "cdf"))
    buf = np.frombuffer(data, np.uint8).reshape(B, T)
    ids = [0, 1, 32767, 32768, 65535]
    ref = quantise.softmax(model.logits_for_chunks(w, buf[ids]))
    err = np.abs(_np(d["probs"][ids]).astype(np.float64) - ref).max()
    print(f"[parity] cfg4 model, 65536 streams, streams {ids}: max |p_gpu - p_oracle| = {err:.3e}")
    assert err <= PROB_TOL
    lg = _np(d["logits"][ids])
    assert np.array_equal(_np(d["cdf"][ids]).astype(np.int64).reshape(-1, 257), quantise.quantise(lg.reshape(-1, 256)))


def test_time_slab_encoder_writes_the_bytes_of_the_step_path(boa):
    """Encode-side time slabs (compression advances 16 steps per pass over the stream state) must be
    bit-identical to stepping one byte at a time - the decoder always steps - for ragged lengths around the slab size."""
    cfg = synth.CONFIGS[1]
    for blob in (cfg.weights(emb_std=0.25), synth.make_weights(synth.CONFIGS[2].shape, 1, emb_std=0.25),
                 synth.make_weights(synth.CONFIGS[6].shape, 4, emb_std=0.25, ffn_std=0.1)):
        gm = boa.Model(blob)
        for n, chunk in [(150 * 41 + 13, 41), (300 * 9, 9), (5 * 200 + 10, 200), (130 * 17, 17)]:
            data = cfg.data(n)
            a = _np(gm.compress(data, chunk)).tobytes()
            gm.debug_set_slab(False)
            try:
                b = _np(gm.compress(data, chunk)).tobytes()
            finally:
                gm.debug_set_slab(True)
            assert a == b, (n, chunk)
            assert _np(gm.decompress(torch.frombuffer(bytearray(a), dtype=torch.uint8).cuda())).tobytes() == data


@pytest.mark.parametrize("world", [2, 3, 5])
def test_one_container_from_several_gpus_run_one_after_the_other(boa, world):
    """contiguous chunk ranges per GPU, parts -> ONE container.  The ranks are run one after
    the other on this GPU (chunks are independent, so that is what N GPUs compute): boa_compress_shard of every
    range + boa_container_assemble must be byte-identical to boa_compress of the whole input, and boa_decompress_shard
    of every range of that container must give back the range's bytes."""
    from paper_2511_11337_b200 import shard
    cfg = synth.CONFIGS[1]
    gm = boa.Model(cfg.weights(emb_std=0.25))
    chunk = 150
    data = cfg.data(11 * chunk + 77)                               # 12 chunks, ragged tail
    n = len(data)
    src = torch.frombuffer(bytearray(data), dtype=torch.uint8).cuda()
    whole = gm.compress(src, chunk)
    parts, pays = [], []
    for r in range(world):
        lo, hi = shard.byte_range(n, chunk, r, world)
        buf = torch.empty(2 * (hi - lo) + 4 * 12, dtype=torch.uint8, device="cuda" if r % 2 == 0 else "cpu")
        plen, sizes, first = gm.compress_shard(src[lo:hi] if r % 2 == 0 else src[lo:hi].cpu(), chunk, buf)
        assert plen == int(sizes.sum()) and sizes.numel() == -(-(hi - lo) // chunk)
        parts.append((sizes, first)); pays.append(buf[:plen])
    for dev in ("cuda", "cpu"):
        out = torch.zeros(boa.compress_bound(n, chunk), dtype=torch.uint8, device=dev)
        ln, offs = gm.container_assemble(n, chunk, parts, out, pays)
        assert ln == whole.numel() and torch.equal(out[:ln].cpu(), whole.cpu()), dev
        assert offs[0] == boa.container_index_bytes(n, chunk) and offs[-1] == ln
    # index only + blocks placed by the caller (what the NCCL exchange does: blocks are received in place)
    out = torch.zeros(boa.compress_bound(n, chunk), dtype=torch.uint8, device="cuda")
    _, offs = gm.container_assemble(n, chunk, parts, out, None)
    for r in range(world):
        out[offs[r]: offs[r + 1]] = pays[r].cuda()
    ln2, _ = gm.container_assemble(n, chunk, parts, out, [out[offs[r]: offs[r + 1]] for r in range(world)])
    assert torch.equal(out[:ln2], whole)
    # decode: every rank its own chunk range of the shared container
    back = torch.zeros(n, dtype=torch.uint8, device="cuda")
    for r in range(world):
        c_lo, c_hi = shard.chunk_range(12, r, world)
        lo, hi = shard.byte_range(n, chunk, r, world)
        got = gm.decompress_shard(whole if r % 2 == 0 else whole.cpu(), c_lo, c_hi - c_lo, back[lo:hi])
        assert got == hi - lo
    assert torch.equal(back, src)
    with pytest.raises(boa.BoaError) as e:
        gm.decompress_shard(whole, 11, 2, back)
    assert e.value.code == boa.E_ARG
    assert gm.decompress_shard(whole, 12, 0, back) == 0


def test_streaming_front_end(boa):
    """Fig. 2: groups of chunks -> concatenated shards through the two-lane
    pre-load / compress / collect pipeline.  Every shard must be the bytes boa_compress writes for its group alone, the
    stream must round-trip, parse with the oracle's reader, and match the oracle's stream size within 0.5 %."""
    cfg = synth.CONFIGS[1]
    blob = cfg.weights(emb_std=0.25)
    gm, w = boa.Model(blob), model.load_weights(blob)
    chunk, group = 100, 3
    data = cfg.data(10 * chunk + 37)                               # 11 chunks: groups of 3, 3, 3, 2 (ragged tail)
    stream, lens = gm.stream_compress(data, chunk, group)
    assert stream.device.type == "cpu" and len(lens) == 4 and sum(lens) == stream.numel()
    assert stream.numel() <= boa.stream_bound(len(data), chunk, group)
    raw = _np(stream).tobytes()
    shards = container.split_shards(raw)
    assert [len(s) for s in shards] == lens
    for k, s in enumerate(shards):
        part = data[k * chunk * group:(k + 1) * chunk * group]
        assert s == _np(gm.compress(part, chunk)).tobytes(), k
        assert container.unpack(s, gm.fingerprint)[0] == len(part)
    assert _np(gm.stream_decompress(stream)).tobytes() == data
    ref = b"".join(codec.stream_compress(w, data, chunk, group))
    assert abs(len(raw) - len(ref)) <= SIZE_TOL * len(ref)
    # many groups (both lanes reused several times), one group, empty input
    data = cfg.data(64 * 40)
    for group in (1, 5, 64, 1000):
        s2, l2 = gm.stream_compress(data, 40, group)
        assert len(l2) == -(-64 // group) and _np(gm.stream_decompress(s2)).tobytes() == data
    s0, l0 = gm.stream_compress(b"", 40, 4)
    assert s0.numel() == 0 and l0 == [] and gm.stream_decompress(s0).numel() == 0
    # errors: a cut stream, a stream from another model
    with pytest.raises(boa.BoaError) as e:
        gm.stream_decompress(stream[:-5])
    assert e.value.code == boa.E_FORMAT
    with pytest.raises(boa.BoaError) as e:
        boa.Model(cfg.weights()).stream_decompress(stream)
    assert e.value.code == boa.E_MODEL_MISMATCH

