// boa_fx.cuh — host side of FX1, the deterministic fixed-point pipeline (include/boa.h "boa_fx_*").
// Included at the end of boa_api.cu (one translation unit: it reuses GrowBuf, BlobReader, the coder / container helpers).
// Product path: nothing here touches oracle/; without a usable device every computing entry point returns BOA_E_CUDA.
#pragma once
#include "fx_coder.cuh"
#include "fx_gemm_tc.cuh"
#include "fx_kernels.cuh"

struct FxLayerDev {
  const int32_t *norm_w, *conv_w, *conv_b, *b_dt, *a_neg, *d_skip;     // Q
  const uint8_t *q_in, *q_x, *q_out;                                   // int8 rows as tensor-core operand images
  const int8_t* q_dt;                                                  // int8 rows [E][R] (read by the scan)
  const int32_t *s_in, *s_x, *s_dt, *s_out;                            // row exponents
};

struct boa_fx_model {
  int L = 0, D = 0, E = 0, R = 0, J = 0, ldj = 0;
  uint32_t blob_crc = 0;
  int64_t sqrt_d = 0;
  GrowBuf w32, w8;                      // device copies of all int32 / int8 weight data
  const int8_t* q_emb = nullptr;        // [256][D] rows (embedding look-up)
  const uint8_t* q_head = nullptr;      // the same rows as an operand image (tied head)
  const int32_t* s_emb = nullptr;
  fx::Tables tab{};
  std::vector<FxLayerDev> layers;
  // workspace of a wave
  uint64_t Bcap = 0;
  GrowBuf u, xz, xs, dbc, logits, qa, ka, h, win;
  GrowBuf pos, len, low, range, pending, wpos, cache, started, v, rpos, off, size, scratch, first, err, total;
  GrowBuf stage_in, stage_out;
  PinBuf pin;
  cudaStream_t own = nullptr;
  cudaEvent_t user_ev = nullptr;
  uint64_t launches = 0;
  ~boa_fx_model() {
    for (GrowBuf* b : {&w32, &w8, &u, &xz, &xs, &dbc, &logits, &qa, &ka, &h, &win, &pos, &len, &low, &range, &pending,
                       &wpos, &cache, &started, &v, &rpos, &off, &size, &scratch, &first, &err, &total, &stage_in, &stage_out})
      b->release();
    pin.release();
    if (user_ev) cudaEventDestroy(user_ev);
    if (own) cudaStreamDestroy(own);
  }
};

namespace {

constexpr uint32_t kFxArith = 0x46583031u;     // 'FX01'

// w rows [N][K] (fp32 / bf16 values, widened exactly) -> int8 rows q [N][ldq] and exponents s [N]:
// s = the largest exponent with max|w_row| 2^s <= 127, within [-8, 40] (0 for a zero row); q = round-half-even(w 2^s).
void fx_quantise_rows(const std::vector<float>& w, size_t N, size_t K, size_t ldq, std::vector<int8_t>& q, std::vector<int32_t>& s) {
  const size_t q0 = q.size(), s0 = s.size();
  q.resize(q0 + N * ldq, 0);
  s.resize(s0 + N, 0);
  for (size_t n = 0; n < N; ++n) {
    double m = 0.0;
    for (size_t k = 0; k < K; ++k) m = std::max(m, fabs((double)w[n * K + k]));
    int e = 0;
    if (m > 0.0) {
      e = (int)floor(log2(127.0 / m));
      e = std::min(40, std::max(-8, e));
      for (int it = 0; it < 2; ++it) {             // floor(log2) may be off by one at powers of two: exact comparisons settle it
        if (ldexp(m, e) > 127.0) --e;
        if (ldexp(m, e + 1) <= 127.0 && e < 40) ++e;
      }
    }
    s[s0 + n] = e;
    for (size_t k = 0; k < K; ++k) {
      double v = nearbyint(ldexp((double)w[n * K + k], e));   // exact product, ties to even (default rounding mode)
      v = std::min(127.0, std::max(-127.0, v));
      q[q0 + n * ldq + k] = (int8_t)v;
    }
  }
}
// fp -> Q, round half even, saturating
void fx_to_q(const std::vector<double>& x, std::vector<int32_t>& out) {
  for (double v : x) {
    double t = nearbyint(ldexp(v, fx::F));
    t = std::min(2147483647.0, std::max(-2147483648.0, t));
    out.push_back((int32_t)t);
  }
}
size_t fx_kb(size_t k) { return (k + fx::TBK - 1) / fx::TBK; }
// int8 rows q [N][K] -> operand image [ceil(N/64)][KB][64 x 128 bytes, swizzled], zero beyond N and K; appended 1024-aligned
size_t fx_weight_image(const int8_t* q, size_t N, size_t K, std::vector<int8_t>& w8) {
  while (w8.size() % 1024) w8.push_back(0);
  const size_t o = w8.size(), KB = fx_kb(K), NT = (N + fx::TBN - 1) / fx::TBN;
  w8.resize(o + NT * KB * fx::W_BLK, 0);
  for (size_t n = 0; n < N; ++n)
    for (size_t k = 0; k < K; ++k) w8[o + fx::w_img_off((int)n, (int)k, (int)KB)] = q[n * K + k];
  return o;
}

}  // namespace

extern "C" {

uint64_t boa_fx_model_fingerprint(const boa_fx_model* m) { return m ? (((uint64_t)kFxArith << 32) | m->blob_crc) : 0; }
void boa_fx_model_free(boa_fx_model* m) { delete m; }

int boa_fx_model_load(const void* weights, size_t nbytes, boa_fx_model** out) {
  if (!weights || !out || nbytes < 64) return BOA_E_ARG;
  *out = nullptr;
  const uint8_t* p = static_cast<const uint8_t*>(weights);
  if (memcmp(p, "BOAW", 4) != 0 || get_u32(p + 4) != 1) return BOA_E_FORMAT;
  const uint32_t dtype = get_u32(p + 8), L = get_u32(p + 12), D = get_u32(p + 16), N = get_u32(p + 20), K = get_u32(p + 24),
                 ex = get_u32(p + 28), R = get_u32(p + 32), flags = get_u32(p + 36), Fw = get_u32(p + 40);
  if (dtype > 1 || (flags & ~3u)) return BOA_E_FORMAT;
  // FX1 covers north_star's block with the tied head
  if (flags != 1u || Fw != 0 || N != (uint32_t)kNState || K != (uint32_t)kDConv || ex != 2 || L == 0 || L > 64 || D == 0 ||
      D % 64 != 0 || D > 1024 || R == 0 || R > 64)
    return BOA_E_UNSUPPORTED;
  BOA_TRY(check_device());
  const size_t E = 2 * (size_t)D, J = R + 2 * kNState;
  boa_fx_model* m = new (std::nothrow) boa_fx_model();
  if (!m) return BOA_E_NOMEM;
  m->L = (int)L; m->D = (int)D; m->E = (int)E; m->R = (int)R; m->J = (int)J; m->ldj = (int)((J + 3) / 4 * 4);
  m->blob_crc = crc32_ieee(p, nbytes);
  m->sqrt_d = (int64_t)floorl(sqrtl((long double)((uint64_t)D << 40)));
  while ((unsigned __int128)m->sqrt_d * m->sqrt_d > ((unsigned __int128)D << 40)) --m->sqrt_d;        // exact floor square root
  while ((unsigned __int128)(m->sqrt_d + 1) * (m->sqrt_d + 1) <= ((unsigned __int128)D << 40)) ++m->sqrt_d;

  // the two tables, computed here in extended precision and checked against the CRC the specification states
  std::vector<int32_t> w32;
  std::vector<int8_t> w8;
  {
    std::vector<int64_t> tabs;
    for (int i = 0; i <= fx::NTAB; ++i) tabs.push_back((int64_t)rintl(1073741824.0L * exp2l(-(long double)i / fx::NTAB)));
    for (int i = 0; i <= fx::NTAB; ++i) tabs.push_back((int64_t)rintl(1073741824.0L * log1pl((long double)i / fx::NTAB)));
    std::vector<uint8_t> bytes(tabs.size() * 8);
    for (size_t i = 0; i < tabs.size(); ++i) put_u64(bytes.data() + 8 * i, (uint64_t)tabs[i]);
    if (crc32_ieee(bytes.data(), bytes.size()) != fx::TABLE_CRC) { delete m; return BOA_E_UNSUPPORTED; }
    for (int64_t v : tabs) w32.push_back((int32_t)v);
  }
  const size_t off_exp2 = 0, off_log1p = fx::NTAB + 1;

  struct Off { size_t norm_w, conv_w, conv_b, b_dt, a_neg, d_skip, s_in, s_x, s_dt, s_out, q_in, q_x, q_dt, q_out; };
  std::vector<Off> offs(L);
  BlobReader br{p, nbytes, 64, (int)dtype};
  std::vector<float> t;
  std::vector<int32_t> sv;
  auto vec_q = [&](const std::vector<float>& f) {
    std::vector<double> d(f.begin(), f.end());
    while (w32.size() % 4) w32.push_back(0);       // 16-byte alignment: the kernels read taps and |A| rows as int4
    const size_t o = w32.size();
    fx_to_q(d, w32);
    return o;
  };
  std::vector<int8_t> rows;
  auto mat_q = [&](size_t Nr, size_t Kc, size_t& q_off, size_t& s_off) {   // int8 rows -> operand image + exponents
    rows.clear();
    sv.clear();
    fx_quantise_rows(t, Nr, Kc, Kc, rows, sv);
    q_off = fx_weight_image(rows.data(), Nr, Kc, w8);
    s_off = w32.size();
    w32.insert(w32.end(), sv.begin(), sv.end());
  };
  size_t q_emb = 0, q_head = 0, s_emb = 0;
  bool ok = br.take(256 * (size_t)D, true, t);
  if (ok) {
    mat_q(256, D, q_head, s_emb);
    while (w8.size() % 16) w8.push_back(0);
    q_emb = w8.size();
    w8.insert(w8.end(), rows.begin(), rows.end());
  }
  for (uint32_t l = 0; l < L && ok; ++l) {
    Off& o = offs[l];
    ok = ok && br.take(D, false, t); if (ok) o.norm_w = vec_q(t);
    ok = ok && br.take(2 * E * D, true, t); if (ok) mat_q(2 * E, D, o.q_in, o.s_in);
    ok = ok && br.take(E * 4, false, t); if (ok) o.conv_w = vec_q(t);
    ok = ok && br.take(E, false, t); if (ok) o.conv_b = vec_q(t);
    ok = ok && br.take(J * E, true, t); if (ok) mat_q(J, E, o.q_x, o.s_x);
    ok = ok && br.take(E * R, true, t);
    if (ok) {                                       // W_dt [E][R]: rows of R bytes, unpadded (read by the scan kernel)
      while (w8.size() % 16) w8.push_back(0);
      o.q_dt = w8.size();
      sv.clear();
      fx_quantise_rows(t, E, R, R, w8, sv);
      o.s_dt = w32.size();
      w32.insert(w32.end(), sv.begin(), sv.end());
    }
    ok = ok && br.take(E, false, t); if (ok) o.b_dt = vec_q(t);
    ok = ok && br.take(E * kNState, false, t);
    if (ok) {                                       // |A| = exp(A_log) in Q
      std::vector<double> d(t.size());
      for (size_t i = 0; i < t.size(); ++i) d[i] = exp((double)t[i]);
      while (w32.size() % 4) w32.push_back(0);
      o.a_neg = w32.size();
      fx_to_q(d, w32);
    }
    ok = ok && br.take(E, false, t); if (ok) o.d_skip = vec_q(t);
    ok = ok && br.take(D * E, true, t); if (ok) mat_q(D, E, o.q_out, o.s_out);
  }
  if (!ok || br.off != nbytes) { delete m; return BOA_E_FORMAT; }

  int rc = m->w32.reserve(w32.size() * 4);
  if (rc == BOA_OK) rc = m->w8.reserve(w8.size());
  if (rc == BOA_OK && (cudaStreamCreateWithFlags(&m->own, cudaStreamNonBlocking) != cudaSuccess ||
                       cudaEventCreateWithFlags(&m->user_ev, cudaEventDisableTiming) != cudaSuccess)) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc == BOA_OK && (cudaMemcpy(m->w32.p, w32.data(), w32.size() * 4, cudaMemcpyHostToDevice) != cudaSuccess ||
                       cudaMemcpy(m->w8.p, w8.data(), w8.size(), cudaMemcpyHostToDevice) != cudaSuccess)) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc == BOA_OK && cudaFuncSetAttribute(fx::k_fx_gemm_tc, cudaFuncAttributeMaxDynamicSharedMemorySize,
                                           fx::TC_MAXST * (fx::A_BLK + fx::W_BLK) + 1024) != cudaSuccess) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc != BOA_OK) { delete m; return rc; }
  const int32_t* b32 = m->w32.as<int32_t>();
  const int8_t* b8 = m->w8.as<int8_t>();
  const uint8_t* bi = m->w8.as<uint8_t>();
  m->tab.exp2 = b32 + off_exp2; m->tab.log1p = b32 + off_log1p;
  m->q_emb = b8 + q_emb; m->q_head = bi + q_head; m->s_emb = b32 + s_emb;
  m->layers.resize(L);
  for (uint32_t l = 0; l < L; ++l) {
    const Off& o = offs[l];
    FxLayerDev& w = m->layers[l];
    w.norm_w = b32 + o.norm_w; w.conv_w = b32 + o.conv_w; w.conv_b = b32 + o.conv_b; w.b_dt = b32 + o.b_dt;
    w.a_neg = b32 + o.a_neg; w.d_skip = b32 + o.d_skip;
    w.q_in = bi + o.q_in; w.q_x = bi + o.q_x; w.q_dt = b8 + o.q_dt; w.q_out = bi + o.q_out;
    w.s_in = b32 + o.s_in; w.s_x = b32 + o.s_x; w.s_dt = b32 + o.s_dt; w.s_out = b32 + o.s_out;
  }
  *out = m;
  return BOA_OK;
}

}  // extern "C"

namespace {

int fx_reserve(boa_fx_model* m, uint64_t B, size_t cap) {
  const size_t D = m->D, E = m->E, L = m->L;
  if (B > m->Bcap) {
    BOA_TRY(m->u.reserve(B * D * 4)); BOA_TRY(m->xz.reserve(B * 2 * E * 4));
    BOA_TRY(m->xs.reserve(B * E * 4)); BOA_TRY(m->dbc.reserve(B * m->ldj * 4));
    BOA_TRY(m->logits.reserve(B * 256 * 4)); BOA_TRY(m->qa.reserve(fx::a_img_bytes(B, fx_kb(E)))); BOA_TRY(m->ka.reserve(B * 4));
    BOA_TRY(m->h.reserve(L * B * E * kNState * 4)); BOA_TRY(m->win.reserve(L * B * 3 * E * 4));
    BOA_TRY(m->pos.reserve(B * 4)); BOA_TRY(m->len.reserve(B * 4)); BOA_TRY(m->low.reserve(B * 8)); BOA_TRY(m->range.reserve(B * 4));
    BOA_TRY(m->pending.reserve(B * 4)); BOA_TRY(m->wpos.reserve(B * 4)); BOA_TRY(m->cache.reserve(B)); BOA_TRY(m->started.reserve(B));
    BOA_TRY(m->v.reserve(B * 4)); BOA_TRY(m->rpos.reserve(B * 4)); BOA_TRY(m->off.reserve(B * 8)); BOA_TRY(m->size.reserve(B * 4));
    BOA_TRY(m->first.reserve(B)); BOA_TRY(m->err.reserve(4)); BOA_TRY(m->total.reserve(16));
    m->Bcap = B;
  }
  if (cap) BOA_TRY(m->scratch.reserve(m->Bcap * cap));
  return BOA_OK;
}

CoderArrays fx_coder_arrays(boa_fx_model* m, uint32_t cap) {
  CoderArrays ca{};
  ca.pos = m->pos.as<uint32_t>(); ca.len = m->len.as<uint32_t>();
  ca.low = m->low.as<uint64_t>(); ca.range = m->range.as<uint32_t>(); ca.pending = m->pending.as<uint32_t>();
  ca.wpos = m->wpos.as<uint32_t>(); ca.cache = m->cache.as<uint8_t>(); ca.started = m->started.as<uint8_t>();
  ca.scratch = m->scratch.as<uint8_t>(); ca.cap = cap;
  ca.v = m->v.as<uint32_t>(); ca.rpos = m->rpos.as<uint32_t>();
  ca.off = m->off.as<uint64_t>(); ca.size = m->size.as<uint32_t>();
  ca.payload = nullptr; ca.err = m->err.as<int>();
  return ca;
}

struct FxCtx {
  boa_fx_model* m;
  cudaStream_t st;
  int B, mode;
  uint8_t* data;
  size_t chunk_bytes;
  CoderArrays ca;
  uint32_t* dump_cdf = nullptr;
  int32_t* dump_logits = nullptr;
  uint32_t dump_steps = 0, dump_t = 0;
};

// a contraction of the step: the activation image in qa and the row shifts in ka (written by the producing kernel)
// against a weight image -> out [B][N] (+ resid)
int fx_contract(FxCtx& c, int K, const uint8_t* qw, const int32_t* sw, int N, int32_t* out, int ldo, const int32_t* resid) {
  boa_fx_model* m = c.m;
  const int KB = (int)fx_kb((size_t)K), nst = std::min(KB, fx::TC_MAXST);
  const dim3 grid((unsigned)((N + fx::TBN - 1) / fx::TBN), (unsigned)((c.B + fx::TBM - 1) / fx::TBM));
  fx::k_fx_gemm_tc<<<grid, 160, (size_t)nst * (fx::A_BLK + fx::W_BLK) + 1024, c.st>>>(m->qa.as<uint8_t>(), m->ka.as<int32_t>(), qw, sw, out,
                                                                                     ldo, resid, c.B, N, KB, nst);
  ++m->launches;
  BOA_CUDA_TRY(cudaPeekAtLastError());
  return BOA_OK;
}

// one model step + one coder step for the B streams of the wave, every operation an FX1 kernel (6 L + 3 launches)
int fx_step(FxCtx& c) {
  boa_fx_model* m = c.m;
  const int B = c.B, D = m->D, E = m->E;
  int32_t* u = m->u.as<int32_t>();
  int32_t* xz = m->xz.as<int32_t>();
  int32_t* xs = m->xs.as<int32_t>();
  int32_t* dbc = m->dbc.as<int32_t>();
  int32_t* logits = m->logits.as<int32_t>();
  int8_t* qa = m->qa.as<int8_t>();
  int32_t* ka = m->ka.as<int32_t>();
  const int ldd = (int)fx_kb((size_t)D), lde = (int)fx_kb((size_t)E);       // k-blocks of the activation images
  const int rgrid = (B + fx::RMS_ROWS - 1) / fx::RMS_ROWS;
  const fx::EmbedSrc es{c.data, c.chunk_bytes, c.ca.pos, c.ca.len, m->q_emb, m->s_emb};
  for (int l = 0; l < m->L; ++l) {
    const FxLayerDev& w = m->layers[l];
    int32_t* hl = m->h.as<int32_t>() + (size_t)l * m->Bcap * E * kNState;
    int32_t* winl = m->win.as<int32_t>() + (size_t)l * m->Bcap * 3 * E;
    if (l == 0) fx::k_fx_rmsnorm_q<true><<<rgrid, 32 * fx::RMS_ROWS, 0, c.st>>>(u, w.norm_w, D, m->sqrt_d, qa, ldd, ka, B, es);   // S1 + S2
    else fx::k_fx_rmsnorm_q<false><<<rgrid, 32 * fx::RMS_ROWS, 0, c.st>>>(u, w.norm_w, D, m->sqrt_d, qa, ldd, ka, B, es);
    BOA_TRY(fx_contract(c, D, w.q_in, w.s_in, 2 * E, xz, 2 * E, nullptr));
    fx::k_fx_conv_silu_q<<<B, 256, 0, c.st>>>(xz, winl, w.conv_w, w.conv_b, xs, m->tab, E, qa, lde, ka);
    BOA_TRY(fx_contract(c, E, w.q_x, w.s_x, m->J, dbc, m->ldj, nullptr));
    fx::k_fx_scan_q<<<B, 256, 0, c.st>>>(dbc, m->ldj, w.q_dt, w.s_dt, w.b_dt, w.a_neg, w.d_skip, xs, xz, hl, m->tab, E, m->R, qa, lde, ka);
    BOA_TRY(fx_contract(c, E, w.q_out, w.s_out, D, u, D, u));
    m->launches += 3;
  }
  fx::k_fx_quant_rows<<<rgrid, 32 * fx::RMS_ROWS, 0, c.st>>>(u, D, D, qa, ldd, ka, B);
  ++m->launches;
  BOA_TRY(fx_contract(c, D, m->q_head, m->s_emb, 256, logits, 256, nullptr));
  if (c.dump_logits)
    BOA_CUDA_TRY(cudaMemcpy2DAsync(c.dump_logits + (size_t)c.dump_t * 256, (size_t)c.dump_steps * 256 * 4, logits, 256 * 4, 256 * 4, B,
                                   cudaMemcpyDeviceToDevice, c.st));
  const int cgrid = (B * 32 + 255) / 256;
  if (c.mode == 0) fx::k_fx_coder_step<0><<<cgrid, 256, 0, c.st>>>(logits, c.data, c.chunk_bytes, c.ca, B, m->tab, c.dump_cdf, c.dump_steps);
  else fx::k_fx_coder_step<1><<<cgrid, 256, 0, c.st>>>(logits, c.data, c.chunk_bytes, c.ca, B, m->tab, nullptr, 0u);
  ++m->launches;
  BOA_CUDA_TRY(cudaPeekAtLastError());
  return BOA_OK;
}

// `steps` lock-step iterations: CUDA-graph batches of kStepsPerGraph steps, the remainder (and every dump step) eagerly
int fx_run_steps(FxCtx& c, uint64_t steps) {
  if (steps == 0) return BOA_OK;
  const bool dump = c.dump_cdf || c.dump_logits;
  const uint64_t S = kStepsPerGraph, n_batches = dump ? 0 : steps / S;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  int rc = BOA_OK;
  if (n_batches > 0) {
    const uint64_t before = c.m->launches;
    BOA_CUDA_TRY(cudaStreamBeginCapture(c.st, cudaStreamCaptureModeThreadLocal));
    for (uint64_t s = 0; s < S && rc == BOA_OK; ++s) rc = fx_step(c);
    cudaError_t e = cudaStreamEndCapture(c.st, &graph);
    const uint64_t per_graph = c.m->launches - before;
    c.m->launches = before;
    if (rc == BOA_OK && e != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
    if (rc == BOA_OK && (e = cudaGraphInstantiate(&exec, graph, 0)) != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
    for (uint64_t b = 0; b < n_batches && rc == BOA_OK; ++b) {
      if ((e = cudaGraphLaunch(exec, c.st)) != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
      c.m->launches += per_graph;
    }
    if (exec) cudaGraphExecDestroy(exec);
    if (graph) cudaGraphDestroy(graph);
  }
  for (uint64_t s = n_batches * S; s < steps && rc == BOA_OK; ++s) {
    c.dump_t = (uint32_t)s;
    rc = fx_step(c);
  }
  return rc;
}

int fx_reset(boa_fx_model* m, cudaStream_t st) {
  BOA_CUDA_TRY(cudaMemsetAsync(m->h.p, 0, (size_t)m->L * m->Bcap * m->E * kNState * 4, st));
  BOA_CUDA_TRY(cudaMemsetAsync(m->win.p, 0, (size_t)m->L * m->Bcap * 3 * m->E * 4, st));
  return BOA_OK;
}

uint64_t fx_wave_streams(const boa_fx_model* m, uint64_t nc, size_t cap) {
  const size_t per = (size_t)m->L * m->E * (kNState + 3) * 4 + (size_t)(m->D + 3 * m->E + m->ldj + 256) * 4 + m->E + 128 + cap;
  size_t free_b = 0, total_b = 0;
  uint64_t w = std::min<uint64_t>(nc, kMaxWaveStreams);
  if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) w = std::min<uint64_t>(w, std::max<uint64_t>(1, (uint64_t)(free_b * 0.8) / per + m->Bcap));
  else (void)cudaGetLastError();
  return std::max<uint64_t>(w, 1);
}

int fx_enter(boa_fx_model* m, void* user_stream, cudaStream_t* st) {
  BOA_CUDA_TRY(cudaEventRecord(m->user_ev, static_cast<cudaStream_t>(user_stream)));
  BOA_CUDA_TRY(cudaStreamWaitEvent(m->own, m->user_ev, 0));
  *st = m->own;
  return BOA_OK;
}

}  // namespace

extern "C" {

int boa_fx_compress(boa_fx_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, uint8_t* out, size_t* out_len, void* cuda_stream) {
  if (!m || !out || !out_len || chunk_bytes == 0 || chunk_bytes > kMaxChunkBytes || (n && !in)) return BOA_E_ARG;
  cudaStream_t st;
  BOA_TRY(fx_enter(m, cuda_stream, &st));
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  if (nc >= (1ull << 32)) return BOA_E_ARG;
  const size_t ib = index_bytes(nc), capacity = *out_len;
  if (capacity < ib) return BOA_E_CAPACITY;
  m->launches = 0;
  const bool in_dev = (n == 0) || is_device_ptr(in), out_dev = is_device_ptr(out);
  const uint8_t* d_in = in;
  if (!in_dev) {
    BOA_TRY(m->stage_in.reserve(n));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->stage_in.p, in, n, cudaMemcpyHostToDevice, st));
    d_in = m->stage_in.as<uint8_t>();
  }
  uint8_t* d_out = out;
  const size_t out_cap = std::min(capacity, boa_compress_bound(n, chunk_bytes));
  if (!out_dev) {
    BOA_TRY(m->stage_out.reserve(out_cap));
    d_out = m->stage_out.as<uint8_t>();
  }
  std::vector<uint8_t> index(ib, 0), first((size_t)nc);
  std::vector<uint32_t> sizes((size_t)nc);
  uint64_t payload_total = 0;
  if (nc) {
    const uint32_t cap = stream_cap(chunk_bytes);
    BOA_TRY(m->pin.reserve(16 + 5 * (size_t)nc));
    uint8_t* pin = m->pin.as<uint8_t>();
    uint32_t* pin_sizes = reinterpret_cast<uint32_t*>(pin + 16);
    uint8_t* pin_first = pin + 16 + 4 * (size_t)nc;
    const uint64_t W = fx_wave_streams(m, nc, cap);
    BOA_TRY(fx_reserve(m, std::min(W, nc), cap));
    BOA_CUDA_TRY(cudaMemsetAsync(m->total.p, 0, 16, st));
    for (uint64_t c0 = 0; c0 < nc; c0 += W) {
      const uint64_t B = std::min(W, nc - c0), wave_base = c0 * chunk_bytes;
      const uint64_t n_wave = std::min<uint64_t>(n - wave_base, B * chunk_bytes);
      BOA_TRY(fx_reset(m, st));
      FxCtx c{m, st, (int)B, 0, const_cast<uint8_t*>(d_in) + wave_base, chunk_bytes, fx_coder_arrays(m, cap)};
      const int g = (int)((B + 255) / 256);
      k_coder_init<0><<<g, 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n_wave, nullptr, nullptr);
      k_first_bytes<<<g, 256, 0, st>>>(c.data, chunk_bytes, m->first.as<uint8_t>(), (int)B);
      BOA_TRY(fx_run_steps(c, std::min<uint64_t>(chunk_bytes, n_wave) - 1));
      k_coder_finish<0><<<g, 256, 0, st>>>(c.ca, (int)B);
      k_wave_offsets<<<1, 1024, 0, st>>>(m->wpos.as<uint32_t>(), m->off.as<uint64_t>(), (int)B, m->total.as<uint64_t>());
      k_compact<<<(int)((B * 32 + 255) / 256), 256, 0, st>>>(m->scratch.as<uint8_t>(), cap, m->wpos.as<uint32_t>(), m->off.as<uint64_t>(),
                                                            d_out + ib, (uint64_t)(out_cap - ib), m->total.as<int>() + 2, (int)B);
      m->launches += 5;
      BOA_CUDA_TRY(cudaPeekAtLastError());
      BOA_CUDA_TRY(cudaMemcpyAsync(pin_sizes + c0, m->wpos.p, B * 4, cudaMemcpyDeviceToHost, st));
      BOA_CUDA_TRY(cudaMemcpyAsync(pin_first + c0, m->first.p, B, cudaMemcpyDeviceToHost, st));
    }
    BOA_CUDA_TRY(cudaMemcpyAsync(pin, m->total.p, 16, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
    int overflow = 0;
    memcpy(&payload_total, pin, 8);
    memcpy(&overflow, pin + 8, 4);
    if (overflow || ib + payload_total > out_cap) return BOA_E_CAPACITY;
    memcpy(sizes.data(), pin_sizes, 4 * (size_t)nc);
    memcpy(first.data(), pin_first, (size_t)nc);
  }
  write_index(index.data(), boa_fx_model_fingerprint(m), n, chunk_bytes, nc, first.data(), sizes.data());
  if (out_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(out, index.data(), ib, cudaMemcpyHostToDevice, st));
  } else {
    memcpy(out, index.data(), ib);
    if (payload_total) BOA_CUDA_TRY(cudaMemcpyAsync(out + ib, d_out + ib, payload_total, cudaMemcpyDeviceToHost, st));
  }
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  *out_len = ib + payload_total;
  return BOA_OK;
}

int boa_fx_decompress(boa_fx_model* m, const uint8_t* in, size_t in_len, uint8_t* out, size_t* out_len, void* cuda_stream) {
  if (!m || !in || !out_len) return BOA_E_ARG;
  if (in_len < kHeaderBytes + 4) return BOA_E_FORMAT;
  cudaStream_t st;
  BOA_TRY(fx_enter(m, cuda_stream, &st));
  const bool in_dev = is_device_ptr(in);
  m->launches = 0;
  Index ix;
  BOA_TRY(read_index(boa_fx_model_fingerprint(m), in, in_len, in_dev, st, ix));
  const uint64_t nc = ix.h.n_chunks;
  const size_t n = (size_t)ix.h.n, chunk_bytes = ix.h.chunk_bytes;
  if (*out_len < n) return BOA_E_CAPACITY;
  if (n && !out) return BOA_E_ARG;
  if (n == 0) { *out_len = 0; return BOA_OK; }
  const uint8_t* d_in = in;
  if (!in_dev) {
    BOA_TRY(m->stage_in.reserve(in_len));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->stage_in.p, in, in_len, cudaMemcpyHostToDevice, st));
    d_in = m->stage_in.as<uint8_t>();
  }
  const bool out_dev = is_device_ptr(out);
  uint8_t* d_out = out;
  if (!out_dev) {
    BOA_TRY(m->stage_out.reserve(n));
    d_out = m->stage_out.as<uint8_t>();
  }
  const uint64_t W = fx_wave_streams(m, nc, 0);
  BOA_TRY(fx_reserve(m, std::min(W, nc), 0));
  BOA_CUDA_TRY(cudaMemsetAsync(m->err.p, 0, 4, st));
  for (uint64_t c0 = 0; c0 < nc; c0 += W) {
    const uint64_t B = std::min(W, nc - c0), wave_base = c0 * chunk_bytes;
    const uint64_t n_wave = std::min<uint64_t>(n - wave_base, B * chunk_bytes);
    BOA_TRY(fx_reset(m, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->off.p, ix.offs.data() + c0, B * 8, cudaMemcpyHostToDevice, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->size.p, ix.sizes.data() + c0, B * 4, cudaMemcpyHostToDevice, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->first.p, ix.bytes.data() + kHeaderBytes + c0, B, cudaMemcpyHostToDevice, st));
    FxCtx c{m, st, (int)B, 1, d_out + wave_base, chunk_bytes, fx_coder_arrays(m, 0)};
    c.ca.payload = d_in + ix.ib;
    const int g = (int)((B + 255) / 256);
    k_coder_init<1><<<g, 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n_wave, m->first.as<uint8_t>(), c.data);
    BOA_TRY(fx_run_steps(c, std::min<uint64_t>(chunk_bytes, n_wave) - 1));
    k_coder_finish<1><<<g, 256, 0, st>>>(c.ca, (int)B);
    m->launches += 2;
    BOA_CUDA_TRY(cudaPeekAtLastError());
  }
  int err = 0;
  BOA_CUDA_TRY(cudaMemcpyAsync(&err, m->err.p, 4, cudaMemcpyDeviceToHost, st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  if (err) return BOA_E_CORRUPT;
  if (!out_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(out, d_out, n, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
  }
  *out_len = n;
  return BOA_OK;
}

uint64_t boa_fx_last_launches(const boa_fx_model* m) { return m ? m->launches : 0; }

int boa_fx_debug_step_dump(boa_fx_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t n_steps, int32_t* logits,
                           uint32_t* cdf, void* cuda_stream) {
  if (!m || !in || chunk_bytes < 2 || n == 0 || n % chunk_bytes != 0 || n_steps == 0 || n_steps > chunk_bytes - 1) return BOA_E_ARG;
  cudaStream_t st;
  BOA_TRY(fx_enter(m, cuda_stream, &st));
  const uint64_t B = n / chunk_bytes;
  if (B > kMaxWaveStreams) return BOA_E_ARG;
  const size_t rows = (size_t)B * n_steps;
  TmpDev tin, tl, tc;
  BOA_TRY(tin.init(in, n, true, false, st));
  BOA_TRY(tl.init(logits, rows * 256 * 4, false, true, st));
  BOA_TRY(tc.init(cdf, rows * 257 * 4, false, true, st));
  const uint32_t cap = stream_cap(chunk_bytes);
  BOA_TRY(fx_reserve(m, B, cap));
  BOA_TRY(fx_reset(m, st));
  FxCtx c{m, st, (int)B, 0, static_cast<uint8_t*>(tin.dev), chunk_bytes, fx_coder_arrays(m, cap)};
  c.dump_logits = static_cast<int32_t*>(tl.dev);
  c.dump_cdf = static_cast<uint32_t*>(tc.dev);
  c.dump_steps = (uint32_t)n_steps;
  k_coder_init<0><<<(int)((B + 255) / 256), 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n, nullptr, nullptr);
  BOA_TRY(fx_run_steps(c, n_steps));
  BOA_TRY(tl.finish(st));
  BOA_TRY(tc.finish(st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  return BOA_OK;
}

}  // extern "C"
