// coder_kernels.cuh — softmax, integer table, range coder (S11-S16 of SURVEY §8(a)).
//
//   softmax        eq. 6
//   integer table  eq. 7: f >= 1, sum f = 2^16; the rounding rule is reading R#5:
//        m = max l ; e[a] = EXP(l[a]-m) ; g[a] = min(floor(e[a]*2^23), 2^23) ; G = prefix sums ; T = G[256]
//        C[a] = a + floor(G[a]*(2^16-256)/T)
//     EXP is a *specified* fp32 algorithm (individually rounded mul/add/sub, no FMA contraction), so the
//     integer g[a] is a pure function of the fp32 logits; all later arithmetic is integer and order-free.
//   encoder        eq. 8-11, carry-propagating form (R#6), 4-byte flush (R#9)
//   decoder        eq. 12-13 with V = C - L (R#7); symbol search without division
//
// One warp per stream-step builds the table (8 symbols per lane, shuffle prefix sums); one lane of
// it carries the coder state of that stream ("one thread per chunk", R#19).
#pragma once
#include "common.cuh"
#include "tc_gemm.cuh"

namespace boa {

// ------------------------------------------------------------------------------------------ EXP (R#5)
__device__ __forceinline__ float exp_spec(float d) {
  const float LOG2E = __uint_as_float(0x3FB8AA3Bu);
  const float t = __fmul_rn(d, LOG2E);
  if (!(t >= -64.0f)) return 0.0f;               // also NaN
  const float n = rintf(t);                      // round half to even
  const float r = __fsub_rn(t, n);               // exact
  float p = __uint_as_float(0x39212C6Cu);
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3AAFA26Eu));
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3C1D9662u));
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3D63576Bu));
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3E75FDEEu));
  p = __fadd_rn(__fmul_rn(p, r), __uint_as_float(0x3F317218u));
  p = __fadd_rn(__fmul_rn(p, r), 1.0f);
  const float sc = __int_as_float(((int)n + 127) << 23);   // 2^n, n in [-64, 64]
  return __fmul_rn(p, sc);                       // exact scaling
}

// Table of one stream-step, distributed over a warp: lane owns symbols a = 8*lane .. 8*lane+7.
struct WarpTable {
  uint32_t g[8];    // g[a]
  uint32_t gex;     // G[8*lane]  (exclusive prefix at the lane's first symbol)
  uint32_t T;       // G[256]
  bool bad;         // non-finite maximum or a NaN logit -> uniform table (R#17)
  float e[8];       // EXP values (for the probability dump)
};

__device__ __forceinline__ void build_table(const float (&l)[8], WarpTable& t) {
  float m = l[0];
  bool nan = (l[0] != l[0]);
#pragma unroll
  for (int k = 1; k < 8; ++k) { m = fmaxf(m, l[k]); nan |= (l[k] != l[k]); }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, o));
  const bool any_nan = __any_sync(0xffffffffu, nan);
  t.bad = any_nan || !(fabsf(m) <= 3.402823466e38f);
  uint32_t sum = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const float e = t.bad ? 0.0f : exp_spec(__fsub_rn(l[k], m));
    t.e[k] = e;
    const uint32_t g = min(__float2uint_rd(__fmul_rn(e, 8388608.0f)), kGOne);
    t.g[k] = g;
    sum += g;
  }
  uint32_t inc = sum;                               // inclusive scan over lanes
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  t.gex = inc - sum;
  t.T = __shfl_sync(0xffffffffu, inc, 31);
}

// C[a] = a + floor(G[a] * 65280 / T)   (64-bit integers; G <= T <= 2^31)
__device__ __forceinline__ uint32_t cdf_value(uint32_t a, uint32_t G, uint32_t T) {
  return a + (uint32_t)(((uint64_t)G * (kM - 256u)) / T);
}

// G[s] for an arbitrary symbol s, fetched from the owning lane (all lanes call).
__device__ __forceinline__ void table_lookup(const WarpTable& t, uint32_t s, uint32_t& Gs, uint32_t& gs) {
  uint32_t run = t.gex, Gl = 0, gl = 0;
  const uint32_t k = s & 7u;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    if (j == (int)k) { Gl = run; gl = t.g[j]; }
    run += t.g[j];
  }
  Gs = __shfl_sync(0xffffffffu, Gl, s >> 3);
  gs = __shfl_sync(0xffffffffu, gl, s >> 3);
}

// [c_lo, c_hi) of symbol s.  Lanes 0 and 1 each do one 64-bit division.
__device__ __forceinline__ void table_interval(const WarpTable& t, uint32_t s, uint32_t& c_lo, uint32_t& c_hi) {
  if (t.bad) { c_lo = s << 8; c_hi = (s + 1u) << 8; return; }
  uint32_t Gs, gs;
  table_lookup(t, s, Gs, gs);
  const int lane = threadIdx.x & 31;
  uint32_t c = 0;
  if (lane < 2) c = cdf_value(s + lane, Gs + (lane ? gs : 0u), t.T);
  c_lo = __shfl_sync(0xffffffffu, c, 0);
  c_hi = __shfl_sync(0xffffffffu, c, 1);
}

// The unique s with C[s] <= x < C[s+1], x in [0, 2^16).
//   C[a] <= x  <=>  a <= x  and  G[a]*65280 < (x - a + 1)*T      (floor(n/T) <= y <=> n < (y+1)T)
// C is strictly increasing, so the predicate is monotone in a and s = (#a in 0..255 with C[a] <= x) - 1.
__device__ __forceinline__ uint32_t table_search(const WarpTable& t, uint32_t x) {
  if (t.bad) return x >> 8;
  const int lane = threadIdx.x & 31;
  uint32_t run = t.gex, cnt = 0;
#pragma unroll
  for (int j = 0; j < 8; ++j) {
    const uint32_t a = 8u * lane + j;
    const bool le = (a <= x) && ((uint64_t)run * (kM - 256u) < (uint64_t)(x - a + 1u) * t.T);
    cnt += le ? 1u : 0u;
    run += t.g[j];
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
  return cnt - 1u;
}

// ------------------------------------------------------------------------------- range coder state
struct EncState {            // eq. 8-11; `low` uses bits 0..32 (bit 32 = carry)
  uint64_t low;
  uint32_t range;
  uint32_t pending;
  uint32_t wpos;             // bytes written so far
  uint8_t cache;
  uint8_t started;
};

// Where the encoder's bytes go.  ByteSink: one store per byte (test kernels, rows of any alignment).  VecSink: the
// stream's payload scratch row in 16-byte blocks ("coalesced vectorised stores", north_star): bytes are collected in four
// registers and leave as one aligned 16-byte store when a block is full; begin() reloads a block left partly filled by
// an earlier launch, end() stores the current partial block (the bytes beyond wpos in it are not payload: the row is
// 16-byte aligned and padded, and the compaction copies sizes[i] bytes only).
struct ByteSink {
  uint8_t* out;
  __device__ __forceinline__ void begin(uint8_t* row, uint32_t) { out = row; }
  __device__ __forceinline__ void put(uint32_t& wpos, uint8_t b) { out[wpos++] = b; }
  __device__ __forceinline__ void end(uint32_t) {}
};
struct VecSink {
  uint8_t* out;
  uint32_t w[4];
  __device__ __forceinline__ void begin(uint8_t* row, uint32_t wpos) {
    out = row;
    uint4 v = make_uint4(0u, 0u, 0u, 0u);
    if (wpos & 15u) v = *reinterpret_cast<const uint4*>(row + (wpos & ~15u));
    w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
  }
  __device__ __forceinline__ void put(uint32_t& wpos, uint8_t b) {
    const uint32_t k = wpos & 15u, sh = (k & 3u) * 8u;
#pragma unroll
    for (int j = 0; j < 4; ++j)
      if ((k >> 2) == (uint32_t)j) w[j] = (w[j] & ~(0xFFu << sh)) | ((uint32_t)b << sh);
    ++wpos;
    if ((wpos & 15u) == 0u) *reinterpret_cast<uint4*>(out + wpos - 16u) = make_uint4(w[0], w[1], w[2], w[3]);
  }
  __device__ __forceinline__ void end(uint32_t wpos) {
    if (wpos & 15u) *reinterpret_cast<uint4*>(out + (wpos & ~15u)) = make_uint4(w[0], w[1], w[2], w[3]);
  }
};

template <class Sink>
__device__ __forceinline__ void enc_shift_low(EncState& s, Sink& out) {
  const uint32_t lo32 = (uint32_t)s.low;
  const uint32_t carry = (uint32_t)(s.low >> 32);
  if (lo32 < 0xFF000000u || carry == 1u) {
    if (s.started) out.put(s.wpos, (uint8_t)(s.cache + carry));
    const uint8_t fill = (uint8_t)(0xFFu + carry);
    for (; s.pending; --s.pending) out.put(s.wpos, fill);
    s.started = 1;
    s.cache = (uint8_t)(lo32 >> 24);
  } else {
    ++s.pending;
  }
  s.low = (uint64_t)(lo32 & 0x00FFFFFFu) << 8;
}

template <class Sink>
__device__ __forceinline__ void enc_symbol(EncState& s, uint32_t c_lo, uint32_t c_hi, Sink& out) {
  s.low += ((uint64_t)s.range * c_lo) >> kFreqBits;                      // eq. 8
  s.range = (uint32_t)(((uint64_t)s.range * (c_hi - c_lo)) >> kFreqBits); // eq. 9
  while (s.range < kRcTop) {                                              // eq. 10-11 (R#6)
    enc_shift_low(s, out);
    s.range <<= 8;
  }
}

struct DecState {
  uint32_t range;
  uint32_t v;                // V = C - L (R#7)
  uint32_t rpos;             // bytes consumed
};

__device__ __forceinline__ uint32_t dec_target(const DecState& s, bool& corrupt) {
  uint64_t x = ((((uint64_t)s.v + 1u) << kFreqBits) - 1u) / s.range;      // eq. 12
  if (x >= kM) { corrupt = true; x = kM - 1u; }
  return (uint32_t)x;
}

__device__ __forceinline__ void dec_consume(DecState& s, uint32_t c_lo, uint32_t c_hi, const uint8_t* in,
                                            uint32_t size, bool& corrupt) {
  s.v -= (uint32_t)(((uint64_t)s.range * c_lo) >> kFreqBits);
  s.range = (uint32_t)(((uint64_t)s.range * (c_hi - c_lo)) >> kFreqBits);
  while (s.range < kRcTop) {
    uint32_t b = 0;
    if (s.rpos < size) b = in[s.rpos]; else corrupt = true;
    ++s.rpos;
    s.v = (s.v << 8) | b;                                                 // eq. 13
    s.range <<= 8;
    if (s.range == 0) { corrupt = true; s.range = 0xFFFFFFFFu; }          // only reachable on corrupt input
  }
}

// Per-wave, per-stream coder arrays (struct of arrays; device memory owned by the workspace).
struct CoderArrays {
  uint32_t* pos;        // symbols coded so far (= model steps taken) per stream
  uint32_t* len;        // stream length in bytes
  // encoder
  uint64_t* low; uint32_t* range; uint32_t* pending; uint32_t* wpos; uint8_t* cache; uint8_t* started;
  uint8_t* scratch;     // [B][cap] per-stream payload scratch
  uint32_t cap;
  // decoder
  uint32_t* v; uint32_t* rpos; const uint64_t* off; const uint32_t* size;
  const uint8_t* payload;   // container payload base (device)
  int* err;             // device flag: != 0 -> BOA_E_CORRUPT
};

// S1 for the NEXT step, fused into the coder step: once the symbol is known the warp writes u = Emb[s] (fp32, the
// residual stream) and the image of u * norm_w(layer 0), the operand of the first in_proj (tc_gemm.cuh).
struct EmbedArgs {
  const float4* emb;       // [256][D/4]
  const float4* norm_w;    // [D/4] RMSNorm weight of layer 0
  float4* u;               // [B][D/4]
  uint8_t* u_img;
  float* ssq;              // [B][D/64] sums of u^2 over 64-column blocks (same order as k_embed)
  int D4;
};
// all 32 lanes call (shuffles inside)
__device__ __forceinline__ void embed_row(const EmbedArgs& ea, int i, uint32_t s, int lane) {
  for (int q0 = 0; q0 < ea.D4; q0 += 32) {
    const int q = q0 + lane;
    const bool live = q < ea.D4;                  // D4 is a multiple of 16: a 16-lane block is live as a whole
    const float4 v = ea.emb[s * ea.D4 + (live ? q : 0)];
    float ss = v.x * v.x;
    ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
#pragma unroll
    for (int d = 8; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
    if (live) {
      ea.u[(size_t)i * ea.D4 + q] = v;
      if ((q & 15) == 0) ea.ssq[(size_t)i * (ea.D4 >> 4) + (q >> 4)] = ss;
      const float4 w = ea.norm_w[q];
      tc::cut4_store(ea.u_img, ea.D4 >> 4, i, q * 4, make_float4(v.x * w.x, v.y * w.y, v.z * w.z, v.w * w.w));
    }
  }
}

// -------------------------------------------------------------------------------------- step kernel
// MODE 0 = encode, 1 = decode.  One warp per stream.  `data` is the input (encode) or output (decode)
// buffer of this wave: stream i, byte t at data[i*chunk + t].
// DUMP: additionally write logits-derived probabilities / the whole CDF for row i*dump_steps + pos.
// One coder step of stream i by one warp (all 32 lanes call): table from the stream's logits, the symbol's interval
// (encode) or the search for the decoder's target (decode), the coder update by lane 0, the embedding of the next byte.
// Shared by k_coder_step (one launch per step) and the persistent step kernel (step_persist.cuh).
template <int MODE, bool DUMP>
__device__ __forceinline__ void coder_step_one(int i, int lane, const float* __restrict__ logits, uint8_t* data, size_t chunk_bytes,
                                               const CoderArrays& ca, const EmbedArgs& ea, float* dump_probs, uint32_t* dump_cdf,
                                               uint32_t dump_steps) {
  const uint32_t pos = ca.pos[i], len = ca.len[i];
  if (pos + 1u >= len) return;                    // finished stream: masked

  float l[8];
  {
    const float4* lp = reinterpret_cast<const float4*>(logits + (size_t)i * 256 + lane * 8);
    const float4 a = lp[0], b = lp[1];
    l[0] = a.x; l[1] = a.y; l[2] = a.z; l[3] = a.w; l[4] = b.x; l[5] = b.y; l[6] = b.z; l[7] = b.w;
  }
  WarpTable t;
  build_table(l, t);

  if (DUMP) {
    const size_t row = (size_t)i * dump_steps + pos;
    if (dump_probs) {
      float se = 0.0f;
#pragma unroll
      for (int k = 0; k < 8; ++k) se += t.e[k];
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) se += __shfl_xor_sync(0xffffffffu, se, o);
#pragma unroll
      for (int k = 0; k < 8; ++k)
        dump_probs[row * 256 + lane * 8 + k] = t.bad ? (1.0f / 256.0f) : t.e[k] / se;
    }
    if (dump_cdf) {
      uint32_t run = t.gex;
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t a = 8u * lane + k;
        dump_cdf[row * 257 + a] = t.bad ? (a << 8) : cdf_value(a, run, t.T);
        run += t.g[k];
      }
      if (lane == 31) dump_cdf[row * 257 + 256] = kM;
    }
  }

  uint8_t* sdata = data + (size_t)i * chunk_bytes;
  if (MODE == 0) {
    const uint32_t s = sdata[pos + 1u];
    embed_row(ea, i, s, lane);
    uint32_t c_lo, c_hi;
    table_interval(t, s, c_lo, c_hi);
    if (lane == 0) {
      EncState st;
      st.low = ca.low[i]; st.range = ca.range[i]; st.pending = ca.pending[i]; st.wpos = ca.wpos[i];
      st.cache = ca.cache[i]; st.started = ca.started[i];
      VecSink sink;
      sink.begin(ca.scratch + (size_t)i * ca.cap, st.wpos);
      enc_symbol(st, c_lo, c_hi, sink);
      sink.end(st.wpos);
      ca.low[i] = st.low; ca.range[i] = st.range; ca.pending[i] = st.pending; ca.wpos[i] = st.wpos;
      ca.cache[i] = st.cache; ca.started[i] = st.started;
      ca.pos[i] = pos + 1u;
    }
  } else {
    DecState st;
    bool corrupt = false;
    uint32_t x = 0;
    if (lane == 0) {
      st.range = ca.range[i]; st.v = ca.v[i]; st.rpos = ca.rpos[i];
      x = dec_target(st, corrupt);
    }
    x = __shfl_sync(0xffffffffu, x, 0);
    const uint32_t s = table_search(t, x);
    embed_row(ea, i, s, lane);
    uint32_t c_lo, c_hi;
    table_interval(t, s, c_lo, c_hi);
    if (lane == 0) {
      dec_consume(st, c_lo, c_hi, ca.payload + ca.off[i], ca.size[i], corrupt);
      ca.range[i] = st.range; ca.v[i] = st.v; ca.rpos[i] = st.rpos;
      sdata[pos + 1u] = (uint8_t)s;
      ca.pos[i] = pos + 1u;
      if (corrupt) *ca.err = 1;
    }
  }
}

template <int MODE, bool DUMP>
__global__ void __launch_bounds__(256)
k_coder_step(const float* __restrict__ logits, uint8_t* data, size_t chunk_bytes, CoderArrays ca, int B,
             EmbedArgs ea, float* dump_probs, uint32_t* dump_cdf, uint32_t dump_steps, uint32_t* zero, int n_zero) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  pdl_launch();
  pdl_wait();                                     // logits, coder state and (decode) the output buffer come from earlier kernels
  // the row-tile counters of this step's chained contractions (tc::k_gemm_chain) start the next step at zero
  for (int k = blockIdx.x * blockDim.x + threadIdx.x; k < n_zero; k += gridDim.x * blockDim.x) zero[k] = 0u;
  if (i >= B) return;
  coder_step_one<MODE, DUMP>(i, lane, logits, data, chunk_bytes, ca, ea, dump_probs, dump_cdf, dump_steps);
}

// Encode-side time slab: the T tables of a stream (logits rows i*T + t) are coded one after the
// other by the stream's warp, the coder state staying in registers.  Per symbol this is the arithmetic of the step
// kernel, so the bytes are the ones the step path writes.
__global__ void __launch_bounds__(256)
k_coder_slab(const float* __restrict__ logits, const uint8_t* __restrict__ data, size_t chunk_bytes, CoderArrays ca,
             int B, int T) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  pdl_launch();
  pdl_wait();
  if (i >= B) return;
  const uint32_t pos = ca.pos[i], len = ca.len[i];
  if (pos + 1u >= len) return;                    // finished stream: masked
  EncState st;
  st.low = ca.low[i]; st.range = ca.range[i]; st.pending = ca.pending[i]; st.wpos = ca.wpos[i];
  st.cache = ca.cache[i]; st.started = ca.started[i];
  const uint8_t* sdata = data + (size_t)i * chunk_bytes;
  VecSink out;                                    // (used by lane 0 only) the slab's bytes leave in 16-byte blocks
  out.begin(ca.scratch + (size_t)i * ca.cap, st.wpos);
  uint32_t done = 0;
  for (int t = 0; t < T && pos + 1u + (uint32_t)t < len; ++t) {
    float l[8];
    const float4* lp = reinterpret_cast<const float4*>(logits + ((size_t)i * T + t) * 256 + lane * 8);
    const float4 a = lp[0], b = lp[1];
    l[0] = a.x; l[1] = a.y; l[2] = a.z; l[3] = a.w; l[4] = b.x; l[5] = b.y; l[6] = b.z; l[7] = b.w;
    WarpTable tb;
    build_table(l, tb);
    const uint32_t s = sdata[pos + 1u + (uint32_t)t];
    uint32_t c_lo, c_hi;
    table_interval(tb, s, c_lo, c_hi);
    if (lane == 0) enc_symbol(st, c_lo, c_hi, out);
    ++done;
  }
  if (lane == 0) {
    out.end(st.wpos);
    ca.low[i] = st.low; ca.range[i] = st.range; ca.pending[i] = st.pending; ca.wpos[i] = st.wpos;
    ca.cache[i] = st.cache; ca.started[i] = st.started;
    ca.pos[i] = pos + done;
  }
}

// S0 / S16: per-stream initialisation.  Encode: coder state reset.  Decode: first byte -> output,
// V = first four payload bytes (big-endian).
template <int MODE>
__global__ void k_coder_init(CoderArrays ca, int B, size_t chunk_bytes, uint64_t n_wave,
                             const uint8_t* first, uint8_t* out_data) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= B) return;
  const uint64_t begin = (uint64_t)i * chunk_bytes;
  const uint64_t l = min((uint64_t)chunk_bytes, n_wave - begin);
  ca.len[i] = (uint32_t)l;
  ca.pos[i] = 0;
  ca.range[i] = 0xFFFFFFFFu;
  if (MODE == 0) {
    ca.low[i] = 0; ca.pending[i] = 0; ca.wpos[i] = 0; ca.cache[i] = 0; ca.started[i] = 0;
  } else {
    out_data[begin] = first[i];
    const uint8_t* p = ca.payload + ca.off[i];
    const uint32_t size = ca.size[i];
    uint32_t v = 0;
    if (size < 4u) { *ca.err = 1; }
    else v = ((uint32_t)p[0] << 24) | ((uint32_t)p[1] << 16) | ((uint32_t)p[2] << 8) | (uint32_t)p[3];
    ca.v[i] = v;
    ca.rpos[i] = 4;
  }
}

// S15: flush (five shift_low, R#9) -> final per-stream sizes in wpos.   Decode: exact-consumption check.
template <int MODE>
__global__ void k_coder_finish(CoderArrays ca, int B) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= B) return;
  if (MODE == 0) {
    EncState st;
    st.low = ca.low[i]; st.range = ca.range[i]; st.pending = ca.pending[i]; st.wpos = ca.wpos[i];
    st.cache = ca.cache[i]; st.started = ca.started[i];
    VecSink out;
    out.begin(ca.scratch + (size_t)i * ca.cap, st.wpos);
    for (int k = 0; k < 5; ++k) enc_shift_low(st, out);
    out.end(st.wpos);
    ca.wpos[i] = st.wpos;
  } else {
    if (ca.rpos[i] != ca.size[i] || ca.pos[i] + 1u != ca.len[i]) *ca.err = 1;
  }
}

// S15: per-stream sizes -> payload offsets.  off[i] = total + sum_{j<i} sizes[j] (exclusive scan), then total += the
// wave's sum, so the next wave continues where this one ends and the host never sees the sizes in between.
// One block of 1024 threads (B <= 65,536: at most 64 consecutive streams per thread); integer sums: order-free.
__global__ void __launch_bounds__(1024) k_wave_offsets(const uint32_t* __restrict__ sizes, uint64_t* __restrict__ off, int B,
                                                       uint64_t* __restrict__ total) {
  __shared__ uint64_t warp_sum[32];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int per = (B + 1023) / 1024, i0 = tid * per, i1 = min(B, i0 + per);
  uint64_t mine = 0;
  for (int i = i0; i < i1; ++i) mine += sizes[i];
  uint64_t inc = mine;                             // inclusive scan over the warp, then over the 32 warp sums
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint64_t v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  if (lane == 31) warp_sum[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    uint64_t w = warp_sum[lane], winc = w;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint64_t v = __shfl_up_sync(0xffffffffu, winc, o);
      if (lane >= o) winc += v;
    }
    warp_sum[lane] = winc - w;                     // exclusive
  }
  __syncthreads();
  const uint64_t base = *total;
  uint64_t run = base + warp_sum[warp] + (inc - mine);
  for (int i = i0; i < i1; ++i) { off[i] = run; run += sizes[i]; }
  __syncthreads();                                 // every thread has read *total
  if (tid == 1023) *total = run;                   // the last thread's running sum is the new total (empty ranges add 0)
}

// S15: pack the per-stream scratch payloads back to back.  One warp per stream; the body moves 16 bytes per lane and
// instruction with stores aligned in the destination (the scratch rows start 16-byte aligned, the packed position does
// not: each 16-byte block is funnel-shifted together from five aligned source words); byte loops for head and tail.
// A payload that would end beyond dst_cap is not written and raises *overflow (BOA_E_CAPACITY).
__global__ void k_compact(const uint8_t* __restrict__ scratch, uint32_t cap, const uint32_t* __restrict__ sizes,
                          const uint64_t* __restrict__ off, uint8_t* __restrict__ dst, uint64_t dst_cap,
                          int* __restrict__ overflow, int B) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= B) return;
  const uint8_t* s = scratch + (size_t)i * cap;
  const uint32_t n = sizes[i];
  const uint64_t o = off[i];
  if (o + n > dst_cap) { if (lane == 0) *overflow = 1; return; }
  uint8_t* d = dst + o;
  const uint32_t head = min(n, (uint32_t)((16u - (uint32_t)(reinterpret_cast<uintptr_t>(d) & 15u)) & 15u));
  for (uint32_t k = lane; k < head; k += 32) d[k] = s[k];
  const uint32_t nblk = (n - head) >> 4;
  const uint32_t sh = (head & 3u) * 8u;            // misalignment of the source of a block, in bits
  const uint32_t* sw = reinterpret_cast<const uint32_t*>(s + (head & ~3u));
  uint4* dv = reinterpret_cast<uint4*>(d + head);
  for (uint32_t b = lane; b < nblk; b += 32) {
    const uint32_t* p = sw + 4 * b;
    const uint32_t w0 = p[0], w1 = p[1], w2 = p[2], w3 = p[3], w4 = sh ? p[4] : 0u;   // p[4] stays inside the row: cap >= n + 4
    dv[b] = make_uint4(__funnelshift_r(w0, w1, sh), __funnelshift_r(w1, w2, sh), __funnelshift_r(w2, w3, sh),
                       __funnelshift_r(w3, w4, sh));
  }
  for (uint32_t k = head + (nblk << 4) + lane; k < n; k += 32) d[k] = s[k];
}

// first byte of each stream
__global__ void k_first_bytes(const uint8_t* __restrict__ in, size_t chunk_bytes, uint8_t* __restrict__ first, int B) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < B) first[i] = in[(size_t)i * chunk_bytes];
}

// ------------------------------------------------------------------------------- test-only kernels
__global__ void k_debug_quantise(const float* __restrict__ logits, uint32_t* __restrict__ cdf, size_t rows) {
  const size_t row = ((size_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (row >= rows) return;
  float l[8];
#pragma unroll
  for (int k = 0; k < 8; ++k) l[k] = logits[row * 256 + lane * 8 + k];
  WarpTable t;
  build_table(l, t);
  uint32_t run = t.gex;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const uint32_t a = 8u * lane + k;
    cdf[row * 257 + a] = t.bad ? (a << 8) : cdf_value(a, run, t.T);
    run += t.g[k];
  }
  if (lane == 31) cdf[row * 257 + 256] = kM;
}

// The coder alone, one thread per stream, driven by explicit tables cdf[i][t][257].
__global__ void k_debug_rc_encode(const uint32_t* __restrict__ cdf, const uint8_t* __restrict__ syms, int B,
                                  uint32_t len, uint8_t* out, uint32_t cap, uint32_t* sizes, int* err) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= B) return;
  EncState st;
  st.low = 0; st.range = 0xFFFFFFFFu; st.pending = 0; st.wpos = 0; st.cache = 0; st.started = 0;
  ByteSink o;
  o.begin(out + (size_t)i * cap, 0u);
  for (uint32_t t = 0; t < len; ++t) {
    if (st.wpos + st.pending + 8u > cap) { *err = 1; sizes[i] = 0; return; }
    const uint32_t* C = cdf + ((size_t)i * len + t) * 257;
    const uint32_t s = syms[(size_t)i * len + t];
    enc_symbol(st, C[s], C[s + 1], o);
  }
  if (st.wpos + st.pending + 8u > cap) { *err = 1; sizes[i] = 0; return; }
  for (int k = 0; k < 5; ++k) enc_shift_low(st, o);
  sizes[i] = st.wpos;
}

__global__ void k_debug_rc_decode(const uint32_t* __restrict__ cdf, const uint8_t* __restrict__ in, uint32_t cap,
                                  const uint32_t* __restrict__ sizes, int B, uint32_t len, uint8_t* syms, int* err) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= B) return;
  const uint8_t* p = in + (size_t)i * cap;
  const uint32_t size = sizes[i];
  bool corrupt = size < 4u;
  DecState st;
  st.range = 0xFFFFFFFFu; st.rpos = 4;
  st.v = corrupt ? 0u : (((uint32_t)p[0] << 24) | ((uint32_t)p[1] << 16) | ((uint32_t)p[2] << 8) | (uint32_t)p[3]);
  for (uint32_t t = 0; t < len; ++t) {
    const uint32_t* C = cdf + ((size_t)i * len + t) * 257;
    const uint32_t x = dec_target(st, corrupt);
    uint32_t lo = 0, hi = 256;                    // C[lo] <= x < C[hi]
    while (hi - lo > 1u) { const uint32_t mid = (lo + hi) >> 1; if (C[mid] <= x) lo = mid; else hi = mid; }
    dec_consume(st, C[lo], C[lo + 1], p, size, corrupt);
    syms[(size_t)i * len + t] = (uint8_t)lo;
  }
  if (st.rpos != size) corrupt = true;
  if (corrupt) *err = 1;
}

}  // namespace boa
