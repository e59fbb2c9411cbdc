// fx_coder.cuh — FX1: the integer table (R#5's rule on the integer exponential) and the coder step.
// The table arithmetic after g (prefix sums, C[a] = a + floor(G[a] 65280 / T), the division-free search) and the range
// coder are those of coder_kernels.cuh; only g comes from fx::exp_neg instead of the fp32 EXP.
#pragma once
#include "coder_kernels.cuh"
#include "fx_kernels.cuh"

namespace boa {
namespace fx {

// lane owns symbols 8 lane .. 8 lane + 7;  d = max - logit >= 0 (Q);  g = exp_neg(d) >> 7 in [0, 2^23]
__device__ __forceinline__ void build_table_fx(const Tables& tb, const int32_t (&l)[8], WarpTable& t) {
  int32_t m = l[0];
#pragma unroll
  for (int k = 1; k < 8; ++k) m = max(m, l[k]);
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = max(m, __shfl_xor_sync(0xffffffffu, m, o));
  t.bad = false;
  uint32_t sum = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int64_t d = (int64_t)m - (int64_t)l[k];
    const uint32_t g = (uint32_t)(exp_neg(tb, d > QMAX ? QMAX : d) >> 7);
    t.g[k] = g;
    t.e[k] = 0.0f;
    sum += g;
  }
  uint32_t inc = sum;
  const int lane = threadIdx.x & 31;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const uint32_t v = __shfl_up_sync(0xffffffffu, inc, o);
    if (lane >= o) inc += v;
  }
  t.gex = inc - sum;
  t.T = __shfl_sync(0xffffffffu, inc, 31);
}

// One warp per stream.  MODE 0 = encode (next symbol from `data`), 1 = decode (symbol from the coder, written to `data`).
// dump_cdf (or nullptr): row i * dump_steps + pos of [.][257] receives the table (test-only).
template <int MODE>
__global__ void __launch_bounds__(256)
k_fx_coder_step(const int32_t* __restrict__ logits, uint8_t* data, size_t chunk_bytes, CoderArrays ca, int B, Tables tb,
                uint32_t* dump_cdf, uint32_t dump_steps) {
  const int i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
  const int lane = threadIdx.x & 31;
  if (i >= B) return;
  const uint32_t pos = ca.pos[i], len = ca.len[i];
  if (pos + 1u >= len) return;                    // finished stream: masked
  int32_t l[8];
  {
    const int4* lp = reinterpret_cast<const int4*>(logits + (size_t)i * 256 + lane * 8);
    const int4 a = lp[0], b = lp[1];
    l[0] = a.x; l[1] = a.y; l[2] = a.z; l[3] = a.w; l[4] = b.x; l[5] = b.y; l[6] = b.z; l[7] = b.w;
  }
  WarpTable t;
  build_table_fx(tb, l, t);
  if (dump_cdf) {
    const size_t row = (size_t)i * dump_steps + pos;
    uint32_t run = t.gex;
#pragma unroll
    for (int k = 0; k < 8; ++k) {
      dump_cdf[row * 257 + 8u * lane + k] = cdf_value(8u * lane + k, run, t.T);
      run += t.g[k];
    }
    if (lane == 31) dump_cdf[row * 257 + 256] = kM;
  }
  uint8_t* sdata = data + (size_t)i * chunk_bytes;
  if (MODE == 0) {
    const uint32_t s = sdata[pos + 1u];
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

}  // namespace fx
}  // namespace boa
