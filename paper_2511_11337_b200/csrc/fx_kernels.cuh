// fx_kernels.cuh — FX1, the deterministic fixed-point pipeline (PAPER "Portability").
//
// The specification is DESIGN.md section 11 (reading R#24): every value an integer, every operation +, -, *, shift,
// comparison, integer division or integer square root with stated widths, every rounding "nearest, ties to even", every
// store saturating - so the tables, and therefore the container bytes, do not depend on the device or on any order of
// summation.  This file is that specification as CUDA device code; it shares nothing with oracle/fixed.py, which states
// it in Python integers and which the GPU tests compare with bit for bit (logits, tables, whole containers).
//
//   Q    int32, 20 fraction bits          U30  exp / sigmoid values in [0, 2^30]
//   int8 rows: a row of Q values is cut to q in [-127, 127] with one shift k (a ~ q 2^(k-20)); weight rows are stored as
//   q in [-127, 127] with an exponent s (w ~ q 2^-s); a contraction is an exact int32 dot product (dp4a) followed by
//   sat(rne(acc, s - k)).
#pragma once
#include "common.cuh"

namespace boa {
namespace fx {

constexpr int F = 20;
constexpr int64_t QMAX = 2147483647ll, QMIN = -2147483648ll;
constexpr int64_t U30 = 1ll << 30;
constexpr int64_t LOG2E_Q30 = 1549082005ll;
constexpr int64_t EPS_Q40 = 10995116ll;
constexpr int TB = 8, NTAB = 1 << TB;                   // 256 intervals, 257 entries per table
constexpr uint32_t TABLE_CRC = 0x6B76FB0Du;             // CRC-32 of both tables as little-endian int64 (part of the specification)

// round-half-even(v / 2^k); k <= 0: exact left shift
__device__ __forceinline__ int64_t rne(int64_t v, int k) {
  if (k <= 0) return v << (-k);
  const int64_t q = v >> k, r = v & ((1ll << k) - 1), half = 1ll << (k - 1);
  return q + ((r > half || (r == half && (q & 1))) ? 1 : 0);
}
__device__ __forceinline__ int64_t sat(int64_t v) { return v > QMAX ? QMAX : (v < QMIN ? QMIN : v); }
__device__ __forceinline__ int64_t qmul(int64_t a, int64_t b) { return sat(rne(a * b, F)); }
// round-half-even(n / d), d > 0
__device__ __forceinline__ int64_t rdiv(int64_t n, int64_t d) {
  int64_t q = n / d, r = n - q * d;
  if (r < 0) { r += d; q -= 1; }                        // floor division
  return q + ((2 * r > d || (2 * r == d && (q & 1))) ? 1 : 0);
}
__device__ __forceinline__ int64_t isqrt64(int64_t x) {  // floor(sqrt(x)) exactly, 0 <= x < 2^62
  int64_t y = (int64_t)floor(sqrt((double)x));
  if (y * y > x) --y;
  if ((y + 1) * (y + 1) <= x) ++y;
  return y;
}
__device__ __forceinline__ int bitlen64(int64_t m) { return 64 - __clzll((long long)m); }   // m >= 0

struct Tables {
  const int32_t* exp2;     // [257]  rne(2^30 2^(-i/256))
  const int32_t* log1p;    // [257]  rne(2^30 ln(1 + i/256))
};

__device__ __forceinline__ int64_t interp(const int32_t* tab, int64_t x, int frac_bits) {
  const int lo = frac_bits - TB;
  int64_t i = x >> lo, r = x & ((1ll << lo) - 1);
  if (i >= NTAB) { i = NTAB; r = 0; }
  const int64_t a = tab[i], b = tab[i + 1 > NTAB ? NTAB : i + 1];
  return a + rne((b - a) * r, lo);
}
__device__ __forceinline__ int64_t exp2_neg(const Tables& t, int64_t x) {   // x >= 0 in Q -> 2^-x in U30
  const int64_t n = x >> F, f = x & ((1ll << F) - 1);
  if (n >= 31) return 0;
  return rne(interp(t.exp2, f, F), (int)n);
}
__device__ __forceinline__ int64_t exp_neg(const Tables& t, int64_t x) { return exp2_neg(t, sat(rne(x * LOG2E_Q30, 30))); }
__device__ __forceinline__ int64_t sigmoid(const Tables& t, int64_t x) {
  const int64_t s = rdiv(1ll << 60, U30 + exp_neg(t, x < 0 ? -x : x));
  return x >= 0 ? s : U30 - s;
}
__device__ __forceinline__ int64_t silu(const Tables& t, int64_t x) { return sat(rne(x * sigmoid(t, x), 30)); }
__device__ __forceinline__ int64_t softplus(const Tables& t, int64_t v) {
  const int64_t l30 = interp(t.log1p, exp_neg(t, v < 0 ? -v : v), 30);
  return sat((v > 0 ? v : 0) + rne(l30, 30 - F));
}

// block-wide max of a non-negative int64 (blockDim.x a multiple of 32, <= 1024); every thread gets the result
__device__ __forceinline__ int64_t block_max(int64_t v, int64_t* red) {
  for (int o = 16; o > 0; o >>= 1) { const int64_t w = __shfl_xor_sync(0xffffffffu, v, o); v = w > v ? w : v; }
  const int warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[warp] = v;
  __syncthreads();
  int64_t m = 0;
  for (int k = 0; k < nw; ++k) m = red[k] > m ? red[k] : m;
  return m;
}
__device__ __forceinline__ int64_t block_sum(int64_t v, int64_t* red) {   // integers: order-free
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  const int warp = threadIdx.x >> 5, nw = blockDim.x >> 5;
  __syncthreads();
  if ((threadIdx.x & 31) == 0) red[warp] = v;
  __syncthreads();
  int64_t s = 0;
  for (int k = 0; k < nw; ++k) s += red[k];
  return s;
}

// ---- S1: u = Emb[previous byte], Q.  One thread per (stream, column).
__global__ void k_fx_embed(const uint8_t* __restrict__ data, size_t chunk_bytes, const uint32_t* __restrict__ pos,
                           const uint32_t* __restrict__ len, const int8_t* __restrict__ qemb, const int32_t* __restrict__ semb,
                           int32_t* __restrict__ u, int B, int D) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= B * D) return;
  const int i = idx / D, d = idx - i * D;
  const uint32_t p = min(pos[i], len[i] - 1u);
  const int b = data[(size_t)i * chunk_bytes + p];
  u[idx] = (int32_t)sat(rne((int64_t)qemb[b * D + d], semb[b] - F));
}

// ---- S2: r = RMSNorm(u) * w in Q (integer only).  One block per row.
__global__ void k_fx_rmsnorm(const int32_t* __restrict__ u, const int32_t* __restrict__ w, int32_t* __restrict__ r, int D,
                             int64_t sqrt_d) {
  __shared__ int64_t red[32];
  const int row = blockIdx.x;
  const int32_t* ur = u + (size_t)row * D;
  int64_t m = 0;
  for (int d = threadIdx.x; d < D; d += blockDim.x) { const int64_t a = ur[d]; m = max(m, a < 0 ? -a : a); }
  m = block_max(m, red);
  if (m == 0) {
    for (int d = threadIdx.x; d < D; d += blockDim.x) r[(size_t)row * D + d] = 0;
    return;
  }
  const int c = min(24 - bitlen64(m), 12);
  int64_t s = 0;
  for (int d = threadIdx.x; d < D; d += blockDim.x) { const int64_t t = rne((int64_t)ur[d], -c); s += t * t; }
  s = block_sum(s, red);
  const int64_t Y = isqrt64(s + (int64_t)D * rne(EPS_Q40, -2 * c));
  for (int d = threadIdx.x; d < D; d += blockDim.x) {
    const int64_t t = rne((int64_t)ur[d], -c);
    r[(size_t)row * D + d] = (int32_t)qmul(rdiv(t * sqrt_d, Y), w[d]);
  }
}

// ---- a row of Q values -> int8 with one shift per row: k = max(0, bitlen(max|a|) - 7), q = clip(rne(a, k), +-127).
// One block per row.  K % 4 == 0; the int8 row is padded with zeros to ldq (a multiple of 16).
__global__ void k_fx_quant_rows(const int32_t* __restrict__ a, int lda, int K, int8_t* __restrict__ q, int ldq,
                                int32_t* __restrict__ kshift) {
  __shared__ int64_t red[32];
  const int row = blockIdx.x;
  const int32_t* ar = a + (size_t)row * lda;
  int64_t m = 0;
  for (int d = threadIdx.x; d < K; d += blockDim.x) { const int64_t v = ar[d]; m = max(m, v < 0 ? -v : v); }
  m = block_max(m, red);
  const int k = max(bitlen64(m) - 7, 0);
  for (int d = threadIdx.x; d < ldq; d += blockDim.x) {
    int64_t v = d < K ? rne((int64_t)ar[d], k) : 0;
    v = v > 127 ? 127 : (v < -127 ? -127 : v);
    q[(size_t)row * ldq + d] = (int8_t)v;
  }
  if (threadIdx.x == 0) kshift[row] = k;
}

// ---- contraction: out[m][n] = sat(rne(sum_k qa[m][k] qw[n][k], s[n] - ka[m])) (+ resid[m][n], saturating).
// 64 x 64 output tile per block of 256 threads (4 x 4 outputs per thread), 64-byte k-slabs through shared memory, dp4a.
// Integer sums: the tile shape has no influence on the result.
constexpr int GT = 64;
__global__ void __launch_bounds__(256) k_fx_gemm(const int8_t* __restrict__ qa, int lda, const int32_t* __restrict__ ka,
                                                 const int8_t* __restrict__ qw, int ldw, const int32_t* __restrict__ sw,
                                                 int32_t* __restrict__ out, int ldo, const int32_t* __restrict__ resid,
                                                 int M, int N, int K) {
  __shared__ __align__(16) int32_t As[GT][17], Ws[GT][17];      // 64 rows x 64 bytes (16 words) + pad
  const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
  const int m0 = blockIdx.y * GT, n0 = blockIdx.x * GT;
  int acc[4][4] = {};
  for (int k0 = 0; k0 < K; k0 += 64) {
    for (int e = threadIdx.x; e < GT * 16; e += 256) {
      const int r = e >> 4, cw = e & 15;
      const int kk = k0 + cw * 4;
      int32_t va = 0, vw = 0;
      if (m0 + r < M && kk < K) va = *reinterpret_cast<const int32_t*>(qa + (size_t)(m0 + r) * lda + kk);
      if (n0 + r < N && kk < K) vw = *reinterpret_cast<const int32_t*>(qw + (size_t)(n0 + r) * ldw + kk);
      As[r][cw] = va; Ws[r][cw] = vw;
    }
    __syncthreads();
#pragma unroll
    for (int cw = 0; cw < 16; ++cw) {
      int a[4], w[4];
#pragma unroll
      for (int i = 0; i < 4; ++i) { a[i] = As[ty * 4 + i][cw]; w[i] = Ws[tx * 4 + i][cw]; }
#pragma unroll
      for (int i = 0; i < 4; ++i)
#pragma unroll
        for (int j = 0; j < 4; ++j) acc[i][j] = __dp4a(a[i], w[j], acc[i][j]);
    }
    __syncthreads();
  }
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const int m = m0 + ty * 4 + i;
    if (m >= M) continue;
    const int km = ka[m];
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int n = n0 + tx * 4 + j;
      if (n >= N) continue;
      int64_t v = sat(rne((int64_t)acc[i][j], max(sw[n] - km, -31)));
      if (resid) v = sat(v + (int64_t)resid[(size_t)m * ldo + n]);
      out[(size_t)m * ldo + n] = (int32_t)v;
    }
  }
}

// ---- S4: causal depthwise conv over the window (x_{t-3}, x_{t-2}, x_{t-1}) and x_t, SiLU; the window shifts.
// xz [B][2E] Q (x | z);  win [B][3][E];  xs [B][E].  One thread per (stream, channel).
__global__ void k_fx_conv_silu(const int32_t* __restrict__ xz, int32_t* __restrict__ win, const int32_t* __restrict__ conv_w,
                               const int32_t* __restrict__ conv_b, int32_t* __restrict__ xs, Tables t, int B, int E) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= B * E) return;
  const int i = idx / E, e = idx - i * E;
  const int64_t x = xz[(size_t)i * 2 * E + e];
  int32_t* w = win + (size_t)i * 3 * E + e;
  const int64_t w0 = w[0], w1 = w[E], w2 = w[2 * E];
  const int32_t* cw = conv_w + (size_t)e * 4;
  const int64_t acc = (int64_t)conv_b[e] + rne((int64_t)cw[3] * x, F) + rne((int64_t)cw[0] * w0, F) + rne((int64_t)cw[1] * w1, F) +
                      rne((int64_t)cw[2] * w2, F);
  w[0] = (int32_t)w1; w[E] = (int32_t)w2; w[2 * E] = (int32_t)x;
  xs[idx] = (int32_t)silu(t, sat(acc));
}

// ---- S6-S8: dt_proj (int8 rows, K = R) + softplus, the recurrence on the 16 state values, D skip, gate.
// dbc [B][ldj] Q = delta[R] | B[16] | C[16];  h [B][E][16] Q;  y [B][E] Q.  One thread per (stream, channel).
__global__ void k_fx_scan(const int32_t* __restrict__ dbc, int ldj, const int8_t* __restrict__ qwdt, const int32_t* __restrict__ swdt,
                          const int32_t* __restrict__ b_dt, const int32_t* __restrict__ a_neg, const int32_t* __restrict__ d_skip,
                          const int32_t* __restrict__ xs, const int32_t* __restrict__ xz, int32_t* __restrict__ h,
                          int32_t* __restrict__ y, Tables t, int B, int E, int R) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= B * E) return;
  const int i = idx / E, e = idx - i * E;
  const int32_t* row = dbc + (size_t)i * ldj;
  // delta's row cut to int8 (every thread of the stream computes the same k and q)
  int64_t m = 0;
  for (int r = 0; r < R; ++r) { const int64_t v = row[r]; m = max(m, v < 0 ? -v : v); }
  const int k = max(bitlen64(m) - 7, 0);
  int acc = 0;
  for (int r = 0; r < R; ++r) {
    int64_t q = rne((int64_t)row[r], k);
    q = q > 127 ? 127 : (q < -127 ? -127 : q);
    acc += (int)q * (int)qwdt[(size_t)e * R + r];
  }
  const int64_t v = sat(rne((int64_t)acc, max(swdt[e] - k, -31)));
  const int64_t dl = softplus(t, sat(v + (int64_t)b_dt[e]));
  const int64_t x = xs[idx], z = xz[(size_t)i * 2 * E + E + e];
  int32_t* hp = h + (size_t)idx * kNState;
  int64_t ya = 0;
#pragma unroll 4
  for (int n = 0; n < kNState; ++n) {
    const int64_t dA = exp_neg(t, qmul(dl, a_neg[(size_t)e * kNState + n]));
    const int64_t hv = sat(rne(dA * (int64_t)hp[n], 30) + qmul(qmul(dl, row[R + n]), x));
    hp[n] = (int32_t)hv;
    ya += rne((int64_t)row[R + kNState + n] * hv, F);
  }
  const int64_t yv = sat(ya + rne((int64_t)d_skip[e] * x, F));
  y[idx] = (int32_t)qmul(yv, silu(t, z));
}

}  // namespace fx
}  // namespace boa
