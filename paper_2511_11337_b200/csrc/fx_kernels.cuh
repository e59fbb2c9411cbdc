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
//   q in [-127, 127] with an exponent s (w ~ q 2^-s); a contraction is an exact int32 dot product (tcgen05.mma kind::i8,
//   fx_gemm_tc.cuh) followed by sat(rne(acc, s - k)).
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
// (the remainder plus half - 1 plus the quotient's low bit carries into bit k exactly when the value rounds up)
__device__ __forceinline__ int64_t rne(int64_t v, int k) {
  if (k <= 0) return v << (-k);
  return (v + ((1ll << (k - 1)) - 1) + ((v >> k) & 1)) >> k;
}
__device__ __forceinline__ int64_t sat(int64_t v) { return v > QMAX ? QMAX : (v < QMIN ? QMIN : v); }
__device__ __forceinline__ int64_t qmul(int64_t a, int64_t b) { return sat(rne(a * b, F)); }
// round-half-even(n / d), d > 0, |n| < 2^62.  The quotient is estimated in double precision and then corrected with
// the exact remainder until 0 <= r < d, and the rounding is decided on that exact remainder: the result is the integer
// the definition names whatever the quality of the estimate (which only decides how many correction steps run: none or
// one with the reciprocal below), without the 64-bit division subroutine.
// rcp ~ 1 / d, passed in so that a row with one divisor computes it once.
__device__ __forceinline__ double rcp_est(int64_t d) {        // two Newton steps on the hardware's approximation
  const double dd = __ll2double_rn(d);
  double x;
  asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(x) : "d"(dd));
  x = fma(fma(-dd, x, 1.0), x, x);
  x = fma(fma(-dd, x, 1.0), x, x);
  return x;
}
__device__ __forceinline__ int64_t rdiv_rcp(int64_t n, int64_t d, double rcp) {
  const int64_t a = n < 0 ? -n : n;
  int64_t q = __double2ll_rz(__ll2double_rz(a) * rcp);
  int64_t r = a - q * d;
  while (r < 0) { q -= 1; r += d; }
  while (r >= d) { q += 1; r -= d; }
  q += (2 * r > d || (2 * r == d && (q & 1))) ? 1 : 0;      // ties to even (symmetric in the sign of n)
  return n < 0 ? -q : q;
}
__device__ __forceinline__ int64_t rdiv(int64_t n, int64_t d) { return rdiv_rcp(n, d, rcp_est(d)); }
__device__ __forceinline__ int64_t isqrt64(int64_t x) {  // floor(sqrt(x)) exactly, 0 <= x < 2^62
  int64_t y = (int64_t)floor(sqrt((double)x));
  if (y * y > x) --y;
  if ((y + 1) * (y + 1) <= x) ++y;
  return y;
}
__device__ __forceinline__ int bitlen64(int64_t m) { return 64 - __clzll((long long)m); }   // m >= 0

// ---- operand images of the tensor-core contractions (fx_gemm_tc.cuh)
constexpr int TBM = 128, TBN = 64, TBK = 128;         // tile rows, tile columns, int8 k per block
constexpr int A_BLK = TBM * TBK, W_BLK = TBN * TBK;   // bytes of one k-block of a row tile / of a column tile
constexpr int TC_MAXST = 8;                           // k-blocks in flight

// Byte offset of element (r, k) inside one k-block of a tile: rows of 128 bytes, the 16-byte chunk index XORed with the
// row index mod 8 (128-byte swizzle), 8-row groups 1024 bytes apart.
__host__ __device__ inline uint32_t blk_off8(int r, int k) {
  return (uint32_t)((r >> 3) * 1024 + (r & 7) * 128 + ((((k >> 4) ^ r) & 7) << 4) + (k & 15));
}
// activation image of A[M][K]: [ceil(M/128)][KB][128 x 128 bytes]
__host__ __device__ inline size_t a_img_off(int m, int k, int KB) {
  return ((size_t)(m >> 7) * KB + (size_t)(k >> 7)) * A_BLK + blk_off8(m & 127, k & 127);
}
__host__ __device__ inline size_t a_img_bytes(size_t M, size_t KB) { return (M + TBM - 1) / TBM * KB * A_BLK; }
// weight image of W[N][K]: [ceil(N/64)][KB][64 x 128 bytes], rows and columns beyond N, K zero
__host__ __device__ inline size_t w_img_off(int n, int k, int KB) {
  return ((size_t)(n >> 6) * KB + (size_t)(k >> 7)) * W_BLK + blk_off8(n & 63, k & 127);
}

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

// int8 cut of one value with the row's shift k
__device__ __forceinline__ int8_t cut8(int32_t a, int k) {
  int64_t v = rne((int64_t)a, k);
  v = v > 127 ? 127 : (v < -127 ? -127 : v);
  return (int8_t)v;
}
__device__ __forceinline__ int64_t abs64(int64_t a) { return a < 0 ? -a : a; }

__device__ __forceinline__ int64_t warp_max64(int64_t v) {
  for (int o = 16; o > 0; o >>= 1) { const int64_t w = __shfl_xor_sync(0xffffffffu, v, o); v = w > v ? w : v; }
  return v;
}
__device__ __forceinline__ int64_t warp_sum64(int64_t v) {                 // integers: order-free
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

// ---- S2: r = RMSNorm(u) * w in Q (integer only), cut to an int8 row for in_proj in the same
// kernel (the Q values of r have no other reader).  One warp per row (shuffle reductions, no block barrier), eight rows
// per block; r waits in shared memory for the row's shift.  D <= 1024.
// EMBED (the first layer of a step): the row is first written as u = Emb[previous byte] (S1) by the same warp.
struct EmbedSrc {
  const uint8_t* data; size_t chunk_bytes; const uint32_t *pos, *len; const int8_t* qemb; const int32_t* semb;
};
constexpr int RMS_ROWS = 8;
template <bool EMBED>
__global__ void __launch_bounds__(32 * RMS_ROWS) k_fx_rmsnorm_q(int32_t* __restrict__ u, const int32_t* __restrict__ w, int D,
                                                                int64_t sqrt_d, int8_t* __restrict__ q, int KB,
                                                                int32_t* __restrict__ kshift, int B, EmbedSrc es) {
  __shared__ int32_t s_r[RMS_ROWS][1024];
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * RMS_ROWS + warp;
  if (row >= B) return;
  int32_t* ur = u + (size_t)row * D;
  if (EMBED) {
    const uint32_t p = min(es.pos[row], es.len[row] - 1u);
    const int b = es.data[(size_t)row * es.chunk_bytes + p];
    const int sh = es.semb[b] - F;
    for (int d = lane; d < D; d += 32) ur[d] = (int32_t)sat(rne((int64_t)es.qemb[b * D + d], sh));
    __syncwarp();                                   // (each lane re-reads only what it wrote; the barrier is for clarity)
  }
  int32_t* rr = s_r[warp];
  int64_t m = 0;
  for (int d = lane; d < D; d += 32) m = max(m, abs64(ur[d]));
  m = warp_max64(m);
  int64_t rm = 0;
  if (m != 0) {
    const int c = min(24 - bitlen64(m), 12);
    int64_t s = 0;
    for (int d = lane; d < D; d += 32) { const int64_t t = rne((int64_t)ur[d], -c); s += t * t; }
    s = warp_sum64(s);
    const int64_t Y = isqrt64(s + (int64_t)D * rne(EPS_Q40, -2 * c));
    const double rcp_y = rcp_est(Y);
#pragma unroll 2
    for (int d = lane; d < D; d += 32) {
      const int32_t r = (int32_t)qmul(rdiv_rcp(rne((int64_t)ur[d], -c) * sqrt_d, Y, rcp_y), w[d]);
      rr[d] = r;
      rm = max(rm, abs64(r));
    }
    rm = warp_max64(rm);
  }
  const int k = max(bitlen64(rm) - 7, 0);
  for (int d = lane; d < D; d += 32) q[a_img_off(row, d, KB)] = m != 0 ? cut8(rr[d], k) : (int8_t)0;
  if (lane == 0) kshift[row] = k;
}

// ---- a row of Q values -> int8 with one shift per row: k = max(0, bitlen(max|a|) - 7), q = clip(rne(a, k), +-127).
// One warp per row; the int8 row goes into the activation image (KB k-blocks per row tile).
__global__ void __launch_bounds__(32 * RMS_ROWS) k_fx_quant_rows(const int32_t* __restrict__ a, int lda, int K, int8_t* __restrict__ q,
                                                                 int KB, int32_t* __restrict__ kshift, int B) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const int row = blockIdx.x * RMS_ROWS + warp;
  if (row >= B) return;
  const int32_t* ar = a + (size_t)row * lda;
  int64_t m = 0;
  for (int d = lane; d < K; d += 32) m = max(m, abs64(ar[d]));
  m = warp_max64(m);
  const int k = max(bitlen64(m) - 7, 0);
  for (int d = lane; d < K; d += 32) q[a_img_off(row, d, KB)] = cut8(ar[d], k);
  if (lane == 0) kshift[row] = k;
}

// ---- 32-bit forms.  The integer ALU pipe is what bounds the scan, so the roundings are written on 32-bit halves: the rounding constant
// rides on the multiply (mad.wide), "ties to even" is "add half, shift, clear the low bit if the shifted-out bits are
// all zero", and a saturation test is a range test of the high word.  Same integers as rne / sat / qmul above.
// (the rounding constants live in constant memory, so that they are the multiply-add's addend operand instead of an
// immediate the compiler adds with a separate 64-bit addition on the bounding pipe)
__constant__ int64_t c_half[3] = {1ll << (F - TB - 1), 1ll << (F - 1), 1ll << 29};
#define FX_HALF12 c_half[0]
#define FX_HALF20 c_half[1]
#define FX_HALF30 c_half[2]
__device__ __forceinline__ int64_t madw(int32_t a, int32_t b, int64_t c) {
  int64_t r;
  asm("mad.wide.s32 %0, %1, %2, %3;" : "=l"(r) : "r"(a), "r"(b), "l"(c));
  return r;
}
__device__ __forceinline__ uint32_t lo32(int64_t v) { return (uint32_t)v; }
__device__ __forceinline__ int32_t hi32(int64_t v) { return (int32_t)(v >> 32); }
__device__ __forceinline__ int32_t add_sat32(int32_t a, int32_t b) {
  int32_t r;
  asm("add.sat.s32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
// low 32 bits of rne(p, K), given p2 = p + 2^(K-1), 1 <= K <= 31
template <int K>
__device__ __forceinline__ uint32_t rne_lo32(int64_t p2) {
  uint32_t q = __funnelshift_r(lo32(p2), (uint32_t)hi32(p2), K);
  if ((lo32(p2) & ((1u << K) - 1u)) == 0u) q &= ~1u;
  return q;
}
// sat(rne(a b, 20));  SAT = false: the caller has shown that the quotient fits 32 bits
template <bool SAT = true>
__device__ __forceinline__ int32_t qmul32(int32_t a, int32_t b) {
  const int64_t p2 = madw(a, b, FX_HALF20);
  uint32_t q = rne_lo32<F>(p2);
  if (SAT) {
    const int32_t h = hi32(p2);                     // the quotient fits 32 bits iff -2^19 <= h < 2^19
    if ((uint32_t)(h + (1 << (F - 1))) >= (1u << F)) q = 0x7FFFFFFFu ^ (uint32_t)(h >> 31);
  }
  return (int32_t)q;
}
// qmul(a, b) for a, b >= 0 as the argument of exp_neg: any value >= 2^25 (32.0) stands for "exp_neg = 0"
// (n >= 46 there), so the saturation is one comparison of the high word (2^13 <-> quotient 2^25)
__device__ __forceinline__ int32_t qmul32_exparg(int32_t a, int32_t b) {
  const int64_t p2 = madw(a, b, FX_HALF20);
  const uint32_t q = rne_lo32<F>(p2);
  return hi32(p2) >= (1 << 13) ? (1 << 26) : (int32_t)q;
}
// exp_neg for 0 <= x <= QMAX from the table (value, difference to the next entry) in shared memory: the same integers
// as fx::exp_neg (n >= 31 rounds to 0 through the shift; val <= 2^30 so the last rounding is 32-bit)
__device__ __forceinline__ int32_t exp_neg_s(const int2* tab, int32_t x) {
  const uint32_t tq = rne_lo32<30>(madw(x, (int32_t)LOG2E_Q30, FX_HALF30));     // < 2^32
  const uint32_t n = min(tq >> F, 31u);
  const int2 e = tab[(tq >> (F - TB)) & (NTAB - 1)];
  const uint32_t val = (uint32_t)e.x + rne_lo32<F - TB>(madw(e.y, (int32_t)(tq & ((1u << (F - TB)) - 1u)), FX_HALF12));
  const uint32_t v2 = val + ((1u << n) >> 1);
  uint32_t q = v2 >> n;
  if ((v2 & ((1u << n) - 1u)) == 0u) q &= ~1u;
  return (int32_t)(n ? q : val);
}
// the table of exp2_neg as (value, difference to the next entry) pairs in shared memory; blockDim.x >= 256
__device__ __forceinline__ void load_exp_table(int2* s_tab, const Tables& t) {
  if (threadIdx.x < NTAB) {
    const int32_t a = t.exp2[threadIdx.x];
    s_tab[threadIdx.x] = make_int2(a, t.exp2[threadIdx.x + 1] - a);
  }
}
// sigmoid, SiLU, softplus on the shared table: the same integers as fx::sigmoid / silu / softplus (|x| = 2^31 is cut to
// QMAX: exp_neg is 0 for both)
__device__ __forceinline__ int64_t sigmoid_s(const int2* tab, int32_t x) {
  const uint32_t ax = min(x < 0 ? -(uint32_t)x : (uint32_t)x, (uint32_t)QMAX);
  const int64_t s = rdiv(1ll << 60, U30 + (int64_t)exp_neg_s(tab, (int32_t)ax));
  return x >= 0 ? s : U30 - s;
}
__device__ __forceinline__ int64_t silu_s(const int2* tab, int32_t x) { return sat(rne((int64_t)x * sigmoid_s(tab, x), 30)); }
__device__ __forceinline__ int64_t softplus_s(const int2* tab, const Tables& t, int32_t v) {
  const uint32_t av = min(v < 0 ? -(uint32_t)v : (uint32_t)v, (uint32_t)QMAX);
  const int64_t l30 = interp(t.log1p, (int64_t)exp_neg_s(tab, (int32_t)av), 30);
  return sat((int64_t)(v > 0 ? v : 0) + rne(l30, 30 - F));
}

// ---- S4: causal depthwise conv over the window (x_{t-3}, x_{t-2}, x_{t-1}) and x_t, SiLU; the window shifts.
// xz [B][2E] Q (x | z);  win [B][3][E];  xs [B][E] Q (read by the scan) and its int8 cut (q, kshift) for x_proj.
// One block of 256 threads per stream, E <= 2048 (<= 8 channels per thread).
__global__ void __launch_bounds__(256) k_fx_conv_silu_q(const int32_t* __restrict__ xz, int32_t* __restrict__ win,
                                                        const int32_t* __restrict__ conv_w, const int32_t* __restrict__ conv_b,
                                                        int32_t* __restrict__ xs, Tables t, int E, int8_t* __restrict__ q, int KB,
                                                        int32_t* __restrict__ kshift) {
  __shared__ int64_t red[32];
  __shared__ int2 s_tab[NTAB];
  load_exp_table(s_tab, t);
  __syncthreads();
  const int i = blockIdx.x;
  int32_t v[8];
  int64_t m = 0;
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const int e = threadIdx.x + 256 * it;
    v[it] = 0;
    if (e < E) {
      const int64_t x = xz[(size_t)i * 2 * E + e];
      int32_t* w = win + (size_t)i * 3 * E + e;
      const int64_t w0 = w[0], w1 = w[E], w2 = w[2 * E];
      const int4 cw = *reinterpret_cast<const int4*>(conv_w + (size_t)e * 4);
      const int64_t acc = (int64_t)conv_b[e] + rne((int64_t)cw.w * x, F) + rne((int64_t)cw.x * w0, F) + rne((int64_t)cw.y * w1, F) +
                          rne((int64_t)cw.z * w2, F);
      w[0] = (int32_t)w1; w[E] = (int32_t)w2; w[2 * E] = (int32_t)x;
      v[it] = (int32_t)silu_s(s_tab, (int32_t)sat(acc));
      xs[(size_t)i * E + e] = v[it];
      m = max(m, abs64(v[it]));
    }
  }
  m = block_max(m, red);
  const int k = max(bitlen64(m) - 7, 0);
#pragma unroll
  for (int it = 0; it < 8; ++it) {
    const int e = threadIdx.x + 256 * it;
    if (e < E) q[a_img_off(i, e, KB)] = cut8(v[it], k);
  }
  if (threadIdx.x == 0) kshift[i] = k;
}

// ---- S6-S8: dt_proj (int8 rows, K = R) + softplus, the recurrence on the 16 state values, D skip, gate; y is cut to an
// int8 row for out_proj in the same kernel (its Q values have no other reader).
// dbc [B][ldj] Q = delta[R] | B[16] | C[16];  h [B][E][16] Q.  One block of 256 threads per stream; a warp takes 32
// channels at a time.  Per-channel values (dt, x, z, the gate) belong to lane = channel; the 2 KB of state of the 32
// channels are read as four fully coalesced 512-byte rows, lane l holding states 4 (l % 4) .. + 3 of channel
// 8 j + l / 4 in row j, so a channel's sum over n is an (order-free, integer) sum over four lanes.
// The recurrence of one state value, every product 32 x 32 -> 64 bits:
//   dA = exp_neg(qmul(dt, |A|));  h = sat(rne(dA h, 30) + qmul(qmul(dt, B_n), x));  y += rne(C_n h, 20)
template <bool SAT>
__device__ __forceinline__ void scan_state(const int2* tab, int32_t dl, int32_t x, int32_t a, int32_t b, int32_t c, int32_t& h,
                                           uint32_t& ya_lo, int32_t& ya_hi) {
  const int32_t dA = exp_neg_s(tab, qmul32_exparg(dl, a));
  h = add_sat32((int32_t)rne_lo32<30>(madw(dA, h, FX_HALF30)), qmul32<SAT>(qmul32<SAT>(dl, b), x));
  // ya += rne(c h, 20): the 64-bit sum kept as two words, the low word's carry through a wide multiply-add
  const int64_t p2 = madw(c, h, FX_HALF20);
  const uint32_t ql = rne_lo32<F>(p2);
  const int32_t qh = hi32(p2) >> F;
  uint64_t s;
  asm("mad.wide.u32 %0, %1, 1, %2;" : "=l"(s) : "r"(ql), "l"((uint64_t)ya_lo));
  ya_lo = (uint32_t)s;
  ya_hi += qh + (int32_t)(s >> 32);
}

__global__ void __launch_bounds__(256, 4) k_fx_scan_q(const int32_t* __restrict__ dbc, int ldj, const int8_t* __restrict__ qwdt,
                                                   const int32_t* __restrict__ swdt, const int32_t* __restrict__ b_dt,
                                                   const int32_t* __restrict__ a_neg, const int32_t* __restrict__ d_skip,
                                                   const int32_t* __restrict__ xs, const int32_t* __restrict__ xz, int32_t* __restrict__ h,
                                                   Tables t, int E, int R, int8_t* __restrict__ q, int KB,
                                                   int32_t* __restrict__ kshift) {
  __shared__ int2 s_tab[NTAB];
  __shared__ __align__(16) int32_t s_bc[2 * kNState];
  __shared__ __align__(16) int8_t s_q[64];
  __shared__ int s_k;
  __shared__ int64_t red[32];
  __shared__ int32_t s_y[2048];                     // E <= 2048
  const int i = blockIdx.x, tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int32_t* row = dbc + (size_t)i * ldj;
  load_exp_table(s_tab, t);
  if (tid < 2 * kNState) s_bc[tid] = row[R + tid];
  if (warp == 1) {                                  // delta's row cut to int8 (R <= 64)
    const int32_t v0 = lane < R ? row[lane] : 0, v1 = lane + 32 < R ? row[lane + 32] : 0;
    int64_t m = max(abs64(v0), abs64(v1));
    for (int o = 16; o > 0; o >>= 1) { const int64_t w = __shfl_xor_sync(0xffffffffu, m, o); m = w > m ? w : m; }
    const int k = max(bitlen64(m) - 7, 0);
    s_q[lane] = cut8(v0, k);
    s_q[lane + 32] = cut8(v1, k);
    if (lane == 0) s_k = k;
  }
  __syncthreads();
  const int kd = s_k;
  int bB = 0;                                       // bit length of max_n |B_n|
#pragma unroll
  for (int n = 0; n < kNState; ++n) bB = max(bB, bitlen64(abs64(s_bc[n])));
  int64_t ym = 0;
#pragma unroll 1
  for (int cg = warp; cg * 32 < E; cg += 8) {       // channel group: warp-uniform
    {
      const int e = cg * 32 + lane;
      int acc = 0;
      if ((R & 3) == 0) {
        const int* wq = reinterpret_cast<const int*>(qwdt + (size_t)e * R);
        const int* sq = reinterpret_cast<const int*>(s_q);
        for (int r = 0; r < (R >> 2); ++r) acc = __dp4a(sq[r], wq[r], acc);
      } else {
        for (int r = 0; r < R; ++r) acc += (int)s_q[r] * (int)qwdt[(size_t)e * R + r];
      }
      const int64_t dv = sat(rne((int64_t)acc, max(swdt[e] - kd, -31)));
      const int32_t dl = (int32_t)softplus_s(s_tab, t, (int32_t)sat(dv + (int64_t)b_dt[e]));
      const int32_t x = xs[(size_t)i * E + e];
      const int32_t z = xz[(size_t)i * 2 * E + E + e];
      int4* hp = reinterpret_cast<int4*>(h + ((size_t)i * E + (size_t)cg * 32) * kNState) + lane;
      const int4* ap = reinterpret_cast<const int4*>(a_neg + (size_t)cg * 32 * kNState) + lane;
      const int4 b4 = reinterpret_cast<const int4*>(s_bc)[lane & 3], c4 = reinterpret_cast<const int4*>(s_bc)[4 + (lane & 3)];
      int4 hv[4];
#pragma unroll
      for (int j = 0; j < 4; ++j) hv[j] = __ldcs(hp + 32 * j);
      int64_t ya_own = 0;
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        const int src = 8 * j + (lane >> 2);
        const int32_t dlj = __shfl_sync(0xffffffffu, dl, src), xj = __shfl_sync(0xffffffffu, x, src);
        const int4 a4 = __ldg(ap + 32 * j);
        uint32_t ya_lo = 0;
        int32_t ya_hi = 0;
        // |dt B_n| 2^-20 <= 2^(bd + bB - 20) and |(dt B_n) x| 2^-40 <= 2^(bd + bB + bx - 39) with bd, bB, bx the bit
        // lengths of dt, max_n |B_n|, |x|: when both stay below 2^31 for every lane the two products cannot saturate
        // and the warp takes the instantiation without the range tests (the same integers either way)
        const int bd = 32 - __clz(dlj), bx = 32 - __clz(xj < 0 ? -(uint32_t)xj : (uint32_t)xj);
        if (__all_sync(0xffffffffu, bd + bB <= 50 && bd + bB + bx <= 69)) {
          scan_state<false>(s_tab, dlj, xj, a4.x, b4.x, c4.x, hv[j].x, ya_lo, ya_hi);
          scan_state<false>(s_tab, dlj, xj, a4.y, b4.y, c4.y, hv[j].y, ya_lo, ya_hi);
          scan_state<false>(s_tab, dlj, xj, a4.z, b4.z, c4.z, hv[j].z, ya_lo, ya_hi);
          scan_state<false>(s_tab, dlj, xj, a4.w, b4.w, c4.w, hv[j].w, ya_lo, ya_hi);
        } else {
          scan_state<true>(s_tab, dlj, xj, a4.x, b4.x, c4.x, hv[j].x, ya_lo, ya_hi);
          scan_state<true>(s_tab, dlj, xj, a4.y, b4.y, c4.y, hv[j].y, ya_lo, ya_hi);
          scan_state<true>(s_tab, dlj, xj, a4.z, b4.z, c4.z, hv[j].z, ya_lo, ya_hi);
          scan_state<true>(s_tab, dlj, xj, a4.w, b4.w, c4.w, hv[j].w, ya_lo, ya_hi);
        }
        __stcs(hp + 32 * j, hv[j]);
        int64_t ya = (int64_t)(((uint64_t)(uint32_t)ya_hi << 32) | ya_lo);
        ya += __shfl_xor_sync(0xffffffffu, ya, 1);
        ya += __shfl_xor_sync(0xffffffffu, ya, 2);
        const int64_t got = __shfl_sync(0xffffffffu, ya, 4 * (lane & 7));
        if ((lane >> 3) == j) ya_own = got;
      }
      const int64_t ys = sat(ya_own + rne((int64_t)d_skip[e] * (int64_t)x, F));
      const int32_t yv = (int32_t)qmul(ys, silu_s(s_tab, z));
      s_y[e] = yv;                                  // read back by the same thread below
      ym = max(ym, abs64(yv));
    }
  }
  ym = block_max(ym, red);
  const int k = max(bitlen64(ym) - 7, 0);
  for (int cg = warp; cg * 32 < E; cg += 8) {
    const int e = cg * 32 + lane;
    q[a_img_off(i, e, KB)] = cut8(s_y[e], k);
  }
  if (tid == 0) kshift[i] = k;
}

}  // namespace fx
}  // namespace boa
