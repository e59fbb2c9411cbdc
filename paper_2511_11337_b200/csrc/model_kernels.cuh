// model_kernels.cuh — the Mamba-1 decode step for B streams (S1-S10 of SURVEY §8(a)).
//
//   k_embed     S1      u = Emb[s_t]                                   (Alg. 1 l.1)
//   k_sgemm_nt  S2+S3   xz = W_in (RMSNorm(u))                         (R#1, R#10)
//               S9      u += W_out y                                   (Alg. 1 l.3)
//               S10     logits = Emb u                                 (Alg. 1 l.5)
//   k_convx     S4-S6   causal conv1d + SiLU, x_proj, dt_proj+softplus (eq. 20-22; R#4, R#11)
//   k_scan      S7+S8   h = exp(dA) h + (dB) x ; y = C.h + D x ; gate  (eq. 16, 18-19; R#3)
//
// Determinism: the value computed for stream i depends only on stream i's inputs and on a
// fixed operation order — never on B, on the tile a stream falls in, or on encode vs decode mode.
// Every reduction below has a fixed order (sequential k-loops, fixed xor-butterflies); there are
// no atomics.  Generation 1 runs all contractions as fp32 FMA on the CUDA cores.
#pragma once
#include "common.cuh"

namespace boa {

__device__ __forceinline__ float warp_sum(float v) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
  return v;
}

__device__ __forceinline__ float sigmoidf_(float x) { return 1.0f / (1.0f + expf(-x)); }
__device__ __forceinline__ float siluf_(float x) { return x * sigmoidf_(x); }
// log(1+exp(v)) in the overflow-free form max(v,0)+log1p(exp(-|v|))  (eq. 20; R#10)
__device__ __forceinline__ float softplusf_(float v) { return fmaxf(v, 0.0f) + log1pf(expf(-fabsf(v))); }

// ---------------------------------------------------------------------------------------------------
// S1: u[i][:] = Emb[src[i*chunk + min(pos_i, len_i-1)]].  In compress mode `src` is the input; in
// decompress mode it is the output buffer, whose byte pos_i was written by the previous coder step.
__global__ void k_embed(const uint8_t* __restrict__ src, size_t chunk_bytes, const uint32_t* __restrict__ pos,
                        const uint32_t* __restrict__ len, const float4* __restrict__ emb, float4* __restrict__ u,
                        int B, int D4) {
  int idx = blockIdx.x * blockDim.x + threadIdx.x;
  if (idx >= B * D4) return;
  int i = idx / D4, q = idx - i * D4;
  uint32_t p = min(pos[i], len[i] - 1u);
  uint32_t s = src[(size_t)i * chunk_bytes + p];
  u[idx] = emb[s * D4 + q];
}

// ---------------------------------------------------------------------------------------------------
// C[M][N] (+)= rowscale[m] * sum_k A[m][k] * (W[n][k] * colscale[k]),  A and W both K-contiguous.
//   NORM : rowscale = rsqrt(mean_k A[m][k]^2 + eps), colscale = norm_w  (RMSNorm folded around the GEMM)
//   RESID: C += result (residual connection), else C = result.
// N % BN == 0 and K % 16 == 0 (guaranteed by boa_model_load); M is ragged (rows clamped on load,
// guarded on store).  Each output element is one sequential fp32 FMA chain over k = 0..K-1.
template <int BM, int BN, int TM, int TN, bool NORM, bool RESID>
__global__ void __launch_bounds__((BM / TM) * (BN / TN))
k_sgemm_nt(const float* __restrict__ A, int lda, const float* __restrict__ W, int ldw,
           const float* __restrict__ norm_w, float* C, int ldc, int M, int N, int K) {
  constexpr int BK = 16;
  constexpr int NT = (BM / TM) * (BN / TN);
  constexpr int A_LD = BM * (BK / 4) / NT;
  constexpr int W_LD = BN * (BK / 4) / NT;
  static_assert(A_LD >= 1 && W_LD >= 1 && TM % 4 == 0 && TN == 4, "tile shape");
  __shared__ __align__(16) float As[2][BK][BM + 4];
  __shared__ __align__(16) float Ws[2][BK][BN + 4];
  __shared__ float rstd_s[BM];

  const int tid = threadIdx.x;
  const int m0 = blockIdx.x * BM, n0 = blockIdx.y * BN;
  const int tx = tid % (BN / TN), ty = tid / (BN / TN);

  if (NORM) {
    const int warp = tid >> 5, lane = tid & 31;
    for (int r = warp; r < BM; r += NT / 32) {
      const float4* row = reinterpret_cast<const float4*>(A + (size_t)min(m0 + r, M - 1) * lda);
      float ss = 0.0f;
      for (int k4 = lane; k4 < K / 4; k4 += 32) {
        float4 v = row[k4];
        ss = fmaf(v.x, v.x, ss); ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
      }
      ss = warp_sum(ss);
      if (lane == 0) rstd_s[r] = 1.0f / sqrtf(ss / (float)K + kEps);
    }
  }

  float4 ra[A_LD], rw[W_LD];
  auto gload = [&](int kt) {
#pragma unroll
    for (int p = 0; p < A_LD; ++p) {
      int f = tid + p * NT, row = f >> 2, kq = f & 3;
      ra[p] = *reinterpret_cast<const float4*>(A + (size_t)min(m0 + row, M - 1) * lda + kt * BK + kq * 4);
    }
#pragma unroll
    for (int p = 0; p < W_LD; ++p) {
      int f = tid + p * NT, row = f >> 2, kq = f & 3;
      float4 w = *reinterpret_cast<const float4*>(W + (size_t)(n0 + row) * ldw + kt * BK + kq * 4);
      if (NORM) {
        float4 s = *reinterpret_cast<const float4*>(norm_w + kt * BK + kq * 4);
        w.x *= s.x; w.y *= s.y; w.z *= s.z; w.w *= s.w;
      }
      rw[p] = w;
    }
  };
  auto sstore = [&](int buf) {
#pragma unroll
    for (int p = 0; p < A_LD; ++p) {
      int f = tid + p * NT, row = f >> 2, kq = f & 3;
      As[buf][kq * 4 + 0][row] = ra[p].x; As[buf][kq * 4 + 1][row] = ra[p].y;
      As[buf][kq * 4 + 2][row] = ra[p].z; As[buf][kq * 4 + 3][row] = ra[p].w;
    }
#pragma unroll
    for (int p = 0; p < W_LD; ++p) {
      int f = tid + p * NT, row = f >> 2, kq = f & 3;
      Ws[buf][kq * 4 + 0][row] = rw[p].x; Ws[buf][kq * 4 + 1][row] = rw[p].y;
      Ws[buf][kq * 4 + 2][row] = rw[p].z; Ws[buf][kq * 4 + 3][row] = rw[p].w;
    }
  };

  float acc[TM][TN];
#pragma unroll
  for (int i = 0; i < TM; ++i)
#pragma unroll
    for (int j = 0; j < TN; ++j) acc[i][j] = 0.0f;

  const int KT = K / BK;
  gload(0);
  sstore(0);
  __syncthreads();
  for (int kt = 0; kt < KT; ++kt) {
    const int buf = kt & 1;
    if (kt + 1 < KT) gload(kt + 1);
#pragma unroll
    for (int k = 0; k < BK; ++k) {
      float a[TM], w[TN];
#pragma unroll
      for (int i = 0; i < TM; i += 4) {
        float4 v = *reinterpret_cast<const float4*>(&As[buf][k][ty * TM + i]);
        a[i] = v.x; a[i + 1] = v.y; a[i + 2] = v.z; a[i + 3] = v.w;
      }
      {
        float4 v = *reinterpret_cast<const float4*>(&Ws[buf][k][tx * TN]);
        w[0] = v.x; w[1] = v.y; w[2] = v.z; w[3] = v.w;
      }
#pragma unroll
      for (int i = 0; i < TM; ++i)
#pragma unroll
        for (int j = 0; j < TN; ++j) acc[i][j] = fmaf(a[i], w[j], acc[i][j]);
    }
    if (kt + 1 < KT) sstore(buf ^ 1);
    __syncthreads();
  }

#pragma unroll
  for (int i = 0; i < TM; ++i) {
    int row = m0 + ty * TM + i;
    if (row >= M) continue;
    float sc = NORM ? rstd_s[ty * TM + i] : 1.0f;
    float4* cp = reinterpret_cast<float4*>(C + (size_t)row * ldc + n0 + tx * TN);
    float4 o = make_float4(acc[i][0] * sc, acc[i][1] * sc, acc[i][2] * sc, acc[i][3] * sc);
    if (RESID) {
      float4 c = *cp;
      o.x += c.x; o.y += c.y; o.z += c.z; o.w += c.w;
    }
    *cp = o;
  }
}

// ---------------------------------------------------------------------------------------------------
// S4-S6 for a tile of TS streams; blockDim.x = E (one thread per channel).
//   xc_e = conv_b[e] + sum_k conv_w[e][k] * (x_{t-3}, x_{t-2}, x_{t-1}, x_t)[k]   (R#11: tap 3 = current)
//   xs = SiLU(xc);  [dlt;Bv;Cv] = W_x xs;  delta = softplus(W_dt dlt + b_dt)
// win   [B][3][E]   conv window of this layer (read, shifted, written)
// xs    [B][E], delta [B][E], bc [B][32] (Bv then Cv) are written for k_scan.
template <int TS>
__global__ void __launch_bounds__(1024)
k_convx(const float* __restrict__ xz, float* __restrict__ win, const float4* __restrict__ conv_w,
        const float* __restrict__ conv_b, const float* __restrict__ W_x, const float* __restrict__ W_dtT,
        const float* __restrict__ b_dt, float* __restrict__ xs, float* __restrict__ delta,
        float* __restrict__ bc, int B, int E, int R) {
  extern __shared__ float sm[];
  const int J = R + 2 * kNState;
  float* xs_s = sm;             // [TS][E]
  float* dbc_s = sm + TS * E;   // [TS][J]
  const int e = threadIdx.x;
  const int i0 = blockIdx.x * TS;
  const int lane = e & 31, warp = e >> 5, nwarps = E >> 5;

  const float4 cw = conv_w[e];
  const float cb = conv_b[e];
#pragma unroll
  for (int s = 0; s < TS; ++s) {
    const int i = i0 + s;
    float v = 0.0f;
    if (i < B) {
      float* wp = win + (size_t)i * 3 * E + e;
      const float x = xz[(size_t)i * 2 * E + e];
      const float w0 = wp[0], w1 = wp[E], w2 = wp[2 * E];
      float xc = fmaf(cw.w, x, cb);
      xc = fmaf(cw.x, w0, xc);
      xc = fmaf(cw.y, w1, xc);
      xc = fmaf(cw.z, w2, xc);
      wp[0] = w1; wp[E] = w2; wp[2 * E] = x;
      v = siluf_(xc);
      xs[(size_t)i * E + e] = v;
    }
    xs_s[s * E + e] = v;
  }
  __syncthreads();

  for (int j = warp; j < J; j += nwarps) {
    float acc[TS];
#pragma unroll
    for (int s = 0; s < TS; ++s) acc[s] = 0.0f;
    for (int k = lane; k < E; k += 32) {
      const float w = W_x[(size_t)j * E + k];
#pragma unroll
      for (int s = 0; s < TS; ++s) acc[s] = fmaf(w, xs_s[s * E + k], acc[s]);
    }
#pragma unroll
    for (int s = 0; s < TS; ++s) acc[s] = warp_sum(acc[s]);
    if (lane == 0) {
#pragma unroll
      for (int s = 0; s < TS; ++s) dbc_s[s * J + j] = acc[s];
    }
  }
  __syncthreads();

  {
    float acc[TS];
    const float b = b_dt[e];
#pragma unroll
    for (int s = 0; s < TS; ++s) acc[s] = b;
    for (int r = 0; r < R; ++r) {
      const float w = W_dtT[(size_t)r * E + e];
#pragma unroll
      for (int s = 0; s < TS; ++s) acc[s] = fmaf(w, dbc_s[s * J + r], acc[s]);
    }
#pragma unroll
    for (int s = 0; s < TS; ++s)
      if (i0 + s < B) delta[(size_t)(i0 + s) * E + e] = softplusf_(acc[s]);
  }
  if (e < 2 * kNState) {
#pragma unroll
    for (int s = 0; s < TS; ++s)
      if (i0 + s < B) bc[(size_t)(i0 + s) * 2 * kNState + e] = dbc_s[s * J + R + e];
  }
}

// ---------------------------------------------------------------------------------------------------
// S7+S8: one thread per (stream, channel) holds the 16 state values of that channel in registers.
//   h[n] = exp(delta*A[n]) * h[n] + (delta*Bv[n]) * xs ;  y = sum_n Cv[n] h[n] + D xs ;  y *= SiLU(z)
// State layout: h[i][j][e] is a float4 holding n = 4j..4j+3, so the 32
// lanes of a warp read 512 contiguous bytes per load.  The state is the only large object on the
// path and is touched once per step: it is loaded/stored with streaming (evict-first) hints so the
// small activations stay in L2.  The next stream's state is prefetched while the current one is
// being updated.
__device__ __forceinline__ void scan_update4(float4& h, const float4 a, const float4 bv, const float4 cv,
                                             float dl, float x, float& y) {
  h.x = fmaf(expf(dl * a.x), h.x, (dl * bv.x) * x); y = fmaf(cv.x, h.x, y);
  h.y = fmaf(expf(dl * a.y), h.y, (dl * bv.y) * x); y = fmaf(cv.y, h.y, y);
  h.z = fmaf(expf(dl * a.z), h.z, (dl * bv.z) * x); y = fmaf(cv.z, h.z, y);
  h.w = fmaf(expf(dl * a.w), h.w, (dl * bv.w) * x); y = fmaf(cv.w, h.w, y);
}

template <int SPC>
__global__ void __launch_bounds__(256)
k_scan(float4* __restrict__ h, const float* __restrict__ delta, const float* __restrict__ xs,
       const float* __restrict__ xz, const float* __restrict__ bc, const float4* __restrict__ A4,
       const float* __restrict__ Dskip, float* __restrict__ y, int B, int E) {
  const int e = blockIdx.y * blockDim.x + threadIdx.x;
  const float4 a0 = A4[e], a1 = A4[E + e], a2 = A4[2 * E + e], a3 = A4[3 * E + e];
  const float dsk = Dskip[e];
  const int i0 = blockIdx.x * SPC;
  const int iend = min(i0 + SPC, B);
  if (i0 >= B) return;

  float4 n0, n1, n2, n3;
  {
    const float4* hp = h + (size_t)i0 * 4 * E + e;
    n0 = __ldcs(hp); n1 = __ldcs(hp + E); n2 = __ldcs(hp + 2 * E); n3 = __ldcs(hp + 3 * E);
  }
  for (int i = i0; i < iend; ++i) {
    float4 h0 = n0, h1 = n1, h2 = n2, h3 = n3;
    if (i + 1 < iend) {
      const float4* hp = h + (size_t)(i + 1) * 4 * E + e;
      n0 = __ldcs(hp); n1 = __ldcs(hp + E); n2 = __ldcs(hp + 2 * E); n3 = __ldcs(hp + 3 * E);
    }
    const float dl = delta[(size_t)i * E + e];
    const float x = xs[(size_t)i * E + e];
    const float z = xz[(size_t)i * 2 * E + E + e];
    const float4* bcp = reinterpret_cast<const float4*>(bc + (size_t)i * 2 * kNState);
    const float4 b0 = __ldg(bcp), b1 = __ldg(bcp + 1), b2 = __ldg(bcp + 2), b3 = __ldg(bcp + 3);
    const float4 c0 = __ldg(bcp + 4), c1 = __ldg(bcp + 5), c2 = __ldg(bcp + 6), c3 = __ldg(bcp + 7);
    float yv = 0.0f;
    scan_update4(h0, a0, b0, c0, dl, x, yv);
    scan_update4(h1, a1, b1, c1, dl, x, yv);
    scan_update4(h2, a2, b2, c2, dl, x, yv);
    scan_update4(h3, a3, b3, c3, dl, x, yv);
    yv = fmaf(dsk, x, yv);
    yv *= siluf_(z);
    float4* hq = h + (size_t)i * 4 * E + e;
    __stcs(hq, h0); __stcs(hq + E, h1); __stcs(hq + 2 * E, h2); __stcs(hq + 3 * E, h3);
    y[(size_t)i * E + e] = yv;
  }
}

}  // namespace boa
