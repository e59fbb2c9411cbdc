// model_kernels.cuh — the CUDA-core kernels of the Mamba-1 decode step for B streams.
//
//   k_embed     S1      u = Emb[s_t]                                   (Alg. 1 l.1)
//   k_scan      S6-S8   delta = softplus(W_dt dlt + b_dt)              (eq. 20; R#10)
//                       h = exp(delta A) h + (delta B) x ; y = C.h + D x ; y *= SiLU(z)
//                                                                      (eq. 16, 18-19; R#3)
// The contractions over the stream batch (in_proj, x_proj, out_proj, head; S2-S5, S9, S10) are tensor-core
// kernels: tc_gemm.cuh.
//
// Determinism: the value computed for stream i depends only on stream i's inputs and on a
// fixed operation order — never on B, on the tile a stream falls in, or on encode vs decode mode.
// Every reduction below has a fixed order (sequential k-loops, fixed xor-butterflies); there are
// no atomics.
#pragma once
#include "common.cuh"
#include "tc_gemm.cuh"

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
// Also writes the image of u * norm_w(layer 0), the operand of the first in_proj (tc_gemm.cuh), and the sums of
// u^2 over each 64-column block (one thread per 4 columns: x, y, z, w, then the xor butterfly 8, 4, 2, 1 over the
// 16 threads of the block) from which in_proj forms the RMSNorm row scale.
__global__ void k_embed(const uint8_t* __restrict__ src, size_t chunk_bytes, const uint32_t* __restrict__ pos,
                        const uint32_t* __restrict__ len, const float4* __restrict__ emb, float4* __restrict__ u,
                        const float4* __restrict__ norm_w, uint8_t* __restrict__ u_img, float* __restrict__ ssq,
                        int B, int D4, int T) {
  // T > 1 (encode-side time slab): rows are stream-major, row i*T + t is byte pos_i + t of stream i
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const bool live = idx < B * T * D4;             // a multiple of 16: a 16-thread block is live as a whole
  const int row = live ? idx / D4 : 0, q = live ? idx - row * D4 : 0;
  const int i = row / T, t = row - i * T;
  const uint32_t p = min(pos[i] + (uint32_t)t, len[i] - 1u);
  const uint32_t s = src[(size_t)i * chunk_bytes + p];
  const float4 v = emb[s * D4 + q];
  float ss = v.x * v.x;
  ss = fmaf(v.y, v.y, ss); ss = fmaf(v.z, v.z, ss); ss = fmaf(v.w, v.w, ss);
#pragma unroll
  for (int d = 8; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
  if (!live) return;
  u[idx] = v;
  if ((q & 15) == 0) ssq[(size_t)row * (D4 >> 4) + (q >> 4)] = ss;
  const float4 w = norm_w[q];
  tc::cut4_store(u_img, D4 >> 4, row, q * 4, make_float4(v.x * w.x, v.y * w.y, v.z * w.z, v.w * w.w));
}

// ---------------------------------------------------------------------------------------------------
// The paper's block only (Alg. 1 l.4; R#23): u = LayerNorm(v), v = FFN(u) as written by
// the second FFN contraction.  One warp per row; lane l holds columns 128 j + 4 l .. + 3.
//   mean = (sum v) / D ;  var = (sum (v - mean)^2) / D (biased) ;  u = (v - mean) / sqrt(var + eps) * ln_w + ln_b
// Both sums: per lane j ascending over x, y, z, w, then the xor butterfly 16, 8, 4, 2, 1.  Like the residual epilogue
// of out_proj it also writes what the next contraction needs: the image of u (times the next layer's RMSNorm weight,
// or plain for the head) and the sums of u^2 over each 64-column block (x, y, z, w, then the butterfly 8, 4, 2, 1
// over the 16 lanes of the block).  D <= 512 (4 float4 per lane).
__global__ void k_layernorm(const float* __restrict__ v, const float* __restrict__ ln_w, const float* __restrict__ ln_b,
                            float* __restrict__ u, const float* __restrict__ next_scale, uint8_t* __restrict__ u_img,
                            float* __restrict__ ssq, int rows, int D) {
  pdl_wait();
  const int row = (int)((blockIdx.x * blockDim.x + threadIdx.x) >> 5), lane = threadIdx.x & 31;
  if (row >= rows) return;                         // warp-uniform
  float4 x[4];
  float s = 0.0f;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int c = 128 * j + 4 * lane;
    x[j] = c < D ? *reinterpret_cast<const float4*>(v + (size_t)row * D + c) : make_float4(0.f, 0.f, 0.f, 0.f);
    s += x[j].x; s += x[j].y; s += x[j].z; s += x[j].w;
  }
  const float mean = warp_sum(s) / (float)D;
  float q = 0.0f;
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    if (128 * j + 4 * lane < D) {
      x[j].x -= mean; x[j].y -= mean; x[j].z -= mean; x[j].w -= mean;
      q = fmaf(x[j].x, x[j].x, q); q = fmaf(x[j].y, x[j].y, q); q = fmaf(x[j].z, x[j].z, q); q = fmaf(x[j].w, x[j].w, q);
    }
  }
  const float rstd = 1.0f / sqrtf(warp_sum(q) / (float)D + kEps);
#pragma unroll
  for (int j = 0; j < 4; ++j) {
    const int c = 128 * j + 4 * lane;
    const bool live = c < D;                       // uniform over each group of 16 lanes (D % 64 == 0)
    float4 o = make_float4(0.f, 0.f, 0.f, 0.f);
    if (live) {
      const float4 w = *reinterpret_cast<const float4*>(ln_w + c), b = *reinterpret_cast<const float4*>(ln_b + c);
      o.x = fmaf(x[j].x * rstd, w.x, b.x); o.y = fmaf(x[j].y * rstd, w.y, b.y);
      o.z = fmaf(x[j].z * rstd, w.z, b.z); o.w = fmaf(x[j].w * rstd, w.w, b.w);
    }
    float ss = o.x * o.x;
    ss = fmaf(o.y, o.y, ss); ss = fmaf(o.z, o.z, ss); ss = fmaf(o.w, o.w, ss);
#pragma unroll
    for (int d = 8; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
    if (live) {
      *reinterpret_cast<float4*>(u + (size_t)row * D + c) = o;
      if ((lane & 15) == 0) ssq[(size_t)row * (D >> 6) + (c >> 6)] = ss;
      float4 sc = make_float4(1.f, 1.f, 1.f, 1.f);
      if (next_scale) sc = *reinterpret_cast<const float4*>(next_scale + c);
      tc::cut4_store(u_img, D >> 6, row, c, make_float4(o.x * sc.x, o.y * sc.y, o.z * sc.z, o.w * sc.w));
    }
  }
}

// ---------------------------------------------------------------------------------------------------
// S6-S8, the kernel that streams the SSM state (the only large object of the path) through the SM.
//   delta = softplus(b_dt[e] + sum_r W_dt[e][r] dlt[r])                      (sequential fp32 FMA chain, r ascending)
//   h[n] = exp(delta*A[n]) * h[n] + (delta*Bv[n]) * xs ;  y = sum_n Cv[n] h[n] + D xs ;  y *= SiLU(z)
//
// State layout: h[i][slice][j][c] is a float4 holding n = 4j..4j+3 of channel slice*EC+c,
// so the state of one stream and a slice of EC channels is ONE contiguous run of EC*64 bytes (one bulk copy in, one
// out) and a warp reads 512 contiguous bytes of it per shared-memory load.  HBM-bound: per stream and slice the
// kernel moves 2*EC*64 bytes of state against ~160 instructions per channel, so the design goal is bytes in
// flight, not arithmetic: a persistent CTA owns a channel slice and walks over streams with a ring of NSTG shared
// memory stages.  Everything a stream-step needs (4 state runs, xs, z, the x_proj row) is brought in by the
// bulk-copy engine (TMA, cp.async.bulk -> UBLKCP) against one mbarrier per stage; threads touch shared memory
// only; the updated state goes back with bulk stores.  State copies carry an L2 evict-first policy so the
// small activations stay resident in L2.  y leaves cut into bf16 pieces, written into the image of out_proj's
// operand tile (tc_gemm.cuh).
// One thread per channel of the slice holds A[e][0..15] in registers; W_dt^T of the slice lives in shared memory.
struct ScanArgs {
  float* h;                 // [B][E/EC][4][EC] float4 (this layer): the state of a stream and channel slice is one contiguous run
  const float* xz;          // [rows][E/EC][xs of the slice | z of the slice] (tc::xz_col): one copy per stream-step and slice
  const float* dbc;         // [rows][KS][ldj] k-split partials of x_proj; their ascending sum is dlt[R] | Bv[16] | Cv[16]
  int KS;                   // the copy warp adds the partials once per stream-step, ((p0+p1)+p2)+...
  const float* W_dtT;       // [R][E]
  const float* b_dt;        // [E]
  const float4* A4;         // [4][E] float4: A * log2(e), A = -exp(A_log)
  const float* Dskip;       // [E]
  uint8_t* y_img;           // image of y[B][E] for out_proj (tc_gemm.cuh)
  int ldj, B, E, R;
};

namespace scan {
constexpr int NSB = 4;           // state buffers (one stream-slice state each): the ring the HBM traffic flows through
constexpr int NSTG = 8;          // step stages (the small per-step inputs and outputs): deeper, a slab step is short
constexpr int KSMAX = 4;         // x_proj k-split partial rows per stage
__host__ __device__ inline int stage_bytes(int EC, int ldj) { return 2 * EC * 4 + EC * 6 + KSMAX * ldj * 4; }   // xs | z | y pieces | dbc partials
__host__ __device__ inline int smem_bytes(int EC, int ldj, int R) {   // R = 0 when W_dt sits in registers
  return NSB * EC * 64 + NSTG * stage_bytes(EC, ldj) + R * EC * 4 + 3 * NSTG * 8 + 128;
}

__device__ __forceinline__ uint32_t s_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void bar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void bar_expect(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
__device__ __forceinline__ void g2s_hint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "l"(pol) : "memory");
}
__device__ __forceinline__ void s2g(void* dst, uint32_t src, uint32_t bytes) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void s2g_hint(void* dst, uint32_t src, uint32_t bytes, uint64_t pol) {
  asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;"
               ::"l"(dst), "r"(src), "r"(bytes), "l"(pol) : "memory");
}
}  // namespace scan

// Fast forms for the stateless activations of the scan (relative error ~1e-6, far inside the 1e-5 probability bar;
// encode and decode run the same code, so determinism is unaffected).
__device__ __forceinline__ float silu_fast(float x) { return __fdividef(x, 1.0f + __expf(-x)); }
__device__ __forceinline__ float softplus_fast(float v) { return fmaxf(v, 0.0f) + log1pf(__expf(-fabsf(v))); }
__device__ __forceinline__ float ex2_approx(float x) {
  float y;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
  return y;
}
// h <- 2^(dl*a2) h + (dl*Bv) x,  a2 = A*log2(e) (folded into the weights at load);  y += Cv h
__device__ __forceinline__ void scan_update4(float4& h, const float4 a2, const float4 bv, const float4 cv,
                                             float dl, float x, float& y) {
  const float dx = dl * x;
  h.x = fmaf(ex2_approx(dl * a2.x), h.x, dx * bv.x); y = fmaf(cv.x, h.x, y);
  h.y = fmaf(ex2_approx(dl * a2.y), h.y, dx * bv.y); y = fmaf(cv.y, h.y, y);
  h.z = fmaf(ex2_approx(dl * a2.z), h.z, dx * bv.z); y = fmaf(cv.z, h.z, y);
  h.w = fmaf(ex2_approx(dl * a2.w), h.w, dx * bv.w); y = fmaf(cv.w, h.w, y);
}

// S6-S8 of one channel for one step: dt_proj + softplus, the recurrence on the 16 state values, D skip and gate.
// `row` = dlt[R] | Bv[16] | Cv[16] (shared memory, broadcast reads).  The one definition used by the step kernel and
// by the encode-side slab kernel, so both produce the same bits.
template <int RR>
__device__ __forceinline__ float scan_channel_step(const float* row, int R, const float (&wr)[RR ? RR : 1], const float* wdt_col,
                                                   int EC, float bdt, const float4 a0, const float4 a1, const float4 a2,
                                                   const float4 a3, float dsk, float x, float z, float4& h0, float4& h1,
                                                   float4& h2, float4& h3) {
  float acc = bdt;
  if constexpr (RR > 0) {
#pragma unroll
    for (int r = 0; r < RR; r += 4) {
      const float4 d = *reinterpret_cast<const float4*>(row + r);
      acc = fmaf(wr[r], d.x, acc);
      acc = fmaf(wr[r + 1], d.y, acc);
      acc = fmaf(wr[r + 2], d.z, acc);
      acc = fmaf(wr[r + 3], d.w, acc);
    }
  } else {
    for (int r = 0; r < R; r += 4) {
      const float4 d = *reinterpret_cast<const float4*>(row + r);
      acc = fmaf(wdt_col[(r + 0) * EC], d.x, acc);
      acc = fmaf(wdt_col[(r + 1) * EC], d.y, acc);
      acc = fmaf(wdt_col[(r + 2) * EC], d.z, acc);
      acc = fmaf(wdt_col[(r + 3) * EC], d.w, acc);
    }
  }
  const float dl = softplus_fast(acc);
  const float4* bcp = reinterpret_cast<const float4*>(row + R);
  float yv = 0.0f;
  scan_update4(h0, a0, bcp[0], bcp[4], dl, x, yv);
  scan_update4(h1, a1, bcp[1], bcp[5], dl, x, yv);
  scan_update4(h2, a2, bcp[2], bcp[6], dl, x, yv);
  scan_update4(h3, a3, bcp[3], bcp[7], dl, x, yv);
  yv = fmaf(dsk, x, yv);
  return yv * silu_fast(z);
}

// The roles of a scan CTA over the streams i_begin + bx, + gx, ... < i_end of channel slice `sl` (EC channels):
// threads 0..EC-1 = one thread per channel, the warp after them drives the bulk copies and moves the y pieces; later
// threads (if the block is larger) only take part in the block barrier.  Initialises its own barriers in `scan_smem`.
// Shared by k_scan (one launch per layer and step) and the persistent step kernel (step_persist.cuh).
// RR = dt_rank when W_dt's row is held in registers (4, 8, 16, 32), else 0 (row kept in shared memory).
template <int RR>
__device__ __forceinline__ void scan_roles(const ScanArgs& a, uint8_t* scan_smem, int EC, int sl, int slices, int bx, int gx,
                                           int i_begin, int i_end) {
  using namespace scan;
  const int tid = threadIdx.x;
  const int e0 = sl * EC;
  const int SB = stage_bytes(EC, a.ldj);
  uint8_t* sbufs = scan_smem;                      // [NSB][EC*64] state buffers
  uint8_t* stages = scan_smem + NSB * EC * 64;     // [NSTG][SB] step stages
  float* wdt = reinterpret_cast<float*>(stages + NSTG * SB);
  uint64_t* bars = reinterpret_cast<uint64_t*>(stages + NSTG * SB + (RR ? 0 : a.R * EC * 4));   // full, done, ready [NSTG] each
  constexpr int T = 1;                             // steps per stream and launch (the time-slab form is k_scan_slab)
  constexpr int LA = NSB;                          // copies run LA iterations ahead: one state buffer each
  const int nk = (i_end - i_begin - bx + gx - 1) / gx;   // streams of this CTA
  if (nk <= 0) return;

  if (tid == 0) {
    for (int s = 0; s < NSTG; ++s) {
      bar_init(s_u32(&bars[s]), 1);                       // full: the bulk copies of a stage have landed
      bar_init(s_u32(&bars[NSTG + s]), (uint32_t)EC);     // done: every channel thread has finished the stream
      bar_init(s_u32(&bars[2 * NSTG + s]), 1);            // ready: the x_proj partial rows have been added up
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_launch();
  if (tid >= EC + 32) return;

  if (tid >= EC) {
    // ===================================================================== copy warp
    const int lane = tid - EC;
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    const int niter = nk * T;                      // iteration kk = stream k of this CTA
    // This warp is one serial instruction stream beside eight channel warps: indices advance incrementally (no
    // divisions), per-lane offsets are computed once.
    static_assert((NSTG & (NSTG - 1)) == 0 && (NSB & (NSB - 1)) == 0, "ring sizes are powers of two");
    const size_t state_stride = (size_t)slices * 4 * EC * 4;        // floats between the states of consecutive streams
    const float* h0p = a.h + (size_t)sl * 4 * EC * 4;
    const float* xz0 = a.xz + (size_t)sl * 2 * EC;
    const uint32_t xz_bytes = (uint32_t)(2 * EC * 4), dbc_bytes = (uint32_t)(a.KS * a.ldj * 4);
    int ik = 0, it_ = 0, ikk = 0;                  // next copy to issue: stream, step, iteration
    size_t ii = (size_t)(i_begin + bx);                        // its stream index in the wave
    auto issue_next = [&]() {   // lane 0
      const int s = ikk & (NSTG - 1);
      const size_t row = (size_t)it_ * a.B + ii;
      const uint32_t st = s_u32(stages + s * SB), bar = s_u32(&bars[s]);
      bar_expect(bar, (it_ == 0 ? (uint32_t)(EC * 64) : 0u) + xz_bytes + dbc_bytes);
      if (it_ == 0) g2s_hint(s_u32(sbufs + (ik & (NSB - 1)) * EC * 64), h0p + ii * state_stride, (uint32_t)(EC * 64), bar, pol);
      g2s(st, xz0 + row * 2 * a.E, xz_bytes, bar);                                                  // xs | z
      g2s(st + 2 * EC * 4 + EC * 6, a.dbc + row * a.KS * a.ldj, dbc_bytes, bar);                     // all partials
      ++ikk;
      if (++it_ == T) { it_ = 0; ++ik; ii += gx; }
    };
    // S5, last step: the k-split partials of the x_proj row are added in ascending order, in place, once per stream-step
    auto reduce_row = [&](int kk) {   // whole warp
      const int s = kk & (NSTG - 1);
      bar_wait(s_u32(&bars[s]), (uint32_t)((kk / NSTG) & 1));
      float* row = reinterpret_cast<float*>(stages + s * SB + 2 * EC * 4 + EC * 6);
      const int KS = a.KS, ldj = a.ldj;
      for (int c = lane; c < ldj; c += 32) {       // every partial of an element in flight before the adds (ascending order)
        float x[KSMAX];
#pragma unroll
        for (int p = 0; p < KSMAX; ++p) x[p] = p < KS ? row[p * ldj + c] : 0.0f;
        float v = x[0];
#pragma unroll
        for (int p = 1; p < KSMAX; ++p)
          if (p < KS) v += x[p];
        row[c] = v;
      }
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(&bars[2 * NSTG + s])) : "memory");
    };
    pdl_wait();                                    // the state, xz and the x_proj rows come from earlier kernels
    if (lane == 0)
      for (int kk = 0; kk < LA && kk < niter; ++kk) issue_next();
    // y pieces: 16-byte chunk c of a stream-step = row (c/8) = (64-channel block, piece) of the staged pieces, chunk c%8
    // of its 128-byte row in out_proj's operand image; this lane's (at most 3) chunks:
    const int nchunks = (EC >> 6) * 24;
    uint32_t ysrc[3], ydst[3];
#pragma unroll
    for (int j = 0; j < 3; ++j) {
      const int c = lane + 32 * j, rowid = c >> 3, kt = rowid / 3, q = rowid - kt * 3;
      ysrc[j] = (uint32_t)(2 * EC * 4 + rowid * 128 + (c & 7) * 16);
      ydst[j] = (uint32_t)(kt * (tc::NPA * tc::A_PLANE) + q * tc::A_PLANE + (c & 7) * 16);
    }
    const size_t img_row_tile = (size_t)(a.E >> 6) * (tc::NPA * tc::A_PLANE);   // bytes of one 128-row tile of the image
    uint8_t* yimg0 = a.y_img + (size_t)(e0 >> 6) * (tc::NPA * tc::A_PLANE);
    const uint64_t keep = tc::policy_evict_last();
    reduce_row(0);
    int k = 0, t = 0;                              // this iteration's stream and step
    size_t i = (size_t)(i_begin + bx);
    for (int kk = 0; kk < niter; ++kk) {
      const int s = kk & (NSTG - 1);
      uint8_t* st = stages + s * SB;
      if (kk + 1 < niter) reduce_row(kk + 1);      // its copies were issued at least one iteration ago
      bar_wait(s_u32(&bars[NSTG + s]), (uint32_t)((kk / NSTG) & 1));     // every channel of this stream-step is done
      if (lane == 0) {
        if (t == T - 1)
          s2g_hint(const_cast<float*>(h0p) + i * state_stride, s_u32(sbufs + (k & (NSB - 1)) * EC * 64), (uint32_t)(EC * 64), pol);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
      }
      const size_t row = (size_t)t * a.B + i;
      const int r = (int)(row & 127);
      uint8_t* ybase = yimg0 + (row >> 7) * img_row_tile + (r >> 3) * 1024 + (r & 7) * 128;
#pragma unroll
      for (int j = 0; j < 3; ++j)
        if (lane + 32 * j < nchunks) tc::st_keep_v4(ybase + ydst[j], *reinterpret_cast<const uint4*>(st + ysrc[j]), keep);
      __syncwarp();
      if (lane == 0 && kk >= 1 && ikk < niter) {
        asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");   // every state store but this iteration's has left its buffer
        issue_next();                              // iteration kk - 1 + LA
      }
      if (++t == T) { t = 0; ++k; i += gx; }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");   // the state stores are complete (the persistent
    return;                                                                     // step kernel reads them back in the next step)
  }

  // ======================================================================= channel threads
  const int e = e0 + tid;
  float wr[RR ? RR : 1];
  if constexpr (RR > 0) {
#pragma unroll
    for (int r = 0; r < RR; ++r) wr[r] = a.W_dtT[(size_t)r * a.E + e];
  } else {
    for (int r = 0; r < a.R; ++r) wdt[r * EC + tid] = a.W_dtT[(size_t)r * a.E + e];   // private column: no sync needed
  }
  const float4 a0 = a.A4[e], a1 = a.A4[a.E + e], a2 = a.A4[2 * a.E + e], a3 = a.A4[3 * a.E + e];
  const float dsk = a.Dskip[e];
  const float bdt = a.b_dt[e];

  const int niter = nk * T;
  float4 h0, h1, h2, h3;                           // the channel's 16 state values: in registers across a slab
  int k = 0, t = 0;
  size_t row_i = (size_t)(i_begin + bx);                       // this iteration's stream index in the wave
  for (int kk = 0; kk < niter; ++kk) {
    const int s = kk & (NSTG - 1);
    uint8_t* st = stages + s * SB;
    bar_wait(s_u32(&bars[2 * NSTG + s]), (uint32_t)((kk / NSTG) & 1));  // copies landed and the x_proj row added up
    float4* hs = reinterpret_cast<float4*>(sbufs + (k % NSB) * EC * 64);
    const float* xs_s = reinterpret_cast<const float*>(st);
    const float* row = reinterpret_cast<const float*>(st + 2 * EC * 4 + EC * 6);
    const float x = xs_s[tid];
    const float z = xs_s[EC + tid];
    if (t == 0) { h0 = hs[tid]; h1 = hs[EC + tid]; h2 = hs[2 * EC + tid]; h3 = hs[3 * EC + tid]; }
    float yv = scan_channel_step<RR>(row, a.R, wr, wdt + tid, EC, bdt, a0, a1, a2, a3, dsk, x, z, h0, h1, h2, h3);
    if (t == T - 1) { hs[tid] = h0; hs[EC + tid] = h1; hs[2 * EC + tid] = h2; hs[3 * EC + tid] = h3; }
    {
      // y -> three bf16 pieces (truncation split, exact), staged as [64-channel block][piece][128-byte swizzled row]
      const int i7 = (int)(((size_t)t * a.B + row_i) & 7);
      uint8_t* yp = st + 2 * EC * 4 + ((tid >> 6) * 3) * 128 + (((((tid & 63) >> 3) ^ i7) & 7) << 4) + (tid & 7) * 2;
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        *reinterpret_cast<uint16_t*>(yp + q * 128) = (uint16_t)(__float_as_uint(yv) >> 16);
        yv = __fsub_rn(yv, tc::trunc_bf16(yv));
      }
    }
    if (t == T - 1) asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // the state leaves by a bulk store
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(&bars[NSTG + s])) : "memory");
    if (++t == T) { t = 0; ++k; row_i += gx; }
  }
}

// grid = (CTAs per slice, E / EC), block = EC + 32 threads (EC = 256 or 128), two CTAs per SM.
template <int RR>
__global__ void __launch_bounds__(288, 2) k_scan(const ScanArgs a) {
  extern __shared__ __align__(128) uint8_t scan_smem[];
  scan_roles<RR>(a, scan_smem, (int)blockDim.x - 32, (int)blockIdx.y, (int)gridDim.y, (int)blockIdx.x, (int)gridDim.x, 0, a.B);
}

// ---------------------------------------------------------------------------------------------------
// S6-S8 over an encode-side time slab: rows are stream-major, row(i, t) = i*T + t, T a multiple
// of G = 8.  One iteration of a CTA = one stream and one group of 8 consecutive steps: the copy warp brings in the 8
// rows of xs | z (one copy: the slab's xz is laid out [slice][row][xs | z]) and of x_proj partials (one copy), plus the
// state with the first group of a stream; the channel threads then run the 8 steps back to back with no
// synchronisation in between, the state in registers across the groups of a stream; the 8 rows of y pieces of a
// (64-channel block, piece) form one contiguous 1 KB block of out_proj's operand image and leave by bulk stores,
// with the state after the last group.  Per step the arithmetic is scan_channel_step, as in k_scan.
namespace scan {
constexpr int G = 8;             // steps per iteration
constexpr int NSL = 2;           // stages
__host__ __device__ inline int slab_stage_bytes(int EC, int ldj) { return EC * 64 + G * 2 * EC * 4 + G * EC * 6 + G * KSMAX * ldj * 4; }
__host__ __device__ inline int slab_smem_bytes(int EC, int ldj, int R) { return NSL * slab_stage_bytes(EC, ldj) + R * EC * 4 + 3 * NSL * 8 + 128; }
}  // namespace scan

struct ScanSlabArgs {
  float* h;                 // [B][E/EC][4][EC] float4 (this layer)
  const float* xz;          // [E/EC][rows][xs of the slice | z of the slice], rows = B*T
  const float* dbc;         // [rows][KS][ldj]
  const float* W_dtT; const float* b_dt; const float4* A4; const float* Dskip;
  uint8_t* y_img;           // image of y[rows][E]
  int KS, ldj, B, E, R, T;
};

template <int RR>
__global__ void __launch_bounds__(288, 2) k_scan_slab(const ScanSlabArgs a) {
  using namespace scan;
  extern __shared__ __align__(128) uint8_t scan_smem[];
  const int EC = blockDim.x - 32, tid = threadIdx.x;
  const int slices = gridDim.y, sl = blockIdx.y;
  const int e0 = sl * EC;
  const int SB = slab_stage_bytes(EC, a.ldj);
  const int XZ_OFF = EC * 64, Y_OFF = XZ_OFF + G * 2 * EC * 4, D_OFF = Y_OFF + G * EC * 6;
  uint8_t* stages = scan_smem;
  float* wdt = reinterpret_cast<float*>(stages + NSL * SB);
  uint64_t* bars = reinterpret_cast<uint64_t*>(stages + NSL * SB + (RR ? 0 : a.R * EC * 4));   // full, done, ready [NSL] each
  const int nk = (a.B - (int)blockIdx.x + (int)gridDim.x - 1) / (int)gridDim.x;   // streams of this CTA
  if (nk <= 0) return;
  const int NG = a.T / G, niter = nk * NG;         // iteration kk = (stream k of this CTA, group g of 8 steps)
  const size_t rows = (size_t)a.B * a.T;

  if (tid == 0) {
    for (int s = 0; s < NSL; ++s) {
      bar_init(s_u32(&bars[s]), 1);
      bar_init(s_u32(&bars[NSL + s]), (uint32_t)EC);
      bar_init(s_u32(&bars[2 * NSL + s]), 1);
    }
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  __syncthreads();
  pdl_launch();
  const size_t state_stride = (size_t)slices * 4 * EC * 4;
  float* h0p = a.h + (size_t)sl * 4 * EC * 4;

  if (tid >= EC) {
    // ===================================================================== copy warp
    const int lane = tid - EC;
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    const float* xz0 = a.xz + (size_t)sl * rows * 2 * EC;
    const uint32_t xz_bytes = (uint32_t)(G * 2 * EC * 4), dbc_bytes = (uint32_t)(G * a.KS * a.ldj * 4);
    int ig = 0, ikk = 0;                           // next copy to issue: group within the stream, iteration
    size_t ii = blockIdx.x;
    auto issue_next = [&]() {   // lane 0
      const int s = ikk & (NSL - 1);
      const size_t row = ii * a.T + (size_t)ig * G;
      const uint32_t st = s_u32(stages + s * SB), bar = s_u32(&bars[s]);
      bar_expect(bar, (ig == 0 ? (uint32_t)(EC * 64) : 0u) + xz_bytes + dbc_bytes);
      if (ig == 0) g2s_hint(st, h0p + ii * state_stride, (uint32_t)(EC * 64), bar, pol);
      g2s(st + XZ_OFF, xz0 + row * 2 * EC, xz_bytes, bar);
      g2s(st + D_OFF, a.dbc + row * a.KS * a.ldj, dbc_bytes, bar);
      ++ikk;
      if (++ig == NG) { ig = 0; ii += gridDim.x; }
    };
    // S5, last step, for the 8 rows of an iteration: partials added in ascending order, in place
    auto reduce_rows = [&](int kk) {   // whole warp
      const int s = kk & (NSL - 1);
      bar_wait(s_u32(&bars[s]), (uint32_t)((kk / NSL) & 1));
      float* d = reinterpret_cast<float*>(stages + s * SB + D_OFF);
      // (this warp is the only producer of `ready`: no divisions, every load of an element in flight before the adds)
      const int KS = a.KS, ldj = a.ldj, rl = KS * ldj;
      int t = 0, col = lane;
      while (col >= ldj) { col -= ldj; ++t; }
      for (int c = lane; c < G * ldj; c += 32) {
        float* p0 = d + t * rl + col;
        float x[KSMAX];
#pragma unroll
        for (int p = 0; p < KSMAX; ++p) x[p] = p < KS ? p0[p * ldj] : 0.0f;
        float v = x[0];
#pragma unroll
        for (int p = 1; p < KSMAX; ++p)
          if (p < KS) v += x[p];
        p0[0] = v;
        col += 32;
        while (col >= ldj) { col -= ldj; ++t; }
      }
      __syncwarp();
      if (lane == 0) asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(&bars[2 * NSL + s])) : "memory");
    };
    pdl_wait();
    if (lane == 0)
      for (int kk = 0; kk < NSL && kk < niter; ++kk) issue_next();
    const size_t img_row_tile = (size_t)(a.E >> 6) * (tc::NPA * tc::A_PLANE);
    uint8_t* yimg0 = a.y_img + (size_t)(e0 >> 6) * (tc::NPA * tc::A_PLANE);
    const int nblk = (EC >> 6) * 3;                // (64-channel block, piece) blocks of 1 KB per iteration
    reduce_rows(0);
    int g = 0;
    size_t i = blockIdx.x;
    for (int kk = 0; kk < niter; ++kk) {
      const int s = kk & (NSL - 1);
      uint8_t* st = stages + s * SB;
      if (kk + 1 < niter) reduce_rows(kk + 1);
      bar_wait(s_u32(&bars[NSL + s]), (uint32_t)((kk / NSL) & 1));       // the 8 steps of this iteration are done
      if (lane == 0) {
        const size_t row = i * a.T + (size_t)g * G;                       // a multiple of 8: one 8-row swizzle group
        uint8_t* ybase = yimg0 + (row >> 7) * img_row_tile + ((row & 127) >> 3) * 1024;
        for (int b = 0; b < nblk; ++b) {
          const int kt = b / 3, q = b - kt * 3;
          s2g(ybase + (size_t)kt * (tc::NPA * tc::A_PLANE) + (size_t)q * tc::A_PLANE, s_u32(st + Y_OFF + b * 1024), 1024u);
        }
        if (g == NG - 1) s2g_hint(h0p + i * state_stride, s_u32(st), (uint32_t)(EC * 64), pol);
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        if (ikk < niter) {
          asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");   // the stage has been read out
          issue_next();                                                   // iteration kk + NSL
        }
      }
      __syncwarp();
      if (++g == NG) { g = 0; i += gridDim.x; }
    }
    if (lane == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    return;
  }

  // ======================================================================= channel threads
  const int e = e0 + tid;
  float wr[RR ? RR : 1];
  if constexpr (RR > 0) {
#pragma unroll
    for (int r = 0; r < RR; ++r) wr[r] = a.W_dtT[(size_t)r * a.E + e];
  } else {
    for (int r = 0; r < a.R; ++r) wdt[r * EC + tid] = a.W_dtT[(size_t)r * a.E + e];
  }
  const float4 a0 = a.A4[e], a1 = a.A4[a.E + e], a2 = a.A4[2 * a.E + e], a3 = a.A4[3 * a.E + e];
  const float dsk = a.Dskip[e];
  const float bdt = a.b_dt[e];
  float4 h0, h1, h2, h3;
  int g = 0;
  const int rl = a.KS * a.ldj;
  // y pieces of step t: block (64-channel block, piece) = 8 rows of 128 bytes; row t, chunk (c ^ t), bf16 (tid & 7)
  const uint32_t yoff = (uint32_t)(((tid >> 6) * 3) * 1024 + (tid & 7) * 2);
  const int ychunk = (tid & 63) >> 3;
  for (int kk = 0; kk < niter; ++kk) {
    const int s = kk & (NSL - 1);
    uint8_t* st = stages + s * SB;
    bar_wait(s_u32(&bars[2 * NSL + s]), (uint32_t)((kk / NSL) & 1));
    float4* hs = reinterpret_cast<float4*>(st);
    if (g == 0) { h0 = hs[tid]; h1 = hs[EC + tid]; h2 = hs[2 * EC + tid]; h3 = hs[3 * EC + tid]; }
    const float* xz_s = reinterpret_cast<const float*>(st + XZ_OFF);
    const float* d = reinterpret_cast<const float*>(st + D_OFF);
#pragma unroll 1
    for (int t = 0; t < G; ++t) {
      const float x = xz_s[t * 2 * EC + tid];
      const float z = xz_s[t * 2 * EC + EC + tid];
      float yv = scan_channel_step<RR>(d + t * rl, a.R, wr, wdt + tid, EC, bdt, a0, a1, a2, a3, dsk, x, z, h0, h1, h2, h3);
      uint8_t* yp = st + Y_OFF + yoff + t * 128 + (((ychunk ^ t) & 7) << 4);
#pragma unroll
      for (int q = 0; q < 3; ++q) {
        *reinterpret_cast<uint16_t*>(yp + q * 1024) = (uint16_t)(__float_as_uint(yv) >> 16);
        yv = __fsub_rn(yv, tc::trunc_bf16(yv));
      }
    }
    if (g == NG - 1) { hs[tid] = h0; hs[EC + tid] = h1; hs[2 * EC + tid] = h2; hs[3 * EC + tid] = h3; }
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // y pieces (and the state) leave by bulk stores
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(s_u32(&bars[NSL + s])) : "memory");
    if (++g == NG) g = 0;
  }
}

}  // namespace boa
