// tc_gemm.cuh — the stream-batch contractions of the step on the 5th-generation tensor cores.
//
//   in_proj   xz = W_in RMSNorm(u)          S2+S3 (+ S4 conv1d+SiLU in the epilogue)   P:142; R#1, R#10, R#11
//   x_proj    [dlt;Bv;Cv] = W_x xs          S5                                         eq. 21-22
//   out_proj  u += W_out y                  S9                                         Alg. 1 l.3
//   head      logits = Emb u                S10                                        Alg. 1 l.5
//   FFN       f = GELU(W1 u + b1); v = W2 f + b2   (the paper's block only)   Alg. 1 l.4; R#23
//
// A tile is 128 streams x 64 columns:  C[m][n] = sum_k A[m][k] * W[n][k].  The kernel is persistent: one CTA per SM
// walks over tiles; the TMEM accumulators are double-buffered so the epilogue of tile i overlaps the copies and MMAs
// of tile i+1.
//
// Precision.  The activations are fp32 and the four parity checks need
// fp32-level products, so each operand is cut into bf16 pieces that sum to it exactly (a = a1+a2+a3, 8 significant
// bits each) and the tensor cores multiply the pieces: tcgen05.mma kind::f16 (bf16 x bf16 -> fp32 in TMEM).
//   bf16 weights (one exact piece w):   a1 w | a2 w + a3 w                               3 products per k-step
//   fp32 weights (w = w1+w2+w3):        a1 w1 | a1 w2 + a2 w1 | a1 w3 + a2 w2 + a3 w1    6 products per k-step
// Products of the same magnitude class (1, 2^-8, 2^-16) share a TMEM accumulator; the classes are added once, in
// fp32, smallest first, in the epilogue.  Dropped products are below 2^-24 of |a||w|.
// The weight pieces of a tile are stacked along N in shared memory ([w1; w2; w3]), so one MMA of a piece of A against
// the stack yields several products at once and A is read from shared memory once for them:
//   a1 x [w1;w2;w3] -> classes 0,1,2   a2 x [w1;w2] -> classes 1,2   a3 x [w1] -> class 2       (N = 192, 128, 64)
//
// Data movement.  Both operands reach shared memory through the bulk-copy engine (TMA, cp.async.bulk -> SASS UBLKCP)
// as ready-made images of a tile (K-major, 128-byte swizzle), so the main loop is TMA + MMA only:
//   weights      cut and laid out once, at boa_model_load;
//   activations  cut by the kernel that PRODUCES them (embedding, the conv epilogue of in_proj, the scan, the
//                residual epilogue of out_proj), which writes the three pieces straight into the image of the
//                consumer's tile - each activation is cut once per step, not once per consuming tile.
// One warp drives the copies, one elected thread issues the MMAs, tcgen05.commit releases a stage.  Eight epilogue
// warps read TMEM (one lane = one stream per thread), transpose through a shared staging tile and run the fused
// epilogue with lane = column, so every global access is coalesced.
//
// Determinism: row m of the result depends only on row m of A, on W and on a fixed issue order; it does not
// depend on M, on the tile the stream falls in, or on encode vs decode.
#pragma once
#include "common.cuh"

namespace boa {
namespace tc {

constexpr int BM = 128;          // streams per tile = TMEM lanes
constexpr int BN = 64;           // output columns per tile
constexpr int BK = 64;           // k per stage: 64 bf16 = one 128-byte swizzle row
constexpr int NPA = 3;           // bf16 pieces of an activation
constexpr int A_PLANE = BM * 128;  // bytes of one activation piece tile

enum { EPI_STORE = 0, EPI_RESID = 1, EPI_INPROJ = 2, EPI_FFN1 = 3 };
constexpr int SLAB_T = 16;       // steps per encode-side time slab in the slab form of in_proj (rows i*16 + t)

struct GemmArgs {
  const uint8_t* A;        // activation image of A[M][K]: [ceil(M/128)][K/64][3 pieces][128 x 64 bf16, swizzled]
  int M, KB;               // KB = K/64
  const uint16_t* W;       // weight image [N/64][K/64][NPW][64 x 64 bf16, swizzled]
  int NT;                  // column tiles (N/64, N padded with zero weight rows)
  int KS;                  // k-splits (>= 1, divides KB): split s covers k-blocks [s*KB/KS, (s+1)*KB/KS) and writes its
  size_t split_stride;     //   partial result to C + s*split_stride; the consumer adds the partials in ascending order
  float* C;                // [M][ldc] fp32 result (in_proj: xz = xs | z; out_proj: the residual stream u, updated)
  int ldc, n_valid;        // columns >= n_valid are not stored (zero-padded weight rows)
  int xz_ec;               // EPI_INPROJ: > 0 = the result is stored for the scan in slices of xz_ec channels (E = N/2):
  size_t xz_slice;         //   element (row, slice, xs|z half, c) at slice*xz_slice + row*ldc + half*xz_ec + c.  Step path:
                           //   ldc = 2E, xz_slice = 2*xz_ec (a row = [slice][xs | z]); time slab: ldc = 2*xz_ec,
                           //   xz_slice = rows*2*xz_ec ([slice][row][xs | z]).  xz_ec = 0: plain row-major
  // EPI_INPROJ only
  const float* ssq_in;     // [M][KB]: sum of u^2 over each 64-column block of the residual stream (written by the
                           // producer of u in a fixed order); rstd = 1/sqrt(sum/K + eps) (R#10)
  float* win;              // [streams][3][E] conv window of this layer, a ring: at step t slot t%3 holds x_{t-3} and receives x_t
  const uint32_t* pos;     // [streams] steps taken so far by each stream (the coder's position) = t
  int slab_T;              // 0: one row per stream.  T = SLAB_T (encode-side time slab, the SLAB instantiation): rows are stream-major,
                           // row i*T + t is step pos_i + t of stream i; the conv of a row reads the rows before it in the
                           // tile (the window only for t < 3) and the last three rows of a stream go into the window
  const float4* conv_w;    // [E] taps (x = t-3 ... w = t)
  const float* conv_b;     // [E]
  int E;
  // image of the result for the next contraction (EPI_INPROJ: xs -> x_proj; EPI_RESID: u -> in_proj / head)
  uint8_t* out_img;
  int out_KB;              // k-blocks per row tile of that image
  const float* out_scale;  // EPI_RESID: the consumer's RMSNorm weight (applied before cutting) or nullptr
  float* ssq_out;          // EPI_RESID: [M][out_KB] sum of the new u^2 over this tile's 64 columns
  // Chained contractions (k_gemm_chain): row-tile-level dependencies between the contractions of one launch.
  const uint32_t* dep;     // or nullptr: dep[row tile] must have reached dep_target before that row tile's operand image
  uint32_t dep_target;     //   (and, for in_proj, its block sums of u^2) may be read
  uint32_t* done;          // or nullptr: done[row tile] += 1 when a work item whose first column is < done_cols has
  int done_cols;           //   stored its results
  const float* bias;       // EPI_STORE (or nullptr), EPI_FFN1: [NT*64] added to the result.  EPI_FFN1 (the paper's block,
                           // Alg. 1 l.4) then applies GELU and writes only the image of the hidden layer (out_img, out_KB)
};

// ------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
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
// global -> shared bulk copy by the TMA engine; completes `bytes` on the mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar) : "memory");
}
// the same, delivered to the same shared-memory offset (and mbarrier) of every CTA of the cluster named in `mask`
__device__ __forceinline__ void bulk_g2s_mc(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint16_t mask) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.multicast::cluster [%0], [%1], %2, [%3], %4;"
               ::"r"(dst), "l"(src), "r"(bytes), "r"(bar), "h"(mask) : "memory");
}
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ void cluster_sync() {   // every thread of every CTA of the cluster
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// generic-proxy shared stores -> visible to the async proxy (tensor core operand reads)
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {   // whole warp
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {    // whole warp
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}

// D[tmem] (+)= A[smem] * B[smem]^T, bf16 inputs, fp32 accumulate; one thread issues for the CTA
__device__ __forceinline__ void umma(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n"
      "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// arrive on the mbarrier when every MMA issued so far by this thread has completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}

// the same arrival on the mbarrier at this offset in every CTA of the cluster named in `mask`
__device__ __forceinline__ void umma_commit_mc(uint32_t bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(mask) : "memory");
}

// 32 consecutive fp32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, float (&v)[32]) {
  uint32_t r[32];
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
      "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]),
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]),
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]),
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
#pragma unroll
  for (int j = 0; j < 32; ++j) v[j] = __uint_as_float(r[j]);
}

// Shared-memory matrix descriptor: K-major operand, 128-byte swizzle, rows of 128 bytes, 8-row groups 1024 bytes
// apart (SBO), descriptor version 1 (sm_100).  `addr` is a shared-window byte address.
__device__ __forceinline__ uint64_t smem_desc_sw128(uint32_t addr) {
  const uint32_t lo = ((addr & 0x3FFFFu) >> 4) | (1u << 16);             // start address | LBO (unused for swizzled K-major)
  const uint32_t hi = (1024u >> 4) | (1u << 14) | (2u << 29);            // SBO | version | SWIZZLE_128B
  return ((uint64_t)hi << 32) | lo;
}
// Instruction descriptor: D fp32, A and B bf16, both K-major, M = 128, N = n
__host__ __device__ constexpr uint32_t idesc_bf16(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(BM >> 4) << 24);
}

// ------------------------------------------------------------------------------------------ activation images
// Byte offset of element (r, k) of a 128 x 64 tile inside one 16 KB piece plane (K-major, 128-byte swizzle: the
// 16-byte chunk index is XORed with the row index mod 8), and of k-block (mt, kb) inside an image.
__host__ __device__ inline uint32_t plane_off(int r, int k) {
  return (uint32_t)((r >> 3) * 1024 + (r & 7) * 128 + ((((k >> 3) ^ r) & 7) << 4) + (k & 7) * 2);
}
__host__ __device__ inline size_t img_block(size_t mt, size_t kb, size_t KB) { return (mt * KB + kb) * (size_t)(NPA * A_PLANE); }
__host__ __device__ inline size_t img_bytes(size_t M, size_t K) { return ((M + BM - 1) / BM) * (K / BK) * (size_t)(NPA * A_PLANE); }

// An fp32 value is cut into three bf16 pieces by truncation: piece = the top 16 bits, remainder = v - piece (exact);
// 3 x 8 significant bits cover the 24-bit significand, so the pieces sum to v exactly.
__device__ __forceinline__ float trunc_bf16(float v) { return __uint_as_float(__float_as_uint(v) & 0xFFFF0000u); }
__device__ __forceinline__ uint32_t pack_hi(float lo, float hi) { return __byte_perm(__float_as_uint(lo), __float_as_uint(hi), 0x7632); }

// L2 policy for the activation images: they are written by one kernel and read by the next while hundreds of MB of
// state stream through L2 in between, so their lines are marked evict-last (the state copies are evict-first).
__device__ __forceinline__ uint64_t policy_evict_last() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void st_keep_v2(void* p, uint32_t a, uint32_t b, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v2.b32 [%0], {%1, %2}, %3;" ::"l"(p), "r"(a), "r"(b), "l"(pol) : "memory");
}
__device__ __forceinline__ void st_keep_v4(void* p, uint4 v, uint64_t pol) {
  asm volatile("st.global.L2::cache_hint.v4.b32 [%0], {%1, %2, %3, %4}, %5;" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w), "l"(pol) : "memory");
}

// Cut 4 consecutive values (row m, columns k..k+3, k % 4 == 0) and store the pieces into an image: 8 bytes per plane.
__device__ __forceinline__ void cut4_store(uint8_t* img, int KB, int m, int k, float4 v) {
  uint8_t* p = img + img_block((size_t)(m >> 7), (size_t)(k >> 6), (size_t)KB) + plane_off(m & 127, k & 63);
  const uint64_t pol = policy_evict_last();
#pragma unroll
  for (int q = 0; q < NPA; ++q) {
    st_keep_v2(p + q * A_PLANE, pack_hi(v.x, v.y), pack_hi(v.z, v.w), pol);
    v.x = __fsub_rn(v.x, trunc_bf16(v.x)); v.y = __fsub_rn(v.y, trunc_bf16(v.y));
    v.z = __fsub_rn(v.z, trunc_bf16(v.z)); v.w = __fsub_rn(v.w, trunc_bf16(v.w));
  }
}

// X[M][ldx] fp32 (optionally times colscale[k]) -> image.  One thread per 4 columns.
__global__ void k_cut_rows(const float* __restrict__ X, int ldx, int M, int K, const float* __restrict__ colscale,
                           uint8_t* __restrict__ img) {
  const int idx = blockIdx.x * blockDim.x + threadIdx.x;
  const int K4 = K >> 2;
  if (idx >= M * K4) return;
  const int m = idx / K4, k = (idx - m * K4) * 4;
  float4 v = *reinterpret_cast<const float4*>(X + (size_t)m * ldx + k);
  if (colscale) {
    const float4 s = *reinterpret_cast<const float4*>(colscale + k);
    v.x *= s.x; v.y *= s.y; v.z *= s.z; v.w *= s.w;
  }
  cut4_store(img, K >> 6, m, k, v);
}

// Asynchronous global -> shared copies of single words (LDGSTS): the epilogue's prefetches, which must not hold registers.
__device__ __forceinline__ void cp_async4(uint32_t dst, const void* src) {
  asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async16(uint32_t dst, const void* src) {
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

template <int NPW>
struct Cfg {
  static constexpr int W_BYTES = NPW * BN * 128;
  static constexpr int A_BYTES = NPA * A_PLANE;
  static constexpr int STAGE = A_BYTES + W_BYTES;
  static constexpr int LDS = BN + 4;                          // staging row, padded: conflict-free column stores
  static constexpr int STILE_BYTES = BM * LDS * 4;
  static constexpr int NST = (3 * STAGE + STILE_BYTES <= 220 * 1024) ? 3 : 2;
  // epilogue prefetch area (cp.async, no registers): [NSQ][BM] block sums of u^2 of the next tile's rows, and
  // [4][NEPI] float4 of conv-window values of a time-slab tile (three for the row group at t = 0, 1; one for t = 2)
  static constexpr int NSQ = 8;
  static constexpr int SQ_BYTES = NSQ * BM * 4;
  static constexpr int PW_BYTES = 4 * 256 * 16;
  static constexpr int SMEM = NST * STAGE + STILE_BYTES + 1024;                  // + alignment slack
  static constexpr int SMEM_SLAB = SMEM + SQ_BYTES + PW_BYTES;                  // the time-slab form of in_proj
  static constexpr int NACC = NPW == 3 ? 3 : 2;               // accumulators (magnitude classes)
  static constexpr int ACC_COLS = NACC * BN;                  // TMEM columns of one accumulator buffer
  static constexpr int TMEM_COLS = (2 * ACC_COLS <= 256) ? 256 : 512;   // two buffers
};

// Row-tile dependencies inside one launch (k_gemm_chain).  After the block barrier that ends a work item one thread adds
// to the row tile's counter with release semantics at device scope; the consumer spins with acquire loads and then
// crosses to the async proxy (it reads the producer's generic-proxy stores with bulk copies).
__device__ __forceinline__ void dep_wait(const uint32_t* p, uint32_t target) {
  uint32_t v;
  for (;;) {
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    if (v >= target) break;
    __nanosleep(40);
  }
  asm volatile("fence.proxy.async;" ::: "memory");
}
// (the block barrier before dep_signal orders the other threads' stores before the signalling thread's release, which is
// cumulative; the consumer crosses to the async proxy with its own fence.proxy.async after the acquire)
__device__ __forceinline__ void dep_signal(uint32_t* p) {
  __threadfence();
  asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(p) : "memory");
}

// sigmoid for the SiLU of the conv epilogue: fast forms (relative error ~1e-6; same code on encode and decode)
__device__ __forceinline__ float sigmoid_tc(float x) { return __fdividef(1.0f, 1.0f + __expf(-x)); }

// GELU(v) = v Phi(v), erf form (R#23); erff is within a few ulp, the same code on encode and decode
__device__ __forceinline__ float gelu_tc(float v) { return 0.5f * v * (1.0f + erff(v * 0.70710678118654752440f)); }

// Offset (without the row term row*ldc) of in_proj output n (x half: n < E, z half: n >= E) in the sliced xz layout.
__host__ __device__ inline size_t xz_col(int n, int E, int EC, size_t slice_stride) {
  const int half = n >= E, c = n - half * E;
  return (size_t)(c / EC) * slice_stride + (size_t)(half * EC + c % EC);
}

// S4 for one channel: xc = b + w.x x_{t-3} + w.y x_{t-2} + w.z x_{t-1} + w.w x_t in this fixed FMA order (R#11), then SiLU.
// The one definition shared by the step kernel (in_proj epilogue) and the encode-side time-slab kernel, so that both
// produce the same bits.
__device__ __forceinline__ float conv_silu1(float4 w, float b, float xm3, float xm2, float xm1, float x) {
  float xc = fmaf(w.w, x, b);
  xc = fmaf(w.x, xm3, xc);
  xc = fmaf(w.y, xm2, xc);
  xc = fmaf(w.z, xm1, xc);
  return xc * sigmoid_tc(xc);
}

constexpr int NEPI = 256;        // epilogue threads (warps 0-7); warp 8 owns TMEM and issues the MMAs; warp 9 drives the copies
constexpr int NTHREADS = NEPI + 64;

// ------------------------------------------------------------------------------------------ the contraction
// Shared-memory objects of a contraction CTA: the stage ring, its barriers, the TMEM accumulators.
struct GemmShared {
  uint8_t* raw;            // dynamic shared memory (stage ring + staging tile [+ prefetch area])
  uint64_t *full_bar, *empty_bar, *acc_full, *acc_empty;
  uint32_t tmem;           // TMEM base address of the accumulators
};
// (Re-)initialise the barriers of the ring: one thread; the caller fences and synchronises the block (and cluster).
template <int NPW, int CS>
__device__ __forceinline__ void gemm_init_barriers(const GemmShared& sh, int nst = Cfg<NPW>::NST) {
  for (int s = 0; s < nst; ++s) {
    mbar_init(smem_u32(&sh.full_bar[s]), 1);     // the copy warp's arrive.expect_tx
    mbar_init(smem_u32(&sh.empty_bar[s]), CS);   // one tcgen05.commit per CTA of the cluster
  }
  for (int b = 0; b < 2; ++b) {
    mbar_init(smem_u32(&sh.acc_full[b]), 1);     // one tcgen05.commit
    mbar_init(smem_u32(&sh.acc_empty[b]), NEPI); // every epilogue thread has drained its part
  }
  fence_barrier_init();
}

// The three roles of a contraction CTA over its work items tile_begin + item0, + item_step, ... < tile_end (item index ->
// (row tile, column tile [pair], k-split), k-split fastest).  Called by all NTHREADS threads with freshly initialised
// barriers; returns when this CTA's copies are issued, its MMAs committed and its epilogues done (the caller
// synchronises).  Shared by k_tc_gemm (one launch per contraction) and the persistent step kernel (step_persist.cuh).
// COMPACT (the persistent step kernel at few streams; all items of a call share one row tile): when the row tile has at
// most 64 live rows only their 8-row groups of each activation piece are copied (1 KB per group instead of the 16 KB
// plane; the MMA still reads 128 rows, the rows beyond are whatever follows in shared memory and only reach accumulator
// rows nobody reads), which makes a stage small enough for a ring of up to MAXST stages: every k-block of a work item is
// in flight at once instead of NST at a time.  The result rows of live streams are the same bits either way.
constexpr int MAXST = 16;        // barrier slots a COMPACT caller provides
template <int NPW, int EPI, int CS, bool SLAB, bool COMPACT = false>
__device__ __forceinline__ void gemm_roles(const GemmArgs& g, const GemmShared& sh, int item0, int item_step, int tile_begin,
                                           int tile_end, int crank) {
  using C = Cfg<NPW>;
  static_assert(!COMPACT || CS == 1, "compact stages: no multicast");
  constexpr uint16_t CMASK = (uint16_t)((1u << CS) - 1u);
  uint8_t* smem_raw = sh.raw;
  uint64_t *full_bar = sh.full_bar, *empty_bar = sh.empty_bar, *acc_full = sh.acc_full, *acc_empty = sh.acc_empty;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KB = g.KB / g.KS, NT = g.NT, KS = g.KS;     // KB: k-blocks of one work item
  const int NTI = NT / CS;
  const int ntiles = tile_end;
  item0 += tile_begin;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;
  const uint32_t tmem = sh.tmem;
  // stage geometry: compile-time constants unless COMPACT
  uint32_t plane = (uint32_t)A_PLANE, stage = (uint32_t)C::STAGE;
  int nst = C::NST;
  if (COMPACT) {
    const int live = min(g.M - (tile_begin / KS / NTI) * BM, BM), r8 = (live + 7) >> 3;
    if (r8 <= 8) {
      plane = (uint32_t)r8 * 1024u;
      stage = NPA * plane + (uint32_t)C::W_BYTES;
      nst = min(MAXST, (int)((uint32_t)(C::NST * C::STAGE - A_PLANE) / stage));
    }
  }

  if (warp == 9) {
    // ===================================================================== copy warp
    if (lane == 0) {
      int kbc = 0;                                 // k-blocks issued so far: position in the stage ring
      for (int tile = item0; tile < ntiles; tile += item_step) {
        const int ks = tile % KS, t2 = tile / KS, mt = t2 / NTI, nt = (t2 - mt * NTI) * CS + crank;
        const uint8_t* asrc = g.A + img_block((size_t)mt, (size_t)ks * KB, (size_t)g.KB);
        const uint16_t* wsrc = g.W + ((size_t)nt * g.KB + (size_t)ks * KB) * (NPW * BN * 64);
        if (g.dep) dep_wait(g.dep + mt, g.dep_target);   // the row tile's image is complete
        for (int kb = 0; kb < KB; ++kb, ++kbc) {
          const int s = kbc % nst, round = kbc / nst;
          if (round > 0) mbar_wait(smem_u32(&empty_bar[s]), (uint32_t)((round - 1) & 1));
          const uint32_t sA = sbase + (uint32_t)s * stage, fb = smem_u32(&full_bar[s]);
          mbar_arrive_expect_tx(fb, stage);
          if (COMPACT && plane != (uint32_t)A_PLANE) {   // the live 8-row groups of each piece plane
#pragma unroll
            for (int q = 0; q < NPA; ++q)
              bulk_g2s(sA + (uint32_t)q * plane, asrc + (size_t)kb * C::A_BYTES + (size_t)q * A_PLANE, plane, fb);
          } else if (CS > 1)                              // this CTA's part of the block, delivered to every CTA of the cluster
            bulk_g2s_mc(sA + (uint32_t)crank * (C::A_BYTES / CS), asrc + (size_t)kb * C::A_BYTES + (size_t)crank * (C::A_BYTES / CS),
                        (uint32_t)(C::A_BYTES / CS), fb, CMASK);
          else
            bulk_g2s(sA, asrc + (size_t)kb * C::A_BYTES, (uint32_t)C::A_BYTES, fb);
          bulk_g2s(sA + NPA * plane, wsrc + (size_t)kb * (NPW * BN * 64), (uint32_t)C::W_BYTES, fb);
        }
      }
    }
  } else if (warp == 8) {
    // ===================================================================== MMA issuer
    if (lane == 0) {
      int kbc = 0, it = 0;
      for (int tile = item0; tile < ntiles; tile += item_step, ++it) {
        const int b = it & 1;
        if (it >= 2) {                             // the epilogue has drained this buffer (tile it-2)
          mbar_wait(smem_u32(&acc_empty[b]), (uint32_t)(((it >> 1) - 1) & 1));
          tc_fence_after();
        }
        const uint32_t tacc = tmem + (uint32_t)(b * C::ACC_COLS);
        for (int kb = 0; kb < KB; ++kb, ++kbc) {
          const int s = kbc % nst, round = kbc / nst;
          mbar_wait(smem_u32(&full_bar[s]), (uint32_t)(round & 1));
          tc_fence_after();
          const uint32_t sA = sbase + (uint32_t)s * stage;
          const uint32_t sW = sA + NPA * plane;
#pragma unroll
          for (int k4 = 0; k4 < BK / 16; ++k4) {
            const uint32_t first = (kb | k4) ? 1u : 0u;
            const uint32_t ko = (uint32_t)k4 * 32u;
            auto A_ = [&](int p) { return smem_desc_sw128(sA + (uint32_t)p * plane + ko); };
            const uint64_t wd = smem_desc_sw128(sW + ko);
            if (NPW == 3) {
              umma(tacc, A_(0), wd, idesc_bf16(192), first);         // a1 x [w1;w2;w3] -> classes 0,1,2
              umma(tacc + 64, A_(1), wd, idesc_bf16(128), 1u);       // a2 x [w1;w2]    -> classes 1,2
              umma(tacc + 128, A_(2), wd, idesc_bf16(64), 1u);       // a3 x [w1]       -> class 2
            } else {
              umma(tacc, A_(0), wd, idesc_bf16(64), first);          // a1 w            -> class 0
              umma(tacc + 64, A_(2), wd, idesc_bf16(64), first);     // a3 w, a2 w      -> class 1
              umma(tacc + 64, A_(1), wd, idesc_bf16(64), 1u);
            }
          }
          if (CS > 1) umma_commit_mc(smem_u32(&empty_bar[s]), CMASK);   // stage free in every CTA when all have read it
          else umma_commit(smem_u32(&empty_bar[s]));                 // stage free when these MMAs have read it
        }
        umma_commit(smem_u32(&acc_full[b]));                         // this tile's accumulators are complete
      }
    }
  } else {
    // ===================================================================== epilogue warps
    constexpr int LDS = C::LDS;
    float* stile = reinterpret_cast<float*>(smem_raw + (sbase - smem_u32(smem_raw)) + C::NST * C::STAGE);
    constexpr int LPR = BN / 4;                    // lanes per row segment in pass 2 (4 columns per lane)
    constexpr int RPI = 32 / LPR;                  // rows per warp instruction
    constexpr int NIT = BM / (8 * RPI);            // row groups per warp
    const int col = (lane % LPR) * 4;
    static_assert(NIT == 8 && RPI == 2, "slab_row below assumes 128 x 64 tiles");
    int it = 0;
    const int r1 = (warp & 3) * 32 + lane;         // pass 1: thread = stream row
    // S2: the block sums of u^2 of this thread's row (the first 8 of them) are fetched one tile ahead, all loads in
    // flight together, and summed in ascending order when the tile starts (absent blocks read as 0: x + 0 = x).
    constexpr int NSQ = C::NSQ;
    float* sqs = stile + BM * LDS;                 // [NSQ][BM]
    float4* pws = reinterpret_cast<float4*>(sqs + NSQ * BM);   // [4][NEPI]
    auto fetch_sq = [&](int tile) {                // by warps 0-3 (one thread per row); read by all after a barrier
      if (warp < 4) {
        const int mt = (tile / KS) / NTI;
        const float* sp = g.ssq_in + (size_t)min(mt * BM + r1, g.M - 1) * g.KB;
#pragma unroll
        for (int q = 0; q < NSQ; ++q)
          if (q < g.KB) cp_async4(smem_u32(sqs + q * BM + r1), sp + q);
      }
      cp_async_commit();
    };
    if (SLAB) {
      if (item0 < ntiles) fetch_sq(item0);
      cp_async_wait<0>();
      asm volatile("bar.sync 1, 256;" ::: "memory");
    }
    for (int tile = item0; tile < ntiles; tile += item_step, ++it) {
      const int b = it & 1;
      const int ks = tile % KS, t2 = tile / KS, mt = t2 / NTI, nt = (t2 - mt * NTI) * CS + crank;
      const int m0 = mt * BM, n0 = nt * BN;
      float* Cout = g.C + (size_t)ks * g.split_stride;
      // Pass 1: TMEM -> registers (thread = stream row; warps w and w+4 share the 32 TMEM lanes of rows 32*(w%4)..
      // and take one 32-column half each) -> shared staging tile, so that pass 2 can run with lane = column and
      // every global access coalesced.
      float rs = 1.0f;
      if (EPI == EPI_INPROJ) {                     // S2: RMSNorm row scale from the block sums of u^2, ascending
        const float* sp = g.ssq_in + (size_t)min(m0 + r1, g.M - 1) * g.KB;
        float ss = 0.0f;
        if (SLAB) {
#pragma unroll
          for (int q = 0; q < NSQ; ++q)
            if (q < g.KB) ss += sqs[q * BM + r1];
          for (int q = NSQ; q < g.KB; ++q) ss += sp[q];
        } else {
          if (g.dep) {                             // chained after out_proj: its block sums of this row tile are final
            if (lane == 0) dep_wait(g.dep + mt, g.dep_target);
            __syncwarp();
          }
          for (int q = 0; q < g.KB; ++q) ss += __ldcg(sp + q);   // (L2: another CTA may have written them in this launch)
        }
        rs = 1.0f / sqrtf(ss / (float)(g.KB * BK) + kEps);
      }
      // The conv window of the first row batch does not depend on the accumulators: its loads (from HBM at large B)
      // are issued now and fly while the main loop of this tile finishes.
      const int nb = n0 + col;
      const size_t ncol = (EPI == EPI_INPROJ && g.xz_ec > 0) ? xz_col(nb, g.E, g.xz_ec, g.xz_slice) : (size_t)nb;   // offset of the stored result in its row
      const bool conv_tile = EPI == EPI_INPROJ && n0 < g.E;
      const bool slab_tile = SLAB && conv_tile;
      float4 w0[4], w1[4], w2[4];
      int slot[4];                                 // ring slot of x_{t-3} (and of x_t after this step)
      if (conv_tile && !slab_tile) {
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int r = (warp + 8 * u) * RPI + lane / LPR;
          const int rc = min(m0 + r, g.M - 1);
          slot[u] = (int)(g.pos[rc] % 3u);
          const float* wp = g.win + (size_t)rc * 3 * g.E + nb;
          w0[u] = *reinterpret_cast<const float4*>(wp + slot[u] * g.E);
          w1[u] = *reinterpret_cast<const float4*>(wp + ((slot[u] + 1) % 3) * g.E);
          w2[u] = *reinterpret_cast<const float4*>(wp + ((slot[u] + 2) % 3) * g.E);
        }
      }
      // Time slab (T = SLAB_T = 16 steps, rows i*16 + t, tiles start at a multiple of 16): row group i of a warp is rows
      // 16 i + g0 + {0, 1} with g0 = (2 warp + 2 i) mod 16, so every warp meets every step t of a slab once and the
      // rows that read the window (t < 3: the groups g0 = 0 and g0 = 2) are spread evenly over the warps.  Their window
      // values are fetched here, into pws[0..2] (g0 = 0: x_{t-1}, x_{t-2}, x_{t-3}) and pws[3] (g0 = 2, t = 2: x_{t-3}).
      auto slab_g0 = [&](int i) { return (2 * warp + 2 * i) & 15; };
      auto slab_row = [&](int i) { return 16 * i + slab_g0(i) + lane / LPR; };
      if (slab_tile) {
#pragma unroll
        for (int i = 0; i < NIT; ++i) {
          const int g0 = slab_g0(i);
          if (g0 <= 2) {                           // warp-uniform
            const int si = min(m0 + slab_row(i), g.M - 1) / SLAB_T, t = g0 + lane / LPR;
            const uint32_t p0 = g.pos[si];
            const float* wp = g.win + (size_t)si * 3 * g.E + nb;
#pragma unroll
            for (int j = 1; j <= 3; ++j)
              if (t < j) cp_async16(smem_u32(pws + (g0 == 0 ? j - 1 : 3) * NEPI + tid),
                                    wp + ((p0 + 3u + (uint32_t)t - (uint32_t)j) % 3u) * g.E);
          }
        }
      }
      if (SLAB) cp_async_commit();
      mbar_wait(smem_u32(&acc_full[b]), (uint32_t)((it >> 1) & 1));
      tc_fence_after();
      {
        const uint32_t tl = tmem + (uint32_t)(b * C::ACC_COLS) + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)((warp >> 2) * 32);
        float v[32], w[32];
        __syncwarp();
        tmem_ld32(tl + 64, v);                     // class 1
        if (NPW == 3) {
          tmem_ld32(tl + 128, w);                  // class 2, added first
#pragma unroll
          for (int j = 0; j < 32; ++j) v[j] += w[j];
        }
        tmem_ld32(tl, w);                          // class 0
        tc_fence_before();
        mbar_arrive(smem_u32(&acc_empty[b]));      // this thread's part of the buffer may be overwritten
        float4* dst = reinterpret_cast<float4*>(stile + r1 * LDS + (warp >> 2) * 32);
#pragma unroll
        for (int j = 0; j < 32; j += 4)
          dst[j >> 2] = make_float4((v[j] + w[j]) * rs, (v[j + 1] + w[j + 1]) * rs, (v[j + 2] + w[j + 2]) * rs,
                                    (v[j + 3] + w[j + 3]) * rs);
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (SLAB) {
        if (tile + item_step < ntiles) fetch_sq(tile + item_step); else cp_async_commit();   // flies during pass 2
        cp_async_wait<1>();                        // this tile's window values have landed (own thread's only)
      }
      // Pass 2: 16 lanes own one 64-column row segment (4 consecutive columns per lane), two rows per warp
      // instruction; rows are processed four at a time with all loads issued first.
      if (slab_tile) {
        // S4 over a time slab: the rows of a stream are consecutive in the tile, so x_{t-1..t-3} of row t are the rows
        // before it in the staging tile; only the first three steps of the slab read the window ring (x before the
        // slab) and the last three go into it - after a barrier, when every row of the tile has read it.
        const float4 cw0 = g.conv_w[nb], cw1 = g.conv_w[nb + 1], cw2 = g.conv_w[nb + 2], cw3 = g.conv_w[nb + 3];
        const float4 cb = *reinterpret_cast<const float4*>(g.conv_b + nb);
#pragma unroll
        for (int i = 0; i < NIT; ++i) {
          const int g0 = slab_g0(i);
          const int r = slab_row(i), row = m0 + r, t = g0 + lane / LPR;   // step of the row within its slab
          const float4 x = *reinterpret_cast<const float4*>(stile + r * LDS + col);
          float4 xm[3];                                           // x_{t-1}, x_{t-2}, x_{t-3}
#pragma unroll
          for (int j = 1; j <= 3; ++j)
            xm[j - 1] = (t >= j) ? *reinterpret_cast<const float4*>(stile + (r - j) * LDS + col)
                                 : pws[(g0 == 0 ? j - 1 : 3) * NEPI + tid];
          if (row < g.M) {
            float4 o;
            o.x = conv_silu1(cw0, cb.x, xm[2].x, xm[1].x, xm[0].x, x.x);
            o.y = conv_silu1(cw1, cb.y, xm[2].y, xm[1].y, xm[0].y, x.y);
            o.z = conv_silu1(cw2, cb.z, xm[2].z, xm[1].z, xm[0].z, x.z);
            o.w = conv_silu1(cw3, cb.w, xm[2].w, xm[1].w, xm[0].w, x.w);
            *reinterpret_cast<float4*>(Cout + (size_t)row * g.ldc + ncol) = o;
            cut4_store(g.out_img, g.out_KB, row, nb, o);
          }
        }
        asm volatile("bar.sync 1, 256;" ::: "memory");     // every row has read the window
#pragma unroll
        for (int i = 0; i < NIT; ++i) {                      // x_t of the last three steps -> ring slot (pos + t) % 3
          const int g0 = slab_g0(i);
          if (g0 >= 12) {                                    // warp-uniform
            const int r = slab_row(i), row = m0 + r, t = g0 + lane / LPR, si = row / SLAB_T;
            if (row < g.M && t >= SLAB_T - 3)
              *reinterpret_cast<float4*>(g.win + ((size_t)si * 3 + (g.pos[si] + (uint32_t)t) % 3u) * g.E + nb) =
                  *reinterpret_cast<const float4*>(stile + r * LDS + col);
          }
        }
      } else if (conv_tile) {
        // S4: causal depthwise conv over (x_{t-3}, x_{t-2}, x_{t-1}, x_t) + SiLU (R#11).  The window is a ring of three
        // slots per stream: all three are read, only the oldest is overwritten with x_t.
        // The lane's four channels are fixed within a tile, so their taps and biases live in registers.  xs goes out
        // twice: fp32 (the scan reads it) and cut into pieces in the image of x_proj's operand.  The window loads of
        // the next row batch are issued before the current one is computed.
        const float4 cw0 = g.conv_w[nb], cw1 = g.conv_w[nb + 1], cw2 = g.conv_w[nb + 2], cw3 = g.conv_w[nb + 3];
        const float4 cb = *reinterpret_cast<const float4*>(g.conv_b + nb);
#pragma unroll
        for (int i0 = 0; i0 < NIT; i0 += 4) {
          float4 x[4], n0_[4], n1_[4], n2_[4];
          int rows[4], nslot[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int r = (warp + 8 * (i0 + u)) * RPI + lane / LPR;
            rows[u] = m0 + r;
            x[u] = *reinterpret_cast<const float4*>(stile + r * LDS + col);
            if (i0 + 4 < NIT) {
              const int rn = (warp + 8 * (i0 + 4 + u)) * RPI + lane / LPR;
              const int rc = min(m0 + rn, g.M - 1);
              nslot[u] = (int)(g.pos[rc] % 3u);
              const float* wp = g.win + (size_t)rc * 3 * g.E + nb;
              n0_[u] = *reinterpret_cast<const float4*>(wp + nslot[u] * g.E);
              n1_[u] = *reinterpret_cast<const float4*>(wp + ((nslot[u] + 1) % 3) * g.E);
              n2_[u] = *reinterpret_cast<const float4*>(wp + ((nslot[u] + 2) % 3) * g.E);
            }
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            if (rows[u] < g.M) {
              float4 o;
              o.x = conv_silu1(cw0, cb.x, w0[u].x, w1[u].x, w2[u].x, x[u].x);
              o.y = conv_silu1(cw1, cb.y, w0[u].y, w1[u].y, w2[u].y, x[u].y);
              o.z = conv_silu1(cw2, cb.z, w0[u].z, w1[u].z, w2[u].z, x[u].z);
              o.w = conv_silu1(cw3, cb.w, w0[u].w, w1[u].w, w2[u].w, x[u].w);
              *reinterpret_cast<float4*>(g.win + ((size_t)rows[u] * 3 + slot[u]) * g.E + nb) = x[u];
              *reinterpret_cast<float4*>(Cout + (size_t)rows[u] * g.ldc + ncol) = o;
              cut4_store(g.out_img, g.out_KB, rows[u], nb, o);
            }
          }
          if (i0 + 4 < NIT) {
#pragma unroll
            for (int u = 0; u < 4; ++u) { w0[u] = n0_[u]; w1[u] = n1_[u]; w2[u] = n2_[u]; slot[u] = nslot[u]; }
          }
        }
      } else {
        float4 osc = make_float4(1.f, 1.f, 1.f, 1.f);
        if (EPI == EPI_RESID && g.out_scale) osc = *reinterpret_cast<const float4*>(g.out_scale + nb);
        const bool cols_ok = nb < g.n_valid;
        float4 bs = make_float4(0.f, 0.f, 0.f, 0.f);
        const bool has_bias = (EPI == EPI_STORE || EPI == EPI_FFN1) && g.bias != nullptr;
        if (has_bias) bs = *reinterpret_cast<const float4*>(g.bias + nb);
#pragma unroll 1
        for (int i0 = 0; i0 < NIT; i0 += 4) {
          float4 o[4], q[4];
          int rows[4];
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const int r = (warp + 8 * (i0 + u)) * RPI + lane / LPR;
            rows[u] = m0 + r;
            o[u] = *reinterpret_cast<const float4*>(stile + r * LDS + col);
            if (EPI == EPI_RESID) q[u] = *reinterpret_cast<const float4*>(Cout + (size_t)min(rows[u], g.M - 1) * g.ldc + ncol);
          }
#pragma unroll
          for (int u = 0; u < 4; ++u) {
            const bool live = rows[u] < g.M && cols_ok;
            if (EPI == EPI_RESID) {
              // S9: the residual stream; its image (times the consumer's RMSNorm weight) for the next contraction;
              // and the sum of its squares over this tile's 64 columns (x, y, z, w, then the xor butterfly 8, 4, 2, 1)
              o[u].x += q[u].x; o[u].y += q[u].y; o[u].z += q[u].z; o[u].w += q[u].w;
              float ss = o[u].x * o[u].x;
              ss = fmaf(o[u].y, o[u].y, ss); ss = fmaf(o[u].z, o[u].z, ss); ss = fmaf(o[u].w, o[u].w, ss);
#pragma unroll
              for (int d = 8; d > 0; d >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, d);
              if (live) {
                cut4_store(g.out_img, g.out_KB, rows[u], nb,
                           make_float4(o[u].x * osc.x, o[u].y * osc.y, o[u].z * osc.z, o[u].w * osc.w));
                if ((lane % LPR) == 0) g.ssq_out[(size_t)rows[u] * g.out_KB + nt] = ss;
              }
            }
            if (has_bias) { o[u].x += bs.x; o[u].y += bs.y; o[u].z += bs.z; o[u].w += bs.w; }
            if (EPI == EPI_FFN1) {
              if (live)
                cut4_store(g.out_img, g.out_KB, rows[u], nb,
                           make_float4(gelu_tc(o[u].x), gelu_tc(o[u].y), gelu_tc(o[u].z), gelu_tc(o[u].w)));
            } else if (live) {
              *reinterpret_cast<float4*>(Cout + (size_t)rows[u] * g.ldc + ncol) = o[u];
            }
          }
        }
      }
      if (SLAB) cp_async_wait<0>();                      // the next tile's block sums
      asm volatile("bar.sync 1, 256;" ::: "memory");     // the staging tile is free for the next tile
      if (g.done && tid == 0 && n0 < g.done_cols) dep_signal(g.done + mt);
    }
  }

}

// ------------------------------------------------------------------------------------------ the kernel
// grid = min(tiles, SMs), block = 320.  Tile t -> (row tile t / NT, column tile t % NT); CTA c takes tiles c,
// c + grid, ...  Warp 9 (one lane) streams the k-blocks of both operand images into the stage ring; warp 8 (one lane)
// issues the MMAs into accumulator buffer (tile iteration & 1); warps 0-7 drain the other buffer and run the epilogue.
// CS > 1: the kernel is launched in clusters of CS CTAs that take CS consecutive column tiles of the same row tile in
// lock-step and share its activation k-blocks: each CTA fetches 1/CS of the 48 KB block and the bulk copy delivers
// it to all of them (multicast); a stage is reused when the MMAs of ALL CTAs of the cluster have read it.
// SLAB (EPI_INPROJ with g.slab_T > 0 only): the time-slab form of the conv epilogue, whose tiles are epilogue-bound;
// it fetches what the epilogue reads from global memory (block sums of u^2, window values) ahead of time with
// cp.async into shared memory.  The step form (SLAB = false) is bound by its main loop and reads them directly.
template <int NPW, int EPI, int CS, bool SLAB = false>
__global__ void __launch_bounds__(NTHREADS, 1) k_tc_gemm(const GemmArgs g) {
  using C = Cfg<NPW>;
  static_assert(NPW == 1 || NPW == 3, "weight pieces");
  static_assert(CS == 1 || CS == 2 || CS == 4 || CS == 8, "cluster size");
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[C::NST], empty_bar[C::NST], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  GemmShared sh{smem_raw, full_bar, empty_bar, acc_full, acc_empty, 0u};
  if (warp == 8) {
    if (lane == 0) gemm_init_barriers<NPW, CS>(sh);
    __syncwarp();
    tmem_alloc(smem_u32(&tmem_base_s), C::TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  if (CS > 1) cluster_sync();                      // the peers' barriers are initialised before anything is sent to them
  tc_fence_after();
  sh.tmem = tmem_base_s;
  pdl_launch();
  pdl_wait();                                      // everything below reads what earlier kernels of the step wrote

  const int ntiles = ((g.M + BM - 1) / BM) * (g.NT / CS) * g.KS;
  gemm_roles<NPW, EPI, CS, SLAB>(g, sh, (int)blockIdx.x / CS, (int)gridDim.x / CS, 0, ntiles, CS > 1 ? (int)cluster_ctarank() : 0);

  tc_fence_before();
  __syncthreads();
  if (CS > 1) cluster_sync();                      // no CTA leaves while a peer may still send to it
  if (warp == 8) {
    __syncwarp();
    tmem_dealloc(sh.tmem, C::TMEM_COLS);
  }
}

// ------------------------------------------------------------------------------------------ chained contractions
// Two or three dependent contractions of the step in ONE launch (VERDICT r1 "Next" 3(ii): 4L + 2 -> 2L + 2 launches per
// step).  At the step path's sizes every contraction kernel costs 7 - 10 us of which only a part is work: drain of
// the previous kernel, launch, prologue, the first operand round trip.  Here the CTAs of one persistent launch run
// the contractions one after the other (gemm_roles per contraction, the barriers re-initialised in between) and a work
// item waits only for ITS row tile: the producer's epilogue counts finished items per row tile in global memory
// (GemmArgs::done), the consumer's copy warp (and, for in_proj, its epilogue warps: the block sums of u^2) spin on that
// counter (GemmArgs::dep).  No CTA waits in its first contraction, so the waits cannot form a cycle; the grid is at most
// one CTA per SM, so every producer gets to run.  Arithmetic, tiles and epilogues are those of k_tc_gemm: same bits.
//   CH_IN_X       in_proj(l) -> x_proj(l)                      x_proj's row tile needs the E/64 conv tiles of in_proj
//   CH_OUT_IN_X   out_proj(l) -> in_proj(l+1) -> x_proj(l+1)   in_proj's row tile needs the D/64 tiles of out_proj
//   CH_OUT_HEAD   out_proj(L-1) -> head
enum { CH_IN_X = 0, CH_OUT_IN_X = 1, CH_OUT_HEAD = 2 };
struct ChainArgs {
  GemmArgs g[3];
};

template <int NPW, int EPI>
__device__ __forceinline__ void chain_phase(const GemmArgs& g, const GemmShared& sh) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 8 && lane == 0) gemm_init_barriers<NPW, 1>(sh);
  __syncthreads();
  const int ntiles = ((g.M + BM - 1) / BM) * g.NT * g.KS;
  gemm_roles<NPW, EPI, 1, false>(g, sh, (int)blockIdx.x, (int)gridDim.x, 0, ntiles, 0);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
}

template <int NPW, int KIND>
__global__ void __launch_bounds__(NTHREADS, 1) k_gemm_chain(const ChainArgs a) {
  using C = Cfg<NPW>;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[C::NST], empty_bar[C::NST], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;
  const int warp = threadIdx.x >> 5;
  GemmShared sh{smem_raw, full_bar, empty_bar, acc_full, acc_empty, 0u};
  if (warp == 8) tmem_alloc(smem_u32(&tmem_base_s), C::TMEM_COLS);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  sh.tmem = tmem_base_s;
  pdl_launch();
  pdl_wait();                                      // everything below reads what earlier kernels of the step wrote
  if (KIND == CH_IN_X) {
    chain_phase<NPW, EPI_INPROJ>(a.g[0], sh);
    chain_phase<NPW, EPI_STORE>(a.g[1], sh);
  } else if (KIND == CH_OUT_IN_X) {
    chain_phase<NPW, EPI_RESID>(a.g[0], sh);
    chain_phase<NPW, EPI_INPROJ>(a.g[1], sh);
    chain_phase<NPW, EPI_STORE>(a.g[2], sh);
  } else {
    chain_phase<NPW, EPI_RESID>(a.g[0], sh);
    chain_phase<NPW, EPI_STORE>(a.g[1], sh);
  }
  if (warp == 8) {
    __syncwarp();
    tmem_dealloc(sh.tmem, C::TMEM_COLS);
  }
}

}  // namespace tc
}  // namespace boa
