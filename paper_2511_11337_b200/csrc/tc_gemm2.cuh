// tc_gemm2.cuh — the step-path contractions as CTA-pair tiles: tcgen05.mma.cta_group::2, 256 streams x 128 columns.
//
// Same contractions, operand images, piece arithmetic and epilogues as tc_gemm.cuh (read that header first); what
// changes is the tile.  tc_gemm.cuh's 128 x 64 tile pulls 72 KB of operand pieces through L2 -> SM per k-block for
// 128 x 64 outputs, and on the step path every contraction is bound by exactly that traffic.  Here two
// CTAs of a cluster (one SM pair) own a 256 x 128 tile:
//   CTA r of the pair holds the 128 activation rows of row tile 2*mp + r        (48 KB per k-block, as before)
//   and the weight pieces [w1; w2; w3] of the 64 output columns nt*128 + 64*r   (24 KB / 8 KB per k-block, as before)
// and one tcgen05.mma.cta_group::2 (M = 256, N = 128) multiplies the 256 rows of both CTAs with the 128 weight rows of
// both: each CTA's TMEM receives its own 128 rows x all 128 columns.  The same bytes per CTA and k-block now yield
// 128 x 128 outputs per CTA: operand traffic per output is halved.
//
// Arithmetic.  Per k-step of 16 the products are issued as N = 128 MMAs into three accumulator classes of 128 columns,
//   fp32 blobs:  a1 w1 -> c0 ;  a1 w2, a2 w1 -> c1 ;  a1 w3, a2 w2, a3 w1 -> c2        (6 MMAs)
//   bf16 blobs:  a1 w  -> c0 ;  a3 w,  a2 w  -> c1                                     (3 MMAs)
// i.e. per output element the same products enter the same class in the same order as in tc_gemm.cuh (whose stacked
// N = 192 / 128 / 64 MMAs are these products side by side), and the epilogue adds (c1 + c2) + c0 as there, so a row's
// result is bit-identical in both kernels - the encode-side time slabs (tc_gemm.cuh) and this step kernel must agree
// (tests: slab bytes == step bytes).
//
// Pipeline.  Per CTA: warp 9 (one lane) streams its A block and its W block of every k-block into a ring of stages
// (cp.async.bulk against a local mbarrier); CTA 1's warp 8 forwards "my stage has landed" to CTA 0 (remote mbarrier
// arrive); CTA 0's warp 8 (one lane) waits for both and issues the MMAs for the pair; tcgen05.commit (multicast) frees
// the stage in both CTAs and, after the last k-block, tells both epilogues that the accumulators are complete.  The
// accumulators are single-buffered for fp32 blobs (3 x 128 = 384 of 512 TMEM columns) and double-buffered for bf16
// blobs (2 x 256); each CTA's eight epilogue warps move their 128 x 128 results through a shared staging tile
// (pass 1), release the accumulators (one arrival per CTA on CTA 0's barrier), and run the fused epilogue with
// lane = column (pass 2) while the next tile is being multiplied.
#pragma once
#include "tc_gemm.cuh"

namespace boa {
namespace tc2 {

using namespace tc;

constexpr int BN2 = 128;         // output columns per tile (64 per CTA's weight block)

template <int NPW>
struct Cfg2 {
  static constexpr int W_BYTES = NPW * BN * 128;               // this CTA's weight block of a k-block
  static constexpr int A_BYTES = NPA * A_PLANE;
  static constexpr int STAGE = A_BYTES + W_BYTES;
  static constexpr int NST = 2;
  static constexpr int LDS = BN2 + 4;                          // staging row, padded
  static constexpr int STILE_BYTES = BM * LDS * 4;
  static constexpr int SMEM = NST * STAGE + STILE_BYTES + 1024;
  static constexpr int NACC = NPW == 3 ? 3 : 2;                // accumulator classes
  static constexpr int ACC_COLS = NACC * BN2;
  static constexpr int NBUF = (2 * ACC_COLS <= 512) ? 2 : 1;   // accumulator buffers
  static constexpr int TMEM_COLS = 512;
};

__device__ __forceinline__ uint32_t mapa_u32(uint32_t addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(addr), "r"(rank));
  return r;
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_addr) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void mbar_wait_cluster(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred P1;\n"
      "LAB_WAIT:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 P1, [%0], %1;\n"
      "@P1 bra DONE;\n"
      "bra LAB_WAIT;\n"
      "DONE:\n"
      "}" ::"r"(bar), "r"(parity) : "memory");
}
__device__ __forceinline__ void tmem_alloc2(uint32_t dst_smem, uint32_t ncols) {   // one warp in EACH CTA of the pair
  asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem of both CTAs] (+)= A[256 rows: 128 per CTA] * B[128 rows: 64 per CTA]^T; issued by one thread of CTA 0
__device__ __forceinline__ void umma2(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n"
      "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
__device__ __forceinline__ void umma2_commit_mc(uint32_t bar, uint16_t mask) {
  asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
               ::"r"(bar), "h"(mask) : "memory");
}
// Instruction descriptor: D fp32, A and B bf16, both K-major, M = 256 (128 per CTA), N = n
__host__ __device__ constexpr uint32_t idesc2_bf16(int n) {
  return (1u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(256 >> 4) << 24);
}

// grid = 2 * min(items, SMs / 2) in clusters of 2, block = 320.  Item t -> (row-tile pair t / NT2, column tile t % NT2),
// NT2 = ceil(NT / 2) tiles of 128 columns.  KS must be 1.
template <int NPW, int EPI>
__global__ void __launch_bounds__(NTHREADS, 1) k_tc_gemm2(const GemmArgs g) {
  using C = Cfg2<NPW>;
  static_assert(NPW == 1 || NPW == 3, "weight pieces");
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[C::NST], peer_full[C::NST], empty_bar[C::NST], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;

  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int KB = g.KB, NT = g.NT;
  const int NT2 = (NT + 1) / 2, MT = (g.M + BM - 1) / BM, MP = (MT + 1) / 2;
  const int nitems = MP * NT2;
  const int crank = (int)cluster_ctarank();
  const int item0 = (int)blockIdx.x / 2, item_step = (int)gridDim.x / 2;
  const uint32_t sbase = (smem_u32(smem_raw) + 1023u) & ~1023u;

  if (warp == 8) {
    if (lane == 0) {
      for (int s = 0; s < C::NST; ++s) {
        mbar_init(smem_u32(&full_bar[s]), 1);      // this CTA's copy warp (arrive.expect_tx)
        mbar_init(smem_u32(&peer_full[s]), 1);     // CTA 0 only: CTA 1's stage has landed (remote arrive)
        mbar_init(smem_u32(&empty_bar[s]), 1);     // tcgen05.commit of the pair's MMAs (multicast)
      }
      for (int b = 0; b < 2; ++b) {
        mbar_init(smem_u32(&acc_full[b]), 1);      // tcgen05.commit (multicast)
        mbar_init(smem_u32(&acc_empty[b]), 2);     // CTA 0 only: one arrival per CTA when its epilogue has drained TMEM
      }
      fence_barrier_init();
    }
    __syncwarp();
    tmem_alloc2(smem_u32(&tmem_base_s), C::TMEM_COLS);
  }
  tc_fence_before();
  __syncthreads();
  cluster_sync();                                  // the peer's barriers are initialised before anything is sent to them
  tc_fence_after();
  const uint32_t tmem = tmem_base_s;
  pdl_launch();
  pdl_wait();                                      // everything below reads what earlier kernels of the step wrote

  if (warp == 9) {
    // ===================================================================== copy warp (both CTAs)
    if (lane == 0) {
      int kbc = 0;
      for (int item = item0; item < nitems; item += item_step) {
        const int mp = item / NT2, n2 = item - mp * NT2;
        const int mt = 2 * mp + crank, nt = 2 * n2 + crank;      // this CTA's row tile and 64-column weight tile
        const bool have_a = mt < MT, have_w = nt < NT;
        const uint8_t* asrc = g.A + img_block((size_t)min(mt, MT - 1), 0, (size_t)KB);
        const uint16_t* wsrc = g.W + (size_t)min(nt, NT - 1) * KB * (NPW * BN * 64);
        for (int kb = 0; kb < KB; ++kb, ++kbc) {
          const int s = kbc % C::NST, round = kbc / C::NST;
          if (round > 0) mbar_wait(smem_u32(&empty_bar[s]), (uint32_t)((round - 1) & 1));
          const uint32_t sA = sbase + (uint32_t)s * C::STAGE, fb = smem_u32(&full_bar[s]);
          mbar_arrive_expect_tx(fb, (uint32_t)((have_a ? C::A_BYTES : 0) + (have_w ? C::W_BYTES : 0)));
          if (have_a) bulk_g2s(sA, asrc + (size_t)kb * C::A_BYTES, (uint32_t)C::A_BYTES, fb);
          if (have_w) bulk_g2s(sA + C::A_BYTES, wsrc + (size_t)kb * (NPW * BN * 64), (uint32_t)C::W_BYTES, fb);
        }
      }
    }
  } else if (warp == 8) {
    if (lane == 0 && crank == 1) {
      // ===================================================================== CTA 1: forward "stage landed" to CTA 0
      int kbc = 0;
      for (int item = item0; item < nitems; item += item_step)
        for (int kb = 0; kb < KB; ++kb, ++kbc) {
          const int s = kbc % C::NST, round = kbc / C::NST;
          mbar_wait(smem_u32(&full_bar[s]), (uint32_t)(round & 1));
          mbar_arrive_remote(mapa_u32(smem_u32(&peer_full[s]), 0));
        }
    } else if (lane == 0) {
      // ===================================================================== CTA 0: MMA issuer for the pair
      int kbc = 0, it = 0;
      for (int item = item0; item < nitems; item += item_step, ++it) {
        const int b = C::NBUF == 2 ? (it & 1) : 0;
        if (it >= C::NBUF) {                       // both epilogues have drained this buffer
          mbar_wait_cluster(smem_u32(&acc_empty[b]), (uint32_t)((it / C::NBUF - 1) & 1));
          tc_fence_after();
        }
        const uint32_t tacc = tmem + (uint32_t)(b * C::ACC_COLS);
        for (int kb = 0; kb < KB; ++kb, ++kbc) {
          const int s = kbc % C::NST, round = kbc / C::NST;
          mbar_wait(smem_u32(&full_bar[s]), (uint32_t)(round & 1));
          mbar_wait_cluster(smem_u32(&peer_full[s]), (uint32_t)(round & 1));
          tc_fence_after();
          const uint32_t sA = sbase + (uint32_t)s * C::STAGE;
          const uint32_t sW = sA + C::A_BYTES;
          constexpr uint32_t ID = idesc2_bf16(BN2);
#pragma unroll
          for (int k4 = 0; k4 < BK / 16; ++k4) {
            const uint32_t first = (kb | k4) ? 1u : 0u;
            const uint32_t ko = (uint32_t)k4 * 32u;
            auto A_ = [&](int p) { return smem_desc_sw128(sA + p * A_PLANE + ko); };
            auto W_ = [&](int p) { return smem_desc_sw128(sW + p * (BN * 128) + ko); };
            if (NPW == 3) {
              umma2(tacc, A_(0), W_(0), ID, first);                  // a1 w1 -> c0
              umma2(tacc + BN2, A_(0), W_(1), ID, first);            // a1 w2 -> c1
              umma2(tacc + BN2, A_(1), W_(0), ID, 1u);               // a2 w1 -> c1
              umma2(tacc + 2 * BN2, A_(0), W_(2), ID, first);        // a1 w3 -> c2
              umma2(tacc + 2 * BN2, A_(1), W_(1), ID, 1u);           // a2 w2 -> c2
              umma2(tacc + 2 * BN2, A_(2), W_(0), ID, 1u);           // a3 w1 -> c2
            } else {
              umma2(tacc, A_(0), W_(0), ID, first);                  // a1 w -> c0
              umma2(tacc + BN2, A_(2), W_(0), ID, first);            // a3 w -> c1
              umma2(tacc + BN2, A_(1), W_(0), ID, 1u);               // a2 w -> c1
            }
          }
          umma2_commit_mc(smem_u32(&empty_bar[s]), 3);               // stage free in both CTAs when these MMAs have read it
        }
        umma2_commit_mc(smem_u32(&acc_full[b]), 3);                  // the accumulators of both CTAs are complete
      }
    }
  } else {
    // ===================================================================== epilogue warps (both CTAs)
    constexpr int LDS = C::LDS;
    float* stile = reinterpret_cast<float*>(smem_raw + (sbase - smem_u32(smem_raw)) + C::NST * C::STAGE);
    constexpr int LPR = BN / 4;                    // lanes per 64-column row segment in pass 2 (4 columns per lane)
    constexpr int RPI = 32 / LPR;                  // rows per warp instruction
    constexpr int NIT = BM / (8 * RPI);            // row groups per warp
    const int col = (lane % LPR) * 4;
    const int r1 = (warp & 3) * 32 + lane;         // pass 1: thread = stream row
    const uint32_t acc_empty0 = mapa_u32(smem_u32(&acc_empty[0]), 0), acc_empty1 = mapa_u32(smem_u32(&acc_empty[1]), 0);
    int it = 0;
    for (int item = item0; item < nitems; item += item_step, ++it) {
      const int b = C::NBUF == 2 ? (it & 1) : 0;
      const int mp = item / NT2, n2 = item - mp * NT2;
      const int mt = 2 * mp + crank;
      const int m0 = mt * BM;
      const bool have_rows = mt < MT;
      float rs = 1.0f;
      if (EPI == EPI_INPROJ && have_rows) {        // S2: RMSNorm row scale from the block sums of u^2, ascending
        const float* sp = g.ssq_in + (size_t)min(m0 + r1, g.M - 1) * g.KB;
        float ss = 0.0f;
        for (int q = 0; q < g.KB; ++q) ss += sp[q];
        rs = 1.0f / sqrtf(ss / (float)(g.KB * BK) + kEps);
      }
      mbar_wait(smem_u32(&acc_full[b]), (uint32_t)((it / C::NBUF) & 1));
      tc_fence_after();
      if (have_rows) {
        // Pass 1: TMEM -> registers (thread = stream row; warps w and w+4 share the 32 TMEM lanes of rows 32*(w%4).. and
        // take 64 of the 128 columns each, in two chunks of 32) -> shared staging tile.
#pragma unroll
        for (int h = 0; h < 2; ++h) {
          const int c0 = (warp >> 2) * 64 + h * 32;
          const uint32_t tl = tmem + (uint32_t)(b * C::ACC_COLS) + ((uint32_t)((warp & 3) * 32) << 16) + (uint32_t)c0;
          float v[32], w[32];
          __syncwarp();
          tmem_ld32(tl + BN2, v);                  // class 1
          if (NPW == 3) {
            tmem_ld32(tl + 2 * BN2, w);            // class 2, added first
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] += w[j];
          }
          tmem_ld32(tl, w);                        // class 0
          float4* dst = reinterpret_cast<float4*>(stile + r1 * LDS + c0);
#pragma unroll
          for (int j = 0; j < 32; j += 4)
            dst[j >> 2] = make_float4((v[j] + w[j]) * rs, (v[j + 1] + w[j + 1]) * rs, (v[j + 2] + w[j + 2]) * rs,
                                      (v[j + 3] + w[j + 3]) * rs);
        }
      }
      tc_fence_before();
      asm volatile("bar.sync 1, 256;" ::: "memory");
      if (tid == 0) mbar_arrive_remote(b ? acc_empty1 : acc_empty0);   // this CTA's part of the buffer may be overwritten
      if (have_rows) {
        // Pass 2, per 64-column half: 16 lanes own one 64-column row segment (4 consecutive columns per lane), two rows
        // per warp instruction; rows are processed four at a time with all loads issued first.
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
          const int nt = 2 * n2 + half;
          if (nt >= NT) break;
          const int n0 = nt * BN, nb = n0 + col;
          const float* st_h = stile + half * BN;
          const size_t ncol = (EPI == EPI_INPROJ && g.xz_ec > 0) ? xz_col(nb, g.E, g.xz_ec, g.xz_slice) : (size_t)nb;
          const bool conv_tile = EPI == EPI_INPROJ && n0 < g.E;
          if (conv_tile) {
            // S4: causal depthwise conv over (x_{t-3}, x_{t-2}, x_{t-1}, x_t) + SiLU (R#11); the window is a ring of three
            // slots per stream: all three are read, only the oldest is overwritten with x_t (as in tc_gemm.cuh).
            const float4 cw0 = g.conv_w[nb], cw1 = g.conv_w[nb + 1], cw2 = g.conv_w[nb + 2], cw3 = g.conv_w[nb + 3];
            const float4 cb = *reinterpret_cast<const float4*>(g.conv_b + nb);
#pragma unroll 1
            for (int i0 = 0; i0 < NIT; i0 += 4) {
              float4 x[4], w0[4], w1[4], w2[4];
              int rows[4], slot[4];
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const int r = (warp + 8 * (i0 + u)) * RPI + lane / LPR;
                rows[u] = m0 + r;
                const int rc = min(rows[u], g.M - 1);
                slot[u] = (int)(g.pos[rc] % 3u);
                const float* wp = g.win + (size_t)rc * 3 * g.E + nb;
                w0[u] = *reinterpret_cast<const float4*>(wp + slot[u] * g.E);
                w1[u] = *reinterpret_cast<const float4*>(wp + ((slot[u] + 1) % 3) * g.E);
                w2[u] = *reinterpret_cast<const float4*>(wp + ((slot[u] + 2) % 3) * g.E);
                x[u] = *reinterpret_cast<const float4*>(st_h + r * LDS + col);
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
                  *reinterpret_cast<float4*>(g.C + (size_t)rows[u] * g.ldc + ncol) = o;
                  cut4_store(g.out_img, g.out_KB, rows[u], nb, o);
                }
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
                o[u] = *reinterpret_cast<const float4*>(st_h + r * LDS + col);
                if (EPI == EPI_RESID) q[u] = *reinterpret_cast<const float4*>(g.C + (size_t)min(rows[u], g.M - 1) * g.ldc + ncol);
              }
#pragma unroll
              for (int u = 0; u < 4; ++u) {
                const bool live = rows[u] < g.M && cols_ok;
                if (EPI == EPI_RESID) {
                  // S9: residual stream, its image (times the consumer's RMSNorm weight) and the sum of its squares over
                  // this 64-column block (x, y, z, w, then the xor butterfly 8, 4, 2, 1) - as in tc_gemm.cuh
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
                  *reinterpret_cast<float4*>(g.C + (size_t)rows[u] * g.ldc + ncol) = o[u];
                }
              }
            }
          }
        }
      }
      asm volatile("bar.sync 1, 256;" ::: "memory");     // the staging tile is free for the next tile
    }
  }

  tc_fence_before();
  __syncthreads();
  cluster_sync();                                  // no CTA leaves (or frees TMEM) while the peer may still use the pair
  if (warp == 8) {
    __syncwarp();
    tmem_dealloc2(tmem, C::TMEM_COLS);
  }
}

}  // namespace tc2
}  // namespace boa
