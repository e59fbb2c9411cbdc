// fx_gemm_tc.cuh — FX1's contractions on the 5th-generation tensor cores: tcgen05.mma kind::i8 (int8 x int8 -> int32 in
// TMEM).  DESIGN.md section 11: a contraction is an exact integer dot product of an int8 activation row (one shift k per
// row) and an int8 weight row (one exponent s per row), followed by sat(rne(acc, s - k)) (+ residual, saturating).  The
// int32 accumulation is exact (|acc| <= K 127^2 < 2^31 for K <= 2048), so the tensor-core result is THE integer the
// specification names, whatever the tile shape or issue order.
//
// Operands reach shared memory by the bulk-copy engine as ready-made images of a tile (K-major, 128-byte swizzle, one
// k-block = 128 int8 = one swizzle row): weights laid out once at boa_fx_model_load, activations written in image
// layout by the kernel that quantises them (RMSNorm, conv + SiLU, the scan, the row cut before the head).
// One CTA = one 128 x 64 output tile: warp 4 allocates TMEM, one of its threads issues the copies and the MMAs, warps
// 0-3 read the accumulators (thread = row) and run the epilogue.
#pragma once
#include "fx_kernels.cuh"
#include "tc_gemm.cuh"

namespace boa {
namespace fx {

// Instruction descriptor: D int32, A and B signed 8-bit, both K-major, M = 128, N = 64
__host__ __device__ constexpr uint32_t idesc_i8(int n) {
  return (2u << 4) | (1u << 7) | (1u << 10) | ((uint32_t)(n >> 3) << 17) | ((uint32_t)(TBM >> 4) << 24);
}
__device__ __forceinline__ void umma_i8(uint32_t d_tmem, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "setp.ne.b32 p, %4, 0;\n"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n"
      "}" ::"r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate) : "memory");
}
// 8 consecutive int32 columns of this thread's TMEM lane
__device__ __forceinline__ void tmem_ld8_s32(uint32_t taddr, int32_t (&v)[8]) {
  asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7])
               : "r"(taddr) : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
// sat(rne(acc, s)), -31 <= s: branch-free (s <= 0 is an exact left shift)
__device__ __forceinline__ int32_t shift_round_sat(int32_t acc, int s) {
  const int sr = max(s, 0), sl = max(-s, 0);
  const int64_t v = (int64_t)acc << sl;
  const int64_t r = (v + ((1ll << sr >> 1) - 1) + ((v >> sr) & 1)) >> sr;
  return (int32_t)sat(sr ? r : v);
}

// out[m][n] = sat(rne(sum_k A[m][k] W[n][k], sw[n] - ka[m])) (+ resid[m][n], saturating);  grid (column tiles, row tiles)
__global__ void __launch_bounds__(160) k_fx_gemm_tc(const uint8_t* __restrict__ A, const int32_t* __restrict__ ka,
                                                    const uint8_t* __restrict__ W, const int32_t* __restrict__ sw,
                                                    int32_t* out, int ldo, const int32_t* resid, int M, int N, int KB,
                                                    int nst) {
  extern __shared__ uint8_t fx_smem[];
  __shared__ uint64_t full_bar[TC_MAXST], empty_bar[TC_MAXST], acc_bar;
  __shared__ uint32_t tmem_slot;
  __shared__ int32_t s_sw[TBN];
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const int nt = blockIdx.x, mt = blockIdx.y;
  const uint32_t sbase = (tc::smem_u32(fx_smem) + 1023u) & ~1023u;
  if (tid == 0) {
    for (int s = 0; s < nst; ++s) { tc::mbar_init(tc::smem_u32(&full_bar[s]), 1); tc::mbar_init(tc::smem_u32(&empty_bar[s]), 1); }
    tc::mbar_init(tc::smem_u32(&acc_bar), 1);
    tc::fence_barrier_init();
  }
  if (tid < TBN) s_sw[tid] = nt * TBN + tid < N ? sw[nt * TBN + tid] : 0;
  if (warp == 4) tc::tmem_alloc(tc::smem_u32(&tmem_slot), TBN);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  const uint32_t tmem = tmem_slot;

  if (warp == 4) {
    if (lane == 0) {
      const uint8_t* asrc = A + (size_t)mt * KB * A_BLK;
      const uint8_t* wsrc = W + (size_t)nt * KB * W_BLK;
      auto load = [&](int kb, int s) {
        const uint32_t sA = sbase + (uint32_t)s * (A_BLK + W_BLK), fb = tc::smem_u32(&full_bar[s]);
        tc::mbar_arrive_expect_tx(fb, A_BLK + W_BLK);
        tc::bulk_g2s(sA, asrc + (size_t)kb * A_BLK, A_BLK, fb);
        tc::bulk_g2s(sA + A_BLK, wsrc + (size_t)kb * W_BLK, W_BLK, fb);
      };
      for (int kb = 0; kb < min(KB, nst); ++kb) load(kb, kb);
      for (int kb = 0; kb < KB; ++kb) {
        const int s = kb % nst;
        const uint32_t par = (uint32_t)((kb / nst) & 1);
        tc::mbar_wait(tc::smem_u32(&full_bar[s]), par);
        tc::tc_fence_after();
        const uint32_t sA = sbase + (uint32_t)s * (A_BLK + W_BLK);
#pragma unroll
        for (int k4 = 0; k4 < TBK / 32; ++k4)
          umma_i8(tmem, tc::smem_desc_sw128(sA + (uint32_t)k4 * 32u), tc::smem_desc_sw128(sA + A_BLK + (uint32_t)k4 * 32u),
                  idesc_i8(TBN), (kb | k4) ? 1u : 0u);
        tc::umma_commit(tc::smem_u32(&empty_bar[s]));
        if (kb + nst < KB) {                         // (only K > 128 nst: the stage is refilled once its MMAs have read it)
          tc::mbar_wait(tc::smem_u32(&empty_bar[s]), par);
          load(kb + nst, s);
        }
      }
      tc::umma_commit(tc::smem_u32(&acc_bar));
    }
  } else {
    const int m = mt * TBM + tid;                    // thread = row = TMEM lane
    const int km = m < M ? ka[m] : 0;
    tc::mbar_wait(tc::smem_u32(&acc_bar), 0u);
    tc::tc_fence_after();
    // (a rolled loop: eight columns per pass keeps the kernel's code a few hundred instructions)
#pragma unroll 1
    for (int c0 = 0; c0 < TBN; c0 += 8) {
      int32_t acc[8];
      tmem_ld8_s32(tmem + ((uint32_t)(warp * 32) << 16) + (uint32_t)c0, acc);
      const int n0 = nt * TBN + c0;
      if (m < M && n0 < N) {
        int32_t* orow = out + (size_t)m * ldo + n0;
        const int32_t* rrow = resid ? resid + (size_t)m * ldo + n0 : nullptr;
        int32_t v[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) v[j] = shift_round_sat(acc[j], max(s_sw[c0 + j] - km, -31));
        if (n0 + 7 < N) {
          if (rrow) {
            const int4 r0 = *reinterpret_cast<const int4*>(rrow), r1 = *reinterpret_cast<const int4*>(rrow + 4);
            v[0] = add_sat32(v[0], r0.x); v[1] = add_sat32(v[1], r0.y); v[2] = add_sat32(v[2], r0.z); v[3] = add_sat32(v[3], r0.w);
            v[4] = add_sat32(v[4], r1.x); v[5] = add_sat32(v[5], r1.y); v[6] = add_sat32(v[6], r1.z); v[7] = add_sat32(v[7], r1.w);
          }
          *reinterpret_cast<int4*>(orow) = make_int4(v[0], v[1], v[2], v[3]);
          *reinterpret_cast<int4*>(orow + 4) = make_int4(v[4], v[5], v[6], v[7]);
        } else {
#pragma unroll
          for (int j = 0; j < 8; ++j)
            if (n0 + j < N) orow[j] = rrow ? add_sat32(v[j], rrow[j]) : v[j];
        }
      }
    }
  }
  tc::tc_fence_before();
  __syncthreads();
  if (warp == 4) tc::tmem_dealloc(tmem, TBN);
}

}  // namespace fx
}  // namespace boa
