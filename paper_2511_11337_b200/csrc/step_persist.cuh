// step_persist.cuh — the persistent decode-step kernel for small stream counts (BASELINE.json north_star: "a persistent
// sm_100a decode-step kernel ... steps all B streams together"; SURVEY §7 "Decode dependency chain").
//
// At small B a model step is a chain of 4L + 2 dependent, tiny kernels and the path is pure launch and drain latency
// (configs[4] at B = 1: 34 launches, ~390 us per decoded byte).  Here ONE launch steps a wave for all of its bytes:
//   - a thread-block cluster of CS CTAs owns one row tile of 128 streams (rows of different tiles never meet);
//     clusters are independent, so there is no grid-wide barrier anywhere;
//   - inside a cluster the phases of a step (per layer in_proj -> x_proj -> scan -> out_proj; head; coder + embedding
//     of the next byte) are separated by the hardware cluster barrier (barrier.cluster, ~0.2 us) instead of a kernel
//     boundary;
//   - every phase runs the SAME device code as the one-kernel-per-phase path - gemm_roles (tc_gemm.cuh: same tiles,
//     same MMA order, same epilogues), scan_roles (model_kernels.cuh), coder_step_one (coder_kernels.cuh) - with the
//     cluster's CTAs in the place of the grid, so the bytes are identical (test).
// Memory between phases: producers write with generic-proxy stores; the next phase may read them through the bulk-copy
// engine (async proxy), so every thread executes fence.proxy.async before the barrier; the barrier's release / acquire
// at cluster scope orders the rest, and its acquire invalidates L1, so plain loads of data another CTA wrote in the
// previous phase (pos, block sums of u^2) are not served from a stale line.
// The block of the paper (FFN + LayerNorm) is not handled here; such models use the graph path.
#pragma once
#include "coder_kernels.cuh"
#include "model_kernels.cuh"
#include "tc_gemm.cuh"

namespace boa {
namespace persist {

struct LayerArgs {
  tc::GemmArgs inproj, xproj, outproj;
  ScanArgs scan;
};

struct Args {
  const LayerArgs* layers;   // [L], device memory
  int L;
  tc::GemmArgs head;
  const float* logits;
  uint8_t* data;             // input (encode) or output (decode) bytes of the wave
  size_t chunk_bytes;
  CoderArrays ca;
  EmbedArgs ea;
  int B;                     // streams of the wave
  int mode;                  // 0 encode, 1 decode
  uint32_t n_steps;          // model steps to take (every stream that is not finished advances by one byte per step)
  int ec;                    // channels per scan slice
};

constexpr int NTHREADS = tc::NTHREADS;

// Dynamic shared memory: the contraction ring + staging tile and the scan's rings (RR = 0 form: W_dt in shared memory) are
// used in different phases and share it.
template <int NPW>
inline int smem_bytes(int ec, int ldj, int R) {
  const int scan_b = scan::smem_bytes(ec, ldj, R) + 1024;
  return tc::Cfg<NPW>::SMEM > scan_b ? tc::Cfg<NPW>::SMEM : scan_b;
}

// All threads of all CTAs of the cluster: end of a phase.
__device__ __forceinline__ void phase_sync() {
  asm volatile("fence.proxy.async;" ::: "memory");          // generic-proxy writes -> visible to the next phase's bulk copies
  tc::tc_fence_before();
  asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
  asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
  tc::tc_fence_after();
}

// One contraction phase: this cluster's row tile `rt`, its NT (x KS) work items dealt to the CS CTAs.
template <int NPW, int EPI>
__device__ __forceinline__ void gemm_phase(const tc::GemmArgs& g, const tc::GemmShared& sh, int rt, int crank, int csize) {
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (warp == 8 && lane == 0) tc::gemm_init_barriers<NPW, 1>(sh, tc::MAXST);   // the rings start from phase 0 in every contraction
  __syncthreads();
  const int per_rt = g.NT * g.KS;
  tc::gemm_roles<NPW, EPI, 1, false, true>(g, sh, crank, csize, rt * per_rt, (rt + 1) * per_rt, 0);
  phase_sync();
}

// grid = (row tiles of the wave) x CS CTAs in clusters of CS (launch attribute), block = 320.
template <int NPW>
__global__ void __launch_bounds__(NTHREADS, 1) k_step_persist(const Args p) {
  using C = tc::Cfg<NPW>;
  extern __shared__ uint8_t smem_raw[];
  __shared__ __align__(8) uint64_t full_bar[tc::MAXST], empty_bar[tc::MAXST], acc_full[2], acc_empty[2];
  __shared__ uint32_t tmem_base_s;
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  uint32_t csize_u;
  asm volatile("mov.u32 %0, %%cluster_nctarank;" : "=r"(csize_u));
  const int csize = (int)csize_u, crank = (int)tc::cluster_ctarank();
  const int rt = (int)blockIdx.x / csize;                 // this cluster's row tile
  const int i_begin = rt * tc::BM, i_end = min(p.B, i_begin + tc::BM);

  tc::GemmShared sh{smem_raw, full_bar, empty_bar, acc_full, acc_empty, 0u};
  if (warp == 8) tc::tmem_alloc(tc::smem_u32(&tmem_base_s), C::TMEM_COLS);
  tc::tc_fence_before();
  __syncthreads();
  tc::tc_fence_after();
  sh.tmem = tmem_base_s;
  uint8_t* scan_smem = smem_raw + (((tc::smem_u32(smem_raw) + 1023u) & ~1023u) - tc::smem_u32(smem_raw));   // 1 KB aligned, as the ring
  const int slices = p.layers[0].scan.E / p.ec;

  for (uint32_t step = 0; step < p.n_steps; ++step) {
    for (int l = 0; l < p.L; ++l) {
      const LayerArgs& la = p.layers[l];
      gemm_phase<NPW, tc::EPI_INPROJ>(la.inproj, sh, rt, crank, csize);       // S2-S4
      gemm_phase<NPW, tc::EPI_STORE>(la.xproj, sh, rt, crank, csize);         // S5
      if (csize >= slices) {                                                  // S6-S8: csize / slices CTAs per channel slice
        const int gper = csize / slices, sl = crank / gper;                   // walk over the tile's streams
        if (sl < slices) scan_roles<0>(la.scan, scan_smem, p.ec, sl, slices, crank % gper, gper, i_begin, i_end);
      } else {                                                                // fewer CTAs than slices: slices in turn
        for (int sl = crank; sl < slices; sl += csize) {
          scan_roles<0>(la.scan, scan_smem, p.ec, sl, slices, 0, 1, i_begin, i_end);
          __syncthreads();                                                    // its rings are re-initialised by the next call
        }
      }
      phase_sync();
      gemm_phase<NPW, tc::EPI_RESID>(la.outproj, sh, rt, crank, csize);       // S9
    }
    gemm_phase<NPW, tc::EPI_STORE>(p.head, sh, rt, crank, csize);             // S10
    if (warp < 8) {                                                           // S11-S14, S1 of the next step
      for (int i = i_begin + crank * 8 + warp; i < i_end; i += csize * 8) {
        if (p.mode == 0) coder_step_one<0, false>(i, lane, p.logits, p.data, p.chunk_bytes, p.ca, p.ea, nullptr, nullptr, 0u);
        else coder_step_one<1, false>(i, lane, p.logits, p.data, p.chunk_bytes, p.ca, p.ea, nullptr, nullptr, 0u);
      }
    }
    phase_sync();
  }

  tc::tc_fence_before();
  __syncthreads();
  if (warp == 8) {
    __syncwarp();
    tc::tmem_dealloc(sh.tmem, C::TMEM_COLS);
  }
}

}  // namespace persist
}  // namespace boa
