// boa_api.cu — the C ABI of include/boa.h: host orchestration of the step kernels.
//
// Product path.  Nothing here falls back to the CPU: without a usable CUDA device every entry point
// that computes returns BOA_E_CUDA.  Nothing under oracle/ is included, linked or executed.
#include "../../include/boa.h"

#include <limits.h>
#include <math.h>
#include <stdio.h>
#include <stdlib.h>

#include <algorithm>
#include <utility>
#include <new>
#include <vector>

#include "coder_kernels.cuh"
#include "common.cuh"
#include "container.h"
#include "model_kernels.cuh"
#include "tc_gemm.cuh"
#include "tc_gemm2.cuh"
#include "step_persist.cuh"

using namespace boa;

namespace {

constexpr int kStepsPerGraph = 32;       // model steps captured into one CUDA graph launch
constexpr int kSlabT = tc::SLAB_T;       // steps per encode-side time slab
constexpr int kSlabsPerGraph = 4;        // slabs captured into one CUDA graph launch
constexpr uint64_t kMaxWaveStreams = 65536;  // streams stepped together; more chunks run in waves

struct GrowBuf {   // grow-only device buffer
  void* p = nullptr;
  size_t cap = 0;
  int reserve(size_t bytes) {
    if (bytes <= cap) return BOA_OK;
    if (p) { cudaFree(p); p = nullptr; cap = 0; }
    size_t want = round_up(bytes, 256);
    cudaError_t e = cudaMalloc(&p, want);
    if (e != cudaSuccess) { (void)cudaGetLastError(); p = nullptr; return BOA_E_NOMEM; }
    cap = want;
    return BOA_OK;
  }
  void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

struct PinBuf {    // grow-only pinned host buffer
  void* p = nullptr;
  size_t cap = 0;
  int reserve(size_t bytes) {
    if (bytes <= cap) return BOA_OK;
    if (p) { cudaFreeHost(p); p = nullptr; cap = 0; }
    const size_t want = round_up(bytes, 4096);
    if (cudaHostAlloc(&p, want, cudaHostAllocDefault) != cudaSuccess) { (void)cudaGetLastError(); p = nullptr; return BOA_E_NOMEM; }
    cap = want;
    return BOA_OK;
  }
  void release() { if (p) cudaFreeHost(p); p = nullptr; cap = 0; }
  template <class T> T* as() const { return reinterpret_cast<T*>(p); }
};

struct LayerW {
  const float *norm_w, *conv_b, *w_dtT, *b_dt, *d_skip;
  const float4 *conv_w, *A4;
  const uint16_t *img_in, *img_x, *img_out;   // tensor-core weight images (tc_gemm.cuh)
  // the paper's block (FLAG_FFN; Alg. 1 l.4, R#23) only
  const float *ffn_b1 = nullptr, *ffn_b2 = nullptr, *ln_w = nullptr, *ln_b = nullptr;
  const uint16_t *img_ffn1 = nullptr, *img_ffn2 = nullptr;
};

bool is_device_ptr(const void* p) {
  if (!p) return false;
  cudaPointerAttributes a;
  if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  return a.type == cudaMemoryTypeDevice || a.type == cudaMemoryTypeManaged;
}

}  // namespace

struct boa_model {
  int L = 0, D = 0, E = 0, R = 0, J = 0;
  int F = 0;                   // > 0: the paper's block - every mixer is followed by u <- LayerNorm(FFN(u)), hidden width F
  int npw = 3;                 // bf16 pieces per weight: 3 for fp32 blobs, 1 for bf16 blobs (exact)
  int ldj = 64;                // row stride of the x_proj output = its padded width (64 or 128)
  int ks_x = 1;                // k-splits of x_proj (a function of the model shape only: results must not depend on B)
  int n_sm = 148;              // SM count of the device (persistent grids)
  uint32_t blob_crc = 0;
  uint32_t arith_crc = 0;      // CRC-32 of the logits this device's kernels produce for a fixed probe input (boa_model_load)
  GrowBuf weights, wimg;
  const float* emb = nullptr;
  const uint16_t* img_head = nullptr;
  std::vector<LayerW> layers;

  // workspace (per wave of Bcap streams)
  uint64_t Bcap = 0;           // streams the per-stream buffers (state, window, coder) are sized for
  uint64_t rows_cap = 0;       // rows the per-row activation buffers are sized for (>= Bcap; Bcap * kSlabT for time slabs)
  GrowBuf u, xz, dbc, logits, h, win, ssq;
  GrowBuf u_img, xs_img, y_img;   // activation images: operands of the tensor-core contractions (tc_gemm.cuh)
  GrowBuf f_img, ffn_v;           // F > 0: image of the FFN's hidden layer; the FFN's output [rows][D] before LayerNorm
  GrowBuf pos, len, low, range, pending, wpos, cache, started, v, rpos, off, size, scratch, first, err;
  GrowBuf stage_in, stage_out;
  GrowBuf total;               // [0] u64 payload bytes of the waves so far, [2] int: a payload would not fit (k_wave_offsets, k_compact)
  PinBuf pin;                  // pinned host staging: payload total, per-chunk sizes and first bytes of a compress call

  // the library's own stream (capturable, unlike the legacy default stream) and the event that orders it
  // after the caller's stream
  cudaStream_t own = nullptr;
  cudaEvent_t user_ev = nullptr;

  // test-only switches (boa_debug_set_slab / boa_debug_set_max_wave): results do not depend on them
  bool use_slab = true;        // false: boa_compress steps one byte at a time like the decoder (same bytes)
  uint64_t persist_max_streams = 0;     // waves up to this many streams step inside ONE persistent launch (step_persist.cuh)
  int persist_cluster = 8;              // CTAs per row tile of 128 streams in that launch (8 = the portable maximum)
  GrowBuf persist_layers;               // device copy of the per-layer arguments of that launch
  bool use_chain = false;               // step path: dependent contractions chained inside one launch (tc::k_gemm_chain); measured
                                        // neutral (profiles/r02_chain.md), so off by default
  GrowBuf chain_cnt;                    // [2 (L + 1)][row tiles] uint32 row-tile counters of the chained contractions
  int pair_min_row_tiles = INT_MAX; // step-path contractions use CTA-pair tiles from this many 128-stream row tiles on (use_pair_tiles)
  uint64_t max_wave = 0;       // > 0: at most this many streams are stepped together (more chunks run in waves)

  // profiling
  int sample_every = 0;
  boa_profile prof{};
  std::vector<cudaEvent_t> events;

  ~boa_model() {
    for (GrowBuf* b : {&weights, &wimg, &u, &xz, &dbc, &u_img, &xs_img, &y_img, &f_img, &ffn_v, &logits, &h, &win, &ssq, &pos, &len, &low, &range,
                       &pending, &wpos, &cache, &started, &v, &rpos, &off, &size, &scratch, &first, &err,
                       &stage_in, &stage_out, &total, &persist_layers, &chain_cnt})
      b->release();
    pin.release();
    for (cudaEvent_t e : events) cudaEventDestroy(e);
    if (user_ev) cudaEventDestroy(user_ev);
    if (own) cudaStreamDestroy(own);
  }
};

namespace {

// ------------------------------------------------------------------------------------------ BOAW
float bf16_to_f32(uint16_t b) {
  uint32_t u = (uint32_t)b << 16;
  float f;
  memcpy(&f, &u, 4);
  return f;
}

uint16_t f32_to_bf16_rne(float f) {
  uint32_t u;
  memcpy(&u, &f, 4);
  if ((u & 0x7FFFFFFFu) > 0x7F800000u) return 0x7FC0;     // NaN
  u += 0x7FFFu + ((u >> 16) & 1u);
  return (uint16_t)(u >> 16);
}

// Tensor-core weight image of W[N][K] (tc_gemm.cuh): [ceil(N/BN)][K/64][npw] tiles of BN x 64 bf16 in the
// K-major 128-byte-swizzled shared-memory layout; piece p of w is bf16(w - sum of the earlier pieces).
// Rows >= N are zero.  Returns the offset (in uint16) of the image inside `img`.
size_t append_w_image(const float* W, size_t N, size_t K, int BN, int npw, std::vector<uint16_t>& img) {
  const size_t NT = (N + BN - 1) / BN, KB = K / 64, tile = (size_t)BN * 64;
  const size_t off = img.size();
  img.resize(off + NT * KB * npw * tile, 0);
  uint16_t* base = img.data() + off;
  for (size_t nt = 0; nt < NT; ++nt)
    for (size_t kb = 0; kb < KB; ++kb)
      for (size_t n = 0; n < (size_t)BN; ++n) {
        const size_t row = nt * BN + n;
        if (row >= N) continue;
        for (size_t k = 0; k < 64; ++k) {
          float r = W[row * K + kb * 64 + k];
          const size_t o = (n / 8) * 512 + (n % 8) * 64 + (((k / 8) ^ (n % 8)) * 8) + (k % 8);
          for (int p = 0; p < npw; ++p) {
            const uint16_t b = f32_to_bf16_rne(r);
            base[((nt * KB + kb) * npw + p) * tile + o] = b;
            r -= bf16_to_f32(b);
          }
        }
      }
  return off;
}

struct BlobReader {
  const uint8_t* p;
  size_t n, off;
  int dtype;
  // reads cnt values (bf16 if matrix && dtype==1 else fp32), 16-byte padded; returns false on overrun
  bool take(size_t cnt, bool is_matrix, std::vector<float>& out) {
    const bool bf = is_matrix && dtype == 1;
    const size_t nbytes = cnt * (bf ? 2 : 4);
    const size_t padded = (nbytes + 15) / 16 * 16;
    if (off + padded > n) return false;
    out.resize(cnt);
    if (bf) {
      for (size_t i = 0; i < cnt; ++i) {
        uint16_t b;
        memcpy(&b, p + off + 2 * i, 2);
        out[i] = bf16_to_f32(b);
      }
    } else {
      memcpy(out.data(), p + off, nbytes);
    }
    off += padded;
    return true;
  }
};

// ------------------------------------------------------------------------------------- step launch
struct StepCtx {
  boa_model* m;
  cudaStream_t st;
  int B;
  int mode;                 // 0 encode, 1 decode
  uint8_t* data;            // wave base of input (encode) / output (decode)
  size_t chunk_bytes;
  CoderArrays ca;
  // debug dump
  bool dump = false;
  float* dump_logits = nullptr; float* dump_probs = nullptr; uint32_t* dump_cdf = nullptr;
  uint32_t dump_steps = 0, dump_t = 0;
  int slab_T = 1;           // > 1: one call of launch_step advances every stream by slab_T steps (encode only)
  // accounting
  uint64_t launches = 0;
  bool sample = false;      // record an event after every launch
  std::vector<int>* ev_cls = nullptr;
  size_t ev_used = 0;
};

int mark(StepCtx& c, int cls) {
  ++c.launches;
  BOA_CUDA_TRY(cudaPeekAtLastError());
  if (c.sample) {
    if (c.ev_used >= c.m->events.size()) {
      cudaEvent_t e;
      BOA_CUDA_TRY(cudaEventCreate(&e));
      c.m->events.push_back(e);
    }
    BOA_CUDA_TRY(cudaEventRecord(c.m->events[c.ev_used++], c.st));
    c.ev_cls->push_back(cls);
  }
  return BOA_OK;
}

// ---- tensor-core GEMM launch (tc_gemm.cuh).  The dynamic shared-memory opt-in is set once per instantiation.
// Launch with the programmatic-serialization attribute (PDL, common.cuh): the kernel calls pdl_wait() before it
// touches anything an earlier kernel of the stream wrote.
template <typename... KArgs, typename... Args>
cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, std::forward<Args>(args)...);
}

template <int NPW, int EPI, bool SLAB = false>
int launch_tc(const tc::GemmArgs& g, int n_sm, cudaStream_t st) {
  using C = tc::Cfg<NPW>;
  const int mt = (g.M + tc::BM - 1) / tc::BM;
  cudaLaunchConfig_t cfg{};
  cfg.blockDim = dim3(tc::NTHREADS); cfg.dynamicSmemBytes = SLAB ? C::SMEM_SLAB : C::SMEM; cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  if (g.NT % 2 == 0 && mt > 1) {
    // clusters of two CTAs share the activation k-blocks of a row tile (multicast): persistent, one cluster per SM pair.
    // (Not for a wave of one row tile: there a launch is a chain of latencies and the two cluster barriers are 3 - 6 %
    // of the step - cfg5 at 64 streams 296 -> 283 us per byte; same arithmetic, same bits.)
    const int items = mt * (g.NT / 2) * g.KS;
    cfg.gridDim = dim3(2 * std::min(items, std::max(1, n_sm / 2)));
    at[1].id = cudaLaunchAttributeClusterDimension;
    at[1].val.clusterDim.x = 2; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
    cfg.numAttrs = 2;
    BOA_CUDA_TRY(cudaLaunchKernelEx(&cfg, tc::k_tc_gemm<NPW, EPI, 2, SLAB>, g));
  } else {
    cfg.gridDim = dim3(std::min(mt * g.NT * g.KS, n_sm));             // persistent: one CTA per SM
    BOA_CUDA_TRY(cudaLaunchKernelEx(&cfg, tc::k_tc_gemm<NPW, EPI, 1, SLAB>, g));
  }
  return BOA_OK;
}
// The step path's contractions: CTA-pair tiles of 256 streams x 128 columns (tc_gemm2.cuh).  Persistent, one cluster of
// two CTAs per SM pair.  `max_pairs` > 0 limits the grid (tests: several tiles per pair).
template <int NPW, int EPI>
int launch_tc2(const tc::GemmArgs& g, int n_sm, cudaStream_t st, int max_pairs = 0) {
  using C = tc2::Cfg2<NPW>;
  const int mt = (g.M + tc::BM - 1) / tc::BM;
  const int items = ((mt + 1) / 2) * ((g.NT + 1) / 2);
  int pairs = std::min(items, std::max(1, n_sm / 2));
  if (max_pairs > 0) pairs = std::min(pairs, max_pairs);
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(2 * pairs); cfg.blockDim = dim3(tc::NTHREADS); cfg.dynamicSmemBytes = C::SMEM; cfg.stream = st;
  cudaLaunchAttribute at[2];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  at[1].id = cudaLaunchAttributeClusterDimension;
  at[1].val.clusterDim.x = 2; at[1].val.clusterDim.y = 1; at[1].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 2;
  BOA_CUDA_TRY(cudaLaunchKernelEx(&cfg, tc2::k_tc_gemm2<NPW, EPI>, g));
  return BOA_OK;
}
template <int EPI>
int launch_tc2_npw(int npw, const tc::GemmArgs& g, int n_sm, cudaStream_t st, int max_pairs = 0) {
  return npw == 1 ? launch_tc2<1, EPI>(g, n_sm, st, max_pairs) : launch_tc2<3, EPI>(g, n_sm, st, max_pairs);
}
template <int NPW, int EPI>
int optin_tc2() {
  BOA_CUDA_TRY((cudaFuncSetAttribute(tc2::k_tc_gemm2<NPW, EPI>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc2::Cfg2<NPW>::SMEM)));
  return BOA_OK;
}

template <int NPW, int EPI, bool SLAB = false>
int optin_tc() {
  constexpr int smem = SLAB ? tc::Cfg<NPW>::SMEM_SLAB : tc::Cfg<NPW>::SMEM;
  BOA_CUDA_TRY((cudaFuncSetAttribute(tc::k_tc_gemm<NPW, EPI, 1, SLAB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)));
  BOA_CUDA_TRY((cudaFuncSetAttribute(tc::k_tc_gemm<NPW, EPI, 2, SLAB>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem)));
  return BOA_OK;
}
// Chained contractions of the step path (tc::k_gemm_chain): persistent, at most one CTA per SM, sized for the contraction
// with the most work items.
template <int NPW, int KIND>
int launch_chain_t(const boa_model* m, const tc::ChainArgs& a, cudaStream_t st) {
  int items = 1;
  for (int j = 0; j < (KIND == tc::CH_OUT_IN_X ? 3 : 2); ++j)
    items = std::max(items, ((a.g[j].M + tc::BM - 1) / tc::BM) * a.g[j].NT * a.g[j].KS);
  BOA_CUDA_TRY(launch_pdl(tc::k_gemm_chain<NPW, KIND>, dim3((unsigned)std::min(items, m->n_sm)), dim3(tc::NTHREADS),
                          (size_t)tc::Cfg<NPW>::SMEM, st, a));
  return BOA_OK;
}
int launch_chain(const boa_model* m, int kind, const tc::ChainArgs& a, cudaStream_t st) {
  if (m->npw == 1) {
    if (kind == tc::CH_IN_X) return launch_chain_t<1, tc::CH_IN_X>(m, a, st);
    if (kind == tc::CH_OUT_IN_X) return launch_chain_t<1, tc::CH_OUT_IN_X>(m, a, st);
    return launch_chain_t<1, tc::CH_OUT_HEAD>(m, a, st);
  }
  if (kind == tc::CH_IN_X) return launch_chain_t<3, tc::CH_IN_X>(m, a, st);
  if (kind == tc::CH_OUT_IN_X) return launch_chain_t<3, tc::CH_OUT_IN_X>(m, a, st);
  return launch_chain_t<3, tc::CH_OUT_HEAD>(m, a, st);
}
template <int NPW, int KIND>
int optin_chain() {
  BOA_CUDA_TRY((cudaFuncSetAttribute(tc::k_gemm_chain<NPW, KIND>, cudaFuncAttributeMaxDynamicSharedMemorySize, tc::Cfg<NPW>::SMEM)));
  return BOA_OK;
}

// Shared-memory opt-ins of every kernel instantiation the step can launch (called by boa_model_load, outside
// any stream capture).
int init_kernels() {
  BOA_TRY((optin_tc<1, tc::EPI_INPROJ>()));
  BOA_TRY((optin_tc<3, tc::EPI_INPROJ>()));
  BOA_TRY((optin_tc<1, tc::EPI_INPROJ, true>()));
  BOA_TRY((optin_tc<3, tc::EPI_INPROJ, true>()));
  BOA_TRY((optin_tc<1, tc::EPI_STORE>()));
  BOA_TRY((optin_tc<3, tc::EPI_STORE>()));
  BOA_TRY((optin_tc<1, tc::EPI_RESID>()));
  BOA_TRY((optin_tc<3, tc::EPI_RESID>()));
  BOA_TRY((optin_tc<1, tc::EPI_FFN1>()));
  BOA_TRY((optin_tc<3, tc::EPI_FFN1>()));
  BOA_TRY((optin_tc2<1, tc::EPI_INPROJ>()));
  BOA_TRY((optin_tc2<3, tc::EPI_INPROJ>()));
  BOA_TRY((optin_tc2<1, tc::EPI_STORE>()));
  BOA_TRY((optin_tc2<3, tc::EPI_STORE>()));
  BOA_TRY((optin_tc2<1, tc::EPI_RESID>()));
  BOA_TRY((optin_tc2<3, tc::EPI_RESID>()));
  BOA_TRY((optin_tc2<1, tc::EPI_FFN1>()));
  BOA_TRY((optin_tc2<3, tc::EPI_FFN1>()));
  BOA_TRY((optin_chain<1, tc::CH_IN_X>())); BOA_TRY((optin_chain<1, tc::CH_OUT_IN_X>())); BOA_TRY((optin_chain<1, tc::CH_OUT_HEAD>()));
  BOA_TRY((optin_chain<3, tc::CH_IN_X>())); BOA_TRY((optin_chain<3, tc::CH_OUT_IN_X>())); BOA_TRY((optin_chain<3, tc::CH_OUT_HEAD>()));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::smem_bytes(256, 128, 64)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan_slab<0>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::slab_smem_bytes(256, 128, 64)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan_slab<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::slab_smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan_slab<8>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::slab_smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan_slab<16>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::slab_smem_bytes(256, 128, 0)));
  BOA_CUDA_TRY(cudaFuncSetAttribute(k_scan_slab<32>, cudaFuncAttributeMaxDynamicSharedMemorySize, scan::slab_smem_bytes(256, 128, 0)));
  return BOA_OK;
}

template <int EPI>
int launch_tc_npw(int npw, const tc::GemmArgs& g, int n_sm, cudaStream_t st) {
  return npw == 1 ? launch_tc<1, EPI>(g, n_sm, st) : launch_tc<3, EPI>(g, n_sm, st);
}

// Which tile shape a step-path contraction runs with.  Both kernels return the same bits (tests), so this is a pure
// performance choice.  The CTA-pair tiles (256 x 128, tc_gemm2.cuh) halve the operand traffic per output, but as measured
// (profiles/r02_pair_gemm.md: B = 4,096 ... 65,536, fp32 and bf16 blobs) they are slower than or equal to the single-CTA
// tiles (128 x 64) at every size - fewer and longer work items, a single accumulator buffer for fp32 blobs - so the
// default threshold is "never"; boa_debug_set_pair_tiles selects them for the tests and for measurement.
bool use_pair_tiles(const tc::GemmArgs& g, int min_row_tiles) { return (g.M + tc::BM - 1) / tc::BM >= min_row_tiles; }
template <int EPI>
int launch_gemm_step(const boa_model* m, const tc::GemmArgs& g, cudaStream_t st) {
  if (use_pair_tiles(g, m->pair_min_row_tiles)) return launch_tc2_npw<EPI>(m->npw, g, m->n_sm, st);
  return launch_tc_npw<EPI>(m->npw, g, m->n_sm, st);
}

// S1 for the first step of a wave: u = Emb[byte 0] (later steps: fused into the coder step).
int launch_embed(StepCtx& c, int T = 1) {
  boa_model* m = c.m;
  const long long total = (long long)c.B * T * (m->D / 4);
  k_embed<<<(unsigned)((total + 255) / 256), 256, 0, c.st>>>(c.data, c.chunk_bytes, c.ca.pos, c.ca.len,
                                                  reinterpret_cast<const float4*>(m->emb), m->u.as<float4>(),
                                                  reinterpret_cast<const float4*>(m->layers[0].norm_w),
                                                  m->u_img.as<uint8_t>(), m->ssq.as<float>(), c.B, m->D / 4, T);
  return mark(c, BOA_K_EMBED);
}

// One model step + one coder step for all B streams of the wave (S2-S14, and S1 of the next step).
// With c.slab_T = T > 1 (encode-side time slab) the same kernels advance every stream by T steps:
// the contractions run on B*T rows (stream-major: row i*T + t), the conv of a row reads the rows before it in its
// tile (the slab form of in_proj's epilogue), the scan keeps the state in registers across the T steps
// (k_scan_slab), the coder codes T symbols per stream (k_coder_slab).
// Per row / per step the arithmetic is that of the step path, so the decoder (always step by step) reproduces it.
int launch_step(StepCtx& c) {
  boa_model* m = c.m;
  const int B = c.B, D = m->D, E = m->E;
  const int T = c.slab_T, rows = B * T;
  float* u = m->u.as<float>();
  float* xz = m->xz.as<float>();
  float* dbc = m->dbc.as<float>();
  float* logits = m->logits.as<float>();
  float* ssq = m->ssq.as<float>();
  uint8_t* u_img = m->u_img.as<uint8_t>();
  uint8_t* xs_img = m->xs_img.as<uint8_t>();
  uint8_t* y_img = m->y_img.as<uint8_t>();
  const int ec = (E % 256 == 0) ? 256 : 128;     // channels per scan slice
  const int mt_rows = (rows + tc::BM - 1) / tc::BM;

  // the arguments of the step's contractions
  auto make_in = [&](int l) {   // S2-S4: xz = [SiLU(conv(W_in_x r)) ; W_in_z r],  r = RMSNorm(u);  xs also as the image for x_proj
    const LayerW& w = m->layers[l];
    tc::GemmArgs g{};
    g.A = u_img; g.M = rows; g.KB = D / 64; g.W = w.img_in; g.NT = 2 * E / 64; g.KS = 1;
    g.n_valid = 2 * E; g.xz_ec = ec;
    g.C = xz;           // step path: a row = [slice][xs | z]; time slab: [slice][row][xs | z] (one copy per stream-group)
    g.ldc = T == 1 ? 2 * E : 2 * ec;
    g.xz_slice = T == 1 ? (size_t)2 * ec : (size_t)rows * 2 * ec;
    g.ssq_in = ssq; g.win = m->win.as<float>() + (size_t)l * m->Bcap * 3 * E; g.pos = c.ca.pos; g.slab_T = T == 1 ? 0 : T;
    g.conv_w = w.conv_w; g.conv_b = w.conv_b; g.E = E;
    g.out_img = xs_img; g.out_KB = E / 64;
    return g;
  };
  auto make_x = [&](int l) {    // S5: [dlt;Bv;Cv] = W_x xs
    tc::GemmArgs g{};
    g.A = xs_img; g.M = rows; g.KB = E / 64; g.W = m->layers[l].img_x; g.NT = m->ldj / 64;
    g.C = dbc; g.ldc = m->ks_x * m->ldj; g.n_valid = m->J;           // row = [k-split][ldj]
    g.KS = m->ks_x; g.split_stride = (size_t)m->ldj;                  // split over k: enough tiles to fill the SMs
    return g;
  };
  auto make_out = [&](int l) {  // S9: u += W_out y;  the new u also as the image for the next in_proj (times its RMSNorm weight) or the head
    tc::GemmArgs g{};
    g.A = y_img; g.M = rows; g.KB = E / 64; g.W = m->layers[l].img_out; g.NT = D / 64; g.KS = 1;
    g.C = u; g.ldc = D; g.n_valid = D;
    g.out_img = u_img; g.out_KB = D / 64; g.ssq_out = ssq;
    // (the paper's block: the FFN reads u itself, not a normalised u)
    g.out_scale = (m->F == 0 && l + 1 < m->L) ? m->layers[l + 1].norm_w : nullptr;
    return g;
  };
  auto make_head = [&]() {      // S10: logits = Emb u
    tc::GemmArgs g{};
    g.A = u_img; g.M = rows; g.KB = D / 64; g.W = m->img_head; g.NT = 4; g.KS = 1;
    g.C = logits; g.ldc = 256; g.n_valid = 256;
    return g;
  };
  auto launch_scan = [&](int l) -> int {   // S6-S8: persistent, two CTAs per SM, each walking over streams for one channel slice
    const LayerW& w = m->layers[l];
    float* hl = m->h.as<float>() + (size_t)l * m->Bcap * E * kNState;
    ScanArgs sa{};
    sa.h = hl; sa.xz = xz; sa.dbc = dbc; sa.W_dtT = w.w_dtT; sa.b_dt = w.b_dt; sa.A4 = w.A4; sa.Dskip = w.d_skip;
    sa.y_img = y_img; sa.ldj = m->ldj; sa.B = B; sa.E = E; sa.R = m->R;
    sa.KS = m->ks_x;
    const int slices = E / ec;
    const int per_slice = std::max(1, std::min(B, (2 * m->n_sm + slices - 1) / slices));
    const dim3 grid(per_slice, slices);
    if (T > 1) {      // time slab: groups of 8 steps per iteration, state in registers across a stream's groups
      ScanSlabArgs ss{};
      ss.h = hl; ss.xz = xz; ss.dbc = dbc; ss.W_dtT = w.w_dtT; ss.b_dt = w.b_dt; ss.A4 = w.A4; ss.Dskip = w.d_skip;
      ss.y_img = y_img; ss.KS = m->ks_x; ss.ldj = m->ldj; ss.B = B; ss.E = E; ss.R = m->R; ss.T = T;
      const int regs = (m->R == 4 || m->R == 8 || m->R == 16 || m->R == 32) ? 0 : m->R;
      const size_t smem = scan::slab_smem_bytes(ec, m->ldj, regs);
      switch (m->R) {
        case 4: BOA_CUDA_TRY(launch_pdl(k_scan_slab<4>, grid, dim3(ec + 32), smem, c.st, ss)); break;
        case 8: BOA_CUDA_TRY(launch_pdl(k_scan_slab<8>, grid, dim3(ec + 32), smem, c.st, ss)); break;
        case 16: BOA_CUDA_TRY(launch_pdl(k_scan_slab<16>, grid, dim3(ec + 32), smem, c.st, ss)); break;
        case 32: BOA_CUDA_TRY(launch_pdl(k_scan_slab<32>, grid, dim3(ec + 32), smem, c.st, ss)); break;
        default: BOA_CUDA_TRY(launch_pdl(k_scan_slab<0>, grid, dim3(ec + 32), smem, c.st, ss)); break;
      }
    } else
    switch (m->R) {   // W_dt's row in registers when it is short enough
      case 4: BOA_CUDA_TRY(launch_pdl(k_scan<4>, grid, dim3(ec + 32), scan::smem_bytes(ec, m->ldj, 0), c.st, sa)); break;
      case 8: BOA_CUDA_TRY(launch_pdl(k_scan<8>, grid, dim3(ec + 32), scan::smem_bytes(ec, m->ldj, 0), c.st, sa)); break;
      case 16: BOA_CUDA_TRY(launch_pdl(k_scan<16>, grid, dim3(ec + 32), scan::smem_bytes(ec, m->ldj, 0), c.st, sa)); break;
      case 32: BOA_CUDA_TRY(launch_pdl(k_scan<32>, grid, dim3(ec + 32), scan::smem_bytes(ec, m->ldj, 0), c.st, sa)); break;
      default: BOA_CUDA_TRY(launch_pdl(k_scan<0>, grid, dim3(ec + 32), scan::smem_bytes(ec, m->ldj, m->R), c.st, sa)); break;
    }
    return mark(c, BOA_K_SCAN);
  };

  // Step path of north_star's block: the dependent contractions between two scans run chained inside ONE launch
  // (tc::k_gemm_chain): in_proj -> x_proj | scan | out_proj -> in_proj -> x_proj | scan | ... | out_proj -> head | coder,
  // 2L + 2 launches per step instead of 4L + 2; row-tile counters order the work items.  Same bits (test).
  const bool chain = m->use_chain && T == 1 && m->F == 0;
  if (chain) {
    uint32_t* cnt = m->chain_cnt.as<uint32_t>();
    const uint32_t in_tiles = (uint32_t)(E / 64), out_tiles = (uint32_t)(D / 64);
    for (int k = 0; k <= m->L; ++k) {
      uint32_t* ca = cnt + (size_t)(2 * k) * mt_rows;
      uint32_t* cb = cnt + (size_t)(2 * k + 1) * mt_rows;
      tc::ChainArgs a{};
      if (k == 0) {
        a.g[0] = make_in(0); a.g[0].done = ca; a.g[0].done_cols = E;
        a.g[1] = make_x(0); a.g[1].dep = ca; a.g[1].dep_target = in_tiles;
        BOA_TRY(launch_chain(m, tc::CH_IN_X, a, c.st));
        BOA_TRY(mark(c, BOA_K_CHAIN_IN_X));
      } else if (k < m->L) {
        a.g[0] = make_out(k - 1); a.g[0].done = ca; a.g[0].done_cols = D;
        a.g[1] = make_in(k); a.g[1].dep = ca; a.g[1].dep_target = out_tiles; a.g[1].done = cb; a.g[1].done_cols = E;
        a.g[2] = make_x(k); a.g[2].dep = cb; a.g[2].dep_target = in_tiles;
        BOA_TRY(launch_chain(m, tc::CH_OUT_IN_X, a, c.st));
        BOA_TRY(mark(c, BOA_K_CHAIN_OUT_IN_X));
      } else {
        a.g[0] = make_out(m->L - 1); a.g[0].done = ca; a.g[0].done_cols = D;
        a.g[1] = make_head(); a.g[1].dep = ca; a.g[1].dep_target = out_tiles;
        BOA_TRY(launch_chain(m, tc::CH_OUT_HEAD, a, c.st));
        BOA_TRY(mark(c, BOA_K_CHAIN_OUT_HEAD));
      }
      if (k < m->L) BOA_TRY(launch_scan(k));
    }
  } else {
  for (int l = 0; l < m->L; ++l) {
    const LayerW& w = m->layers[l];
    {
      const tc::GemmArgs g = make_in(l);
      if (T > 1) {   // the time-slab form of the conv epilogue
        BOA_TRY((m->npw == 1 ? launch_tc<1, tc::EPI_INPROJ, true>(g, m->n_sm, c.st) : launch_tc<3, tc::EPI_INPROJ, true>(g, m->n_sm, c.st)));
      } else {
        BOA_TRY((launch_gemm_step<tc::EPI_INPROJ>(m, g, c.st)));
      }
      BOA_TRY(mark(c, BOA_K_INPROJ));
    }
    {
      const tc::GemmArgs g = make_x(l);
      BOA_TRY((launch_tc_npw<tc::EPI_STORE>(m->npw, g, m->n_sm, c.st)));
      BOA_TRY(mark(c, BOA_K_CONVX));
    }
    BOA_TRY(launch_scan(l));
    {
      const tc::GemmArgs g = make_out(l);
      if (T == 1) BOA_TRY((launch_gemm_step<tc::EPI_RESID>(m, g, c.st)));
      else BOA_TRY((launch_tc_npw<tc::EPI_RESID>(m->npw, g, m->n_sm, c.st)));
      BOA_TRY(mark(c, BOA_K_OUTPROJ));
    }
    if (m->F > 0) {  // the paper's block (Alg. 1 l.4, R#23): u <- LayerNorm(W2 GELU(W1 u + b1) + b2)
      const int F = m->F;
      uint8_t* f_img = m->f_img.as<uint8_t>();
      float* ffn_v = m->ffn_v.as<float>();
      {
        tc::GemmArgs g{};
        g.A = u_img; g.M = rows; g.KB = D / 64; g.W = w.img_ffn1; g.NT = F / 64; g.KS = 1;
        g.n_valid = F; g.bias = w.ffn_b1; g.out_img = f_img; g.out_KB = F / 64;
        if (T == 1) BOA_TRY((launch_gemm_step<tc::EPI_FFN1>(m, g, c.st)));
        else BOA_TRY((launch_tc_npw<tc::EPI_FFN1>(m->npw, g, m->n_sm, c.st)));
        BOA_TRY(mark(c, BOA_K_FFN1));
      }
      {
        tc::GemmArgs g{};
        g.A = f_img; g.M = rows; g.KB = F / 64; g.W = w.img_ffn2; g.NT = D / 64; g.KS = 1;
        g.C = ffn_v; g.ldc = D; g.n_valid = D; g.bias = w.ffn_b2;
        if (T == 1) BOA_TRY((launch_gemm_step<tc::EPI_STORE>(m, g, c.st)));
        else BOA_TRY((launch_tc_npw<tc::EPI_STORE>(m->npw, g, m->n_sm, c.st)));
        BOA_TRY(mark(c, BOA_K_FFN2));
      }
      BOA_CUDA_TRY(launch_pdl(k_layernorm, dim3((unsigned)(((size_t)rows * 32 + 255) / 256)), dim3(256), 0, c.st,
                              (const float*)ffn_v, w.ln_w, w.ln_b, u, (l + 1 < m->L) ? m->layers[l + 1].norm_w : (const float*)nullptr,
                              u_img, ssq, rows, D));
      BOA_TRY(mark(c, BOA_K_LNORM));
    }
  }
  {
    const tc::GemmArgs g = make_head();
    if (T == 1) BOA_TRY((launch_gemm_step<tc::EPI_STORE>(m, g, c.st)));
    else BOA_TRY((launch_tc_npw<tc::EPI_STORE>(m->npw, g, m->n_sm, c.st)));
    BOA_TRY(mark(c, BOA_K_HEAD));
  }
  }

  const int cgrid = (B * 32 + 255) / 256;
  uint32_t* zero_p = chain ? m->chain_cnt.as<uint32_t>() : nullptr;
  const int zero_n = chain ? 2 * (m->L + 1) * mt_rows : 0;
  EmbedArgs ea{};
  ea.emb = reinterpret_cast<const float4*>(m->emb); ea.norm_w = reinterpret_cast<const float4*>(m->layers[0].norm_w);
  ea.u = reinterpret_cast<float4*>(u); ea.u_img = u_img; ea.ssq = ssq; ea.D4 = D / 4;
  if (T > 1) {
    BOA_CUDA_TRY(launch_pdl(k_coder_slab, dim3(cgrid), dim3(256), 0, c.st, (const float*)logits, (const uint8_t*)c.data,
                            c.chunk_bytes, c.ca, B, T));
  } else if (c.dump) {
    if (c.dump_logits) {
      BOA_CUDA_TRY(cudaMemcpy2DAsync(c.dump_logits + (size_t)c.dump_t * 256, (size_t)c.dump_steps * 256 * sizeof(float),
                                     logits, 256 * sizeof(float), 256 * sizeof(float), B,
                                     cudaMemcpyDeviceToDevice, c.st));
    }
    k_coder_step<0, true><<<cgrid, 256, 0, c.st>>>(logits, c.data, c.chunk_bytes, c.ca, B, ea, c.dump_probs,
                                                   c.dump_cdf, c.dump_steps, zero_p, zero_n);
  } else if (c.mode == 0) {
    BOA_CUDA_TRY(launch_pdl(k_coder_step<0, false>, dim3(cgrid), dim3(256), 0, c.st, (const float*)logits, c.data,
                            c.chunk_bytes, c.ca, B, ea, (float*)nullptr, (uint32_t*)nullptr, 0u, zero_p, zero_n));
  } else {
    BOA_CUDA_TRY(launch_pdl(k_coder_step<1, false>, dim3(cgrid), dim3(256), 0, c.st, (const float*)logits, c.data,
                            c.chunk_bytes, c.ca, B, ea, (float*)nullptr, (uint32_t*)nullptr, 0u, zero_p, zero_n));
  }
  BOA_TRY(mark(c, BOA_K_CODER));
  return BOA_OK;
}

// Small waves: all `steps` iterations inside ONE launch of the persistent step kernel (step_persist.cuh) - a cluster of
// CTAs per row tile of 128 streams, cluster barriers between the phases of a step.  Same device code per phase as
// launch_step's kernels, same bytes (test).  The argument structs are those launch_step builds for T = 1.
template <int NPW>
int launch_persist(StepCtx& c, uint64_t steps) {
  boa_model* m = c.m;
  const int B = c.B, D = m->D, E = m->E;
  const int ec = (E % 256 == 0) ? 256 : 128;
  std::vector<persist::LayerArgs> la((size_t)m->L);
  for (int l = 0; l < m->L; ++l) {
    const LayerW& w = m->layers[l];
    float* hl = m->h.as<float>() + (size_t)l * m->Bcap * E * kNState;
    float* winl = m->win.as<float>() + (size_t)l * m->Bcap * 3 * E;
    tc::GemmArgs& gi = la[l].inproj;
    gi = tc::GemmArgs{};
    gi.A = m->u_img.as<uint8_t>(); gi.M = B; gi.KB = D / 64; gi.W = w.img_in; gi.NT = 2 * E / 64; gi.KS = 1;
    gi.n_valid = 2 * E; gi.xz_ec = ec; gi.C = m->xz.as<float>(); gi.ldc = 2 * E; gi.xz_slice = (size_t)2 * ec;
    gi.ssq_in = m->ssq.as<float>(); gi.win = winl; gi.pos = c.ca.pos; gi.slab_T = 0; gi.conv_w = w.conv_w; gi.conv_b = w.conv_b; gi.E = E;
    gi.out_img = m->xs_img.as<uint8_t>(); gi.out_KB = E / 64;
    tc::GemmArgs& gx = la[l].xproj;
    gx = tc::GemmArgs{};
    gx.A = m->xs_img.as<uint8_t>(); gx.M = B; gx.KB = E / 64; gx.W = w.img_x; gx.NT = m->ldj / 64;
    gx.C = m->dbc.as<float>(); gx.ldc = m->ks_x * m->ldj; gx.n_valid = m->J; gx.KS = m->ks_x; gx.split_stride = (size_t)m->ldj;
    ScanArgs& sa = la[l].scan;
    sa = ScanArgs{};
    sa.h = hl; sa.xz = m->xz.as<float>(); sa.dbc = m->dbc.as<float>(); sa.W_dtT = w.w_dtT; sa.b_dt = w.b_dt; sa.A4 = w.A4; sa.Dskip = w.d_skip;
    sa.y_img = m->y_img.as<uint8_t>(); sa.ldj = m->ldj; sa.B = B; sa.E = E; sa.R = m->R; sa.KS = m->ks_x;
    tc::GemmArgs& go = la[l].outproj;
    go = tc::GemmArgs{};
    go.A = m->y_img.as<uint8_t>(); go.M = B; go.KB = E / 64; go.W = w.img_out; go.NT = D / 64; go.KS = 1;
    go.C = m->u.as<float>(); go.ldc = D; go.n_valid = D;
    go.out_img = m->u_img.as<uint8_t>(); go.out_KB = D / 64; go.ssq_out = m->ssq.as<float>();
    go.out_scale = (l + 1 < m->L) ? m->layers[l + 1].norm_w : nullptr;
  }
  BOA_TRY(m->persist_layers.reserve(la.size() * sizeof(persist::LayerArgs)));
  BOA_CUDA_TRY(cudaMemcpyAsync(m->persist_layers.p, la.data(), la.size() * sizeof(persist::LayerArgs), cudaMemcpyHostToDevice, c.st));
  BOA_CUDA_TRY(cudaStreamSynchronize(c.st));      // `la` is pageable host memory: the copy has left it
  persist::Args p{};
  p.layers = m->persist_layers.as<persist::LayerArgs>(); p.L = m->L;
  p.head = tc::GemmArgs{};
  p.head.A = m->u_img.as<uint8_t>(); p.head.M = B; p.head.KB = D / 64; p.head.W = m->img_head; p.head.NT = 4; p.head.KS = 1;
  p.head.C = m->logits.as<float>(); p.head.ldc = 256; p.head.n_valid = 256;
  p.logits = m->logits.as<float>(); p.data = c.data; p.chunk_bytes = c.chunk_bytes; p.ca = c.ca;
  p.ea.emb = reinterpret_cast<const float4*>(m->emb); p.ea.norm_w = reinterpret_cast<const float4*>(m->layers[0].norm_w);
  p.ea.u = m->u.as<float4>(); p.ea.u_img = m->u_img.as<uint8_t>(); p.ea.ssq = m->ssq.as<float>(); p.ea.D4 = D / 4;
  p.B = B; p.mode = c.mode; p.n_steps = (uint32_t)steps; p.ec = ec;
  const int cs = m->persist_cluster, row_tiles = (B + tc::BM - 1) / tc::BM;
  const int smem = persist::smem_bytes<NPW>(ec, m->ldj, m->R);
  BOA_CUDA_TRY(cudaFuncSetAttribute(persist::k_step_persist<NPW>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem));
  if (cs > 8) BOA_CUDA_TRY(cudaFuncSetAttribute(persist::k_step_persist<NPW>, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3((unsigned)(row_tiles * cs)); cfg.blockDim = dim3(persist::NTHREADS); cfg.dynamicSmemBytes = (size_t)smem; cfg.stream = c.st;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeClusterDimension;
  at[0].val.clusterDim.x = (unsigned)cs; at[0].val.clusterDim.y = 1; at[0].val.clusterDim.z = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  BOA_CUDA_TRY(cudaLaunchKernelEx(&cfg, persist::k_step_persist<NPW>, p));
  return mark(c, BOA_K_CODER);
}

// Run `steps` lock-step iterations: CUDA-graph batches of kStepsPerGraph steps, remainder eager.
int run_steps(StepCtx& c, uint64_t steps) {
  boa_model* m = c.m;
  if (steps == 0) return BOA_OK;
  if (!c.dump && m->sample_every == 0 && m->F == 0 && c.slab_T == 1 && (uint64_t)c.B <= m->persist_max_streams)
    return m->npw == 1 ? launch_persist<1>(c, steps) : launch_persist<3>(c, steps);
  const uint64_t S = std::min<uint64_t>(kStepsPerGraph, steps);
  const uint64_t n_batches = steps / S;
  const uint64_t rem = steps - n_batches * S;

  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  uint64_t graph_nodes = 0;
  int rc = BOA_OK;
  if (n_batches > 0 && !c.dump) {
    const uint64_t before = c.launches;
    BOA_CUDA_TRY(cudaStreamBeginCapture(c.st, cudaStreamCaptureModeThreadLocal));
    for (uint64_t s = 0; s < S && rc == BOA_OK; ++s) rc = launch_step(c);
    cudaError_t e = cudaStreamEndCapture(c.st, &graph);
    graph_nodes = c.launches - before;
    c.launches = before;
    if (rc == BOA_OK && e != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
    if (rc == BOA_OK && (e = cudaGraphInstantiate(&exec, graph, 0)) != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
    if (rc != BOA_OK) {
      if (graph) cudaGraphDestroy(graph);
      return rc;
    }
  }

  std::vector<int> ev_cls;
  for (uint64_t b = 0; b < n_batches && rc == BOA_OK; ++b) {
    const bool sample = m->sample_every > 0 && (b % (uint64_t)m->sample_every) == (uint64_t)(m->sample_every / 2);
    if (exec && !sample) {
      cudaError_t ge = cudaGraphLaunch(exec, c.st);
      if (ge != cudaSuccess) { rc = note_cuda_error(ge, __FILE__, __LINE__); break; }
      c.launches += graph_nodes;
      continue;
    }
    if (sample) {
      // eager batch, one event after every kernel (and one before the first)
      ev_cls.clear();
      c.ev_cls = &ev_cls;
      c.ev_used = 0;
      c.sample = true;
      --c.launches;                        // the leading marker is not a kernel
      rc = mark(c, -1);
    }
    for (uint64_t s = 0; s < S && rc == BOA_OK; ++s) {
      if (c.dump) c.dump_t = (uint32_t)(b * S + s);
      rc = launch_step(c);
    }
    if (sample) {
      c.sample = false;
      if (rc == BOA_OK && cudaEventSynchronize(m->events[c.ev_used - 1]) != cudaSuccess) { (void)cudaGetLastError(); rc = BOA_E_CUDA; }
      for (size_t k = 1; k < c.ev_used && rc == BOA_OK; ++k) {
        float ms = 0.0f;
        if (cudaEventElapsedTime(&ms, m->events[k - 1], m->events[k]) != cudaSuccess) { (void)cudaGetLastError(); rc = BOA_E_CUDA; break; }
        const int cls = ev_cls[k];
        if (cls >= 0 && cls < BOA_K_COUNT) { m->prof.sampled_ms[cls] += ms; m->prof.sampled_launches[cls] += 1; }
      }
    }
  }
  for (uint64_t s = 0; s < rem && rc == BOA_OK; ++s) {
    if (c.dump) c.dump_t = (uint32_t)(n_batches * S + s);
    rc = launch_step(c);
  }
  if (exec) cudaGraphExecDestroy(exec);
  if (graph) cudaGraphDestroy(graph);
  return rc;
}

// Encode-side time slabs: n_slabs times (embed kSlabT bytes per stream, one launch_step with slab_T = kSlabT),
// CUDA-graph batches of kSlabsPerGraph slabs, remainder eager.
int run_slabs(StepCtx& c, uint64_t n_slabs) {
  if (n_slabs == 0) return BOA_OK;
  const int saved_T = c.slab_T;
  c.slab_T = kSlabT;
  const uint64_t G = std::min<uint64_t>(kSlabsPerGraph, n_slabs);
  const uint64_t n_batches = n_slabs / G, rem = n_slabs - n_batches * G;
  cudaGraph_t graph = nullptr;
  cudaGraphExec_t exec = nullptr;
  int rc = BOA_OK;
  const uint64_t before = c.launches;
  cudaError_t e = cudaStreamBeginCapture(c.st, cudaStreamCaptureModeThreadLocal);
  if (e != cudaSuccess) { c.slab_T = saved_T; return note_cuda_error(e, __FILE__, __LINE__); }
  for (uint64_t s = 0; s < G && rc == BOA_OK; ++s) {
    rc = launch_embed(c, kSlabT);
    if (rc == BOA_OK) rc = launch_step(c);
  }
  e = cudaStreamEndCapture(c.st, &graph);
  const uint64_t graph_nodes = c.launches - before;
  c.launches = before;
  if (rc == BOA_OK && e != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
  if (rc == BOA_OK && (e = cudaGraphInstantiate(&exec, graph, 0)) != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
  for (uint64_t b = 0; b < n_batches && rc == BOA_OK; ++b) {
    if ((e = cudaGraphLaunch(exec, c.st)) != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
    c.launches += graph_nodes;
  }
  for (uint64_t s = 0; s < rem && rc == BOA_OK; ++s) {
    rc = launch_embed(c, kSlabT);
    if (rc == BOA_OK) rc = launch_step(c);
  }
  if (exec) cudaGraphExecDestroy(exec);
  if (graph) cudaGraphDestroy(graph);
  c.slab_T = saved_T;
  return rc;
}

// ------------------------------------------------------------------------------------- workspace
size_t bytes_per_row(const boa_model* m) {   // activations of one stream-step
  const size_t E = m->E, D = m->D;
  return 4 * (D + 2 * E + (size_t)m->ks_x * m->ldj + 256 + D / 64) + 6 * (D + 2 * E) + (m->F ? 6 * (size_t)m->F + 4 * D : 0);
}
size_t bytes_per_stream(const boa_model* m, size_t cap, size_t rows_per_stream = 1) {
  const size_t E = m->E;
  return rows_per_stream * bytes_per_row(m) + (size_t)m->L * 4 * (E * kNState + 3 * E) + 64 + cap;
}

// B streams; `rows` stream-steps of activations (= B on the step path, B * kSlabT for encode-side time slabs)
int reserve_workspace(boa_model* m, uint64_t B, size_t cap, uint64_t rows = 0) {
  const size_t E = m->E, D = m->D, L = m->L;
  rows = std::max(rows, B);
  if (rows > m->rows_cap) {
    BOA_TRY(m->u.reserve(rows * D * 4));
    BOA_TRY(m->xz.reserve(rows * 2 * E * 4));
    BOA_TRY(m->dbc.reserve((size_t)m->ks_x * rows * m->ldj * 4));
    BOA_TRY(m->ssq.reserve(rows * (D / 64) * 4));
    BOA_TRY(m->u_img.reserve(tc::img_bytes(rows, D)));
    BOA_TRY(m->xs_img.reserve(tc::img_bytes(rows, E)));
    BOA_TRY(m->y_img.reserve(tc::img_bytes(rows, E)));
    if (m->F > 0) {
      BOA_TRY(m->f_img.reserve(tc::img_bytes(rows, (size_t)m->F)));
      BOA_TRY(m->ffn_v.reserve(rows * D * 4));
    }
    BOA_TRY(m->logits.reserve(rows * 256 * 4));
    BOA_TRY(m->chain_cnt.reserve((size_t)2 * (L + 1) * ((rows + tc::BM - 1) / tc::BM) * 4));
    m->rows_cap = rows;
  }
  if (B > m->Bcap) {
    // state arrays are indexed [l][Bcap][...]: growing B invalidates nothing (state is reset per wave)
    BOA_TRY(m->h.reserve(L * B * E * kNState * 4));
    BOA_TRY(m->win.reserve(L * B * 3 * E * 4));
    BOA_TRY(m->pos.reserve(B * 4));
    BOA_TRY(m->len.reserve(B * 4));
    BOA_TRY(m->low.reserve(B * 8));
    BOA_TRY(m->range.reserve(B * 4));
    BOA_TRY(m->pending.reserve(B * 4));
    BOA_TRY(m->wpos.reserve(B * 4));
    BOA_TRY(m->cache.reserve(B));
    BOA_TRY(m->started.reserve(B));
    BOA_TRY(m->v.reserve(B * 4));
    BOA_TRY(m->rpos.reserve(B * 4));
    BOA_TRY(m->off.reserve(B * 8));
    BOA_TRY(m->size.reserve(B * 4));
    BOA_TRY(m->first.reserve(B));
    BOA_TRY(m->err.reserve(4));
    m->Bcap = B;
  }
  if (cap) BOA_TRY(m->scratch.reserve(m->Bcap * cap));
  return BOA_OK;
}

CoderArrays coder_arrays(boa_model* m, uint32_t cap) {
  CoderArrays ca{};
  ca.pos = m->pos.as<uint32_t>(); ca.len = m->len.as<uint32_t>();
  ca.low = m->low.as<uint64_t>(); ca.range = m->range.as<uint32_t>(); ca.pending = m->pending.as<uint32_t>();
  ca.wpos = m->wpos.as<uint32_t>(); ca.cache = m->cache.as<uint8_t>(); ca.started = m->started.as<uint8_t>();
  ca.scratch = m->scratch.as<uint8_t>(); ca.cap = cap;
  ca.v = m->v.as<uint32_t>(); ca.rpos = m->rpos.as<uint32_t>();
  ca.off = m->off.as<uint64_t>(); ca.size = m->size.as<uint32_t>();
  ca.payload = nullptr; ca.err = m->err.as<int>();
  return ca;
}

int reset_state(boa_model* m, cudaStream_t st) {
  // h starts at 0 for every chunk; the conv window is zero before the chunk start
  BOA_CUDA_TRY(cudaMemsetAsync(m->h.p, 0, (size_t)m->L * m->Bcap * m->E * kNState * 4, st));
  BOA_CUDA_TRY(cudaMemsetAsync(m->win.p, 0, (size_t)m->L * m->Bcap * 3 * m->E * 4, st));
  if (m->chain_cnt.p) BOA_CUDA_TRY(cudaMemsetAsync(m->chain_cnt.p, 0, m->chain_cnt.cap, st));   // (the coder step re-zeroes them every step)
  return BOA_OK;
}

// Per-stream payload scratch: f >= 1 of 2^16 bounds a symbol at 2 bytes, + 4 flush bytes.  chunk_bytes <= kMaxChunkBytes
// (2^30) keeps this below 2^32.
uint32_t stream_cap(size_t chunk_bytes) { return (uint32_t)round_up(2 * chunk_bytes + 8, 16); }

uint64_t wave_streams(const boa_model* m, uint64_t nc, size_t cap, size_t rows_per_stream = 1) {
  size_t free_b = 0, total_b = 0;
  uint64_t w = std::min<uint64_t>(nc, kMaxWaveStreams);
  if (m->max_wave) w = std::min(w, m->max_wave);
  if (cudaMemGetInfo(&free_b, &total_b) == cudaSuccess) {
    // what the handle already holds can be reused
    const size_t held = m->Bcap * bytes_per_stream(m, m->scratch.cap / std::max<uint64_t>(m->Bcap, 1), 0) +
                        m->rows_cap * bytes_per_row(m);
    const size_t budget = (size_t)((free_b + held) * 0.85);
    const uint64_t fit = std::max<uint64_t>(1, budget / bytes_per_stream(m, cap, rows_per_stream));
    w = std::min(w, fit);
  } else {
    (void)cudaGetLastError();
  }
  return std::max<uint64_t>(w, 1);
}

void prof_begin(boa_model* m) { memset(&m->prof, 0, sizeof(m->prof)); }

struct CallTimer {
  cudaEvent_t a = nullptr, b = nullptr;
  cudaStream_t st;
  explicit CallTimer(cudaStream_t s) : st(s) {
    if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { (void)cudaGetLastError(); a = b = nullptr; }
    if (a) cudaEventRecord(a, st);
  }
  double stop() {
    float ms = 0.0f;
    if (a && b && cudaEventRecord(b, st) == cudaSuccess && cudaEventSynchronize(b) == cudaSuccess) cudaEventElapsedTime(&ms, a, b);
    (void)cudaGetLastError();
    return ms;
  }
  ~CallTimer() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); }
};

// Order the library's stream after everything already enqueued on the caller's stream.
int enter(boa_model* m, void* user_stream, cudaStream_t* st) {
  BOA_CUDA_TRY(cudaEventRecord(m->user_ev, static_cast<cudaStream_t>(user_stream)));
  BOA_CUDA_TRY(cudaStreamWaitEvent(m->own, m->user_ev, 0));
  *st = m->own;
  return BOA_OK;
}

int check_device() {
  int dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return BOA_E_CUDA; }
  cudaDeviceProp p;
  if (cudaGetDeviceProperties(&p, dev) != cudaSuccess) { (void)cudaGetLastError(); return BOA_E_CUDA; }
  if (p.major != 10) return BOA_E_CUDA;   // the kernels are built for sm_100a only
  return BOA_OK;
}

}  // namespace

// ===================================================================================== public ABI
extern "C" {

const char* boa_last_cuda_error(void) { return last_cuda_error_buf(); }

const char* boa_strerror(int code) {
  switch (code) {
    case BOA_OK: return "ok";
    case BOA_E_ARG: return "invalid argument";
    case BOA_E_FORMAT: return "not a BOA1 container / BOAW blob, or inconsistent lengths";
    case BOA_E_CRC: return "index CRC mismatch";
    case BOA_E_MODEL_MISMATCH: return "container was written with a different model or arithmetic";
    case BOA_E_CAPACITY: return "output buffer too small";
    case BOA_E_CORRUPT: return "compressed stream is corrupt or truncated";
    case BOA_E_CUDA: return "CUDA error or no usable sm_100 device";
    case BOA_E_NOMEM: return "out of memory";
    case BOA_E_UNSUPPORTED: return "model shape not supported by the kernels";
    default: return "unknown error";
  }
}

int boa_model_load(const void* weights, size_t nbytes, boa_model** out) {
  if (!weights || !out || nbytes < 64) return BOA_E_ARG;
  *out = nullptr;
  const uint8_t* p = static_cast<const uint8_t*>(weights);
  if (memcmp(p, "BOAW", 4) != 0 || get_u32(p + 4) != 1) return BOA_E_FORMAT;
  const uint32_t dtype = get_u32(p + 8), L = get_u32(p + 12), D = get_u32(p + 16), N = get_u32(p + 20),
                 K = get_u32(p + 24), ex = get_u32(p + 28), R = get_u32(p + 32), flags = get_u32(p + 36),
                 F = get_u32(p + 40);
  // flags: bit 0 = tied head (Emb^T); bit 1 = the paper's block, FFN of hidden width F + LayerNorm after every mixer
  const bool tied = (flags & 1u) != 0, ffn = (flags & 2u) != 0;
  if (dtype > 1 || (flags & ~3u) || ffn != (F > 0)) return BOA_E_FORMAT;
  if (N != (uint32_t)kNState || K != (uint32_t)kDConv || ex != 2 || L == 0 || L > 64 ||
      D == 0 || D % 64 != 0 || D > 512 || R == 0 || R > 64 || R % 4 != 0 || F % 64 != 0 || F > 4096)
    return BOA_E_UNSUPPORTED;
  BOA_TRY(check_device());
  const size_t E = 2 * (size_t)D, J = R + 2 * kNState;

  boa_model* m = new (std::nothrow) boa_model();
  if (!m) return BOA_E_NOMEM;
  m->L = (int)L; m->D = (int)D; m->E = (int)E; m->R = (int)R; m->J = (int)J; m->F = (int)F;
  m->blob_crc = crc32_ieee(p, nbytes);
  m->npw = dtype == 1 ? 1 : 3;         // a bf16 weight is one exact piece; an fp32 weight is cut into three
  m->ldj = J <= 64 ? 64 : 128;
  m->ks_x = ((E / 64) % 4 == 0) ? 4 : ((E / 64) % 2 == 0) ? 2 : 1;
  {
    int dev = 0, n_sm = 0;
    if (cudaGetDevice(&dev) == cudaSuccess && cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && n_sm > 0)
      m->n_sm = n_sm;
    (void)cudaGetLastError();
  }

  // host image of the device buffers: small fp32 tensors (img) and the tensor-core images of the matrices (wimg);
  // bf16 matrices are widened exactly (R#13)
  const size_t per_layer = D + 4 * E + E + E * R + E + E * kNState + E;
  std::vector<float> img;
  std::vector<uint16_t> wimg;
  img.reserve(256 * D + L * per_layer + 64);
  wimg.reserve(((size_t)(tied ? 256 : 512) * D + L * (2 * E * D + (size_t)m->ldj * E + D * E + 2 * (size_t)F * D)) * m->npw + 64);
  auto append = [&](const std::vector<float>& v) {
    size_t o = img.size();
    img.insert(img.end(), v.begin(), v.end());
    while (img.size() % 4) img.push_back(0.0f);   // keep every tensor 16-byte aligned
    return o;
  };
  struct Off { size_t norm_w, conv_w, conv_b, w_dtT, b_dt, A4, d_skip, img_in, img_x, img_out,
               ffn_b1, ffn_b2, ln_w, ln_b, img_ffn1, img_ffn2; };
  std::vector<Off> offs(L);
  BlobReader br{p, nbytes, 64, (int)dtype};
  std::vector<float> t, t2;
  bool ok = br.take(256 * (size_t)D, true, t);
  size_t emb_off = 0, head_off = 0;
  if (ok) { emb_off = append(t); if (tied) head_off = append_w_image(t.data(), 256, D, 64, m->npw, wimg); }
  for (uint32_t l = 0; l < L && ok; ++l) {
    Off& o = offs[l];
    ok = ok && br.take(D, false, t); if (ok) o.norm_w = append(t);
    ok = ok && br.take(2 * E * D, true, t); if (ok) o.img_in = append_w_image(t.data(), 2 * E, D, 64, m->npw, wimg);
    ok = ok && br.take(E * 4, false, t); if (ok) o.conv_w = append(t);        // [E][4] = one float4 per channel
    ok = ok && br.take(E, false, t); if (ok) o.conv_b = append(t);
    ok = ok && br.take(J * E, true, t); if (ok) o.img_x = append_w_image(t.data(), J, E, 64, m->npw, wimg);
    ok = ok && br.take(E * R, true, t);
    if (ok) {                                                                 // W_dt [E][R] -> transposed [R][E]
      t2.assign(E * R, 0.0f);
      for (size_t e = 0; e < E; ++e)
        for (size_t r = 0; r < R; ++r) t2[r * E + e] = t[e * R + r];
      o.w_dtT = append(t2);
    }
    ok = ok && br.take(E, false, t); if (ok) o.b_dt = append(t);
    ok = ok && br.take(E * kNState, false, t);
    if (ok) {                                                // A * log2(e), A = -exp(A_log) (eq. 16), layout [4][E][4]:
      t2.assign(E * kNState, 0.0f);                          // the scan computes exp(delta A) as 2^(delta * this)
      for (size_t e = 0; e < E; ++e)
        for (size_t n = 0; n < (size_t)kNState; ++n)
          t2[((n / 4) * E + e) * 4 + (n % 4)] = (float)(-exp((double)t[e * kNState + n]) * 1.4426950408889634);
      o.A4 = append(t2);
    }
    ok = ok && br.take(E, false, t); if (ok) o.d_skip = append(t);
    ok = ok && br.take(D * E, true, t); if (ok) o.img_out = append_w_image(t.data(), D, E, 64, m->npw, wimg);
    if (ffn) {
      ok = ok && br.take((size_t)F * D, true, t); if (ok) o.img_ffn1 = append_w_image(t.data(), F, D, 64, m->npw, wimg);
      ok = ok && br.take(F, false, t); if (ok) o.ffn_b1 = append(t);
      ok = ok && br.take((size_t)D * F, true, t); if (ok) o.img_ffn2 = append_w_image(t.data(), D, F, 64, m->npw, wimg);
      ok = ok && br.take(D, false, t); if (ok) o.ffn_b2 = append(t);
      ok = ok && br.take(D, false, t); if (ok) o.ln_w = append(t);
      ok = ok && br.take(D, false, t); if (ok) o.ln_b = append(t);
    }
  }
  if (!tied) {   // untied head [256][D] after the layers
    ok = ok && br.take(256 * (size_t)D, true, t);
    if (ok) head_off = append_w_image(t.data(), 256, D, 64, m->npw, wimg);
  }
  if (!ok || br.off != nbytes) { delete m; return BOA_E_FORMAT; }

  int rc = m->weights.reserve(img.size() * sizeof(float));
  if (rc == BOA_OK) rc = m->wimg.reserve(wimg.size() * sizeof(uint16_t));
  if (rc == BOA_OK) rc = init_kernels();
  if (rc == BOA_OK && (cudaStreamCreateWithFlags(&m->own, cudaStreamNonBlocking) != cudaSuccess ||
                       cudaEventCreateWithFlags(&m->user_ev, cudaEventDisableTiming) != cudaSuccess)) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc == BOA_OK && cudaMemcpy(m->weights.p, img.data(), img.size() * sizeof(float), cudaMemcpyHostToDevice) != cudaSuccess) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc == BOA_OK && cudaMemcpy(m->wimg.p, wimg.data(), wimg.size() * sizeof(uint16_t), cudaMemcpyHostToDevice) != cudaSuccess) {
    (void)cudaGetLastError();
    rc = BOA_E_CUDA;
  }
  if (rc != BOA_OK) { delete m; return rc; }
  const float* base = m->weights.as<float>();
  const uint16_t* wbase = m->wimg.as<uint16_t>();
  m->emb = base + emb_off;
  m->img_head = wbase + head_off;
  m->layers.resize(L);
  for (uint32_t l = 0; l < L; ++l) {
    const Off& o = offs[l];
    LayerW& w = m->layers[l];
    w.norm_w = base + o.norm_w; w.conv_w = reinterpret_cast<const float4*>(base + o.conv_w);
    w.conv_b = base + o.conv_b; w.w_dtT = base + o.w_dtT; w.b_dt = base + o.b_dt;
    w.A4 = reinterpret_cast<const float4*>(base + o.A4); w.d_skip = base + o.d_skip;
    w.img_in = wbase + o.img_in; w.img_x = wbase + o.img_x; w.img_out = wbase + o.img_out;
    if (ffn) {
      w.ffn_b1 = base + o.ffn_b1; w.ffn_b2 = base + o.ffn_b2; w.ln_w = base + o.ln_w; w.ln_b = base + o.ln_b;
      w.img_ffn1 = wbase + o.img_ffn1; w.img_ffn2 = wbase + o.img_ffn2;
    }
  }
  // Arithmetic probe: the tables are reproducible only with the same per-step arithmetic, and nothing
  // forces a developer to bump kArithVersion when a kernel upstream of the quantiser changes.  So the fingerprint also
  // carries what the arithmetic DOES: three streams of 40 fixed bytes are stepped through this model with the step
  // kernels and the CRC-32 of all their fp32 logits is folded into the arithmetic word.  A build (or device) whose
  // kernels round differently writes and accepts a different fingerprint: BOA_E_MODEL_MISMATCH instead of garbage.
  {
    constexpr size_t kChunks = 3, kLen = 40, kSteps = kLen - 1;
    std::vector<uint8_t> probe(kChunks * kLen);
    for (size_t i = 0; i < probe.size(); ++i) probe[i] = (uint8_t)((i * 37u + 11u) ^ (i >> 3));
    std::vector<float> logits(kChunks * kSteps * 256);
    rc = boa_debug_step_dump(m, probe.data(), probe.size(), kLen, kSteps, logits.data(), nullptr, nullptr, nullptr);
    if (rc != BOA_OK) { delete m; return rc; }
    m->arith_crc = crc32_ieee(reinterpret_cast<const uint8_t*>(logits.data()), logits.size() * sizeof(float));
  }
  *out = m;
  return BOA_OK;
}

void boa_model_free(boa_model* m) { delete m; }

uint64_t boa_model_fingerprint(const boa_model* m) {
  return m ? (((uint64_t)(kArithVersion ^ m->arith_crc) << 32) | m->blob_crc) : 0;
}

size_t boa_compress_bound(size_t n, size_t chunk_bytes) {
  if (chunk_bytes == 0) return 0;
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  // every stream: <= 2 bytes per coded symbol (f >= 1 of 2^16) + 4 flush bytes
  return index_bytes(nc) + 2 * n + 4 * (size_t)nc;
}

int boa_set_profiling(boa_model* m, int sample_every) {
  if (!m || sample_every < 0) return BOA_E_ARG;
  m->sample_every = sample_every;
  return BOA_OK;
}

int boa_get_profile(const boa_model* m, boa_profile* out) {
  if (!m || !out) return BOA_E_ARG;
  *out = m->prof;
  return BOA_OK;
}

namespace {

// Compress the chunks of d_in[0..n) (DEVICE) into d_payload (DEVICE, capacity payload_cap): the range-coder streams back to
// back; per-chunk sizes and first bytes go to the HOST arrays sizes[nc], first[nc].  Waves of streams; per wave the
// sizes -> offsets exclusive scan and the compaction run on the device (k_wave_offsets, k_compact), the sizes and first
// bytes leave through pinned memory, and the host synchronises once, after the last wave.
int compress_parts(boa_model* m, const uint8_t* d_in, size_t n, size_t chunk_bytes, uint8_t* d_payload, size_t payload_cap,
                   uint32_t* sizes, uint8_t* first, uint64_t* payload_total, cudaStream_t st, uint64_t* launches_out) {
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  *payload_total = 0;
  if (nc == 0) return BOA_OK;
  const uint32_t cap = stream_cap(chunk_bytes);
  BOA_TRY(m->pin.reserve(16 + 5 * (size_t)nc));
  uint8_t* pin = m->pin.as<uint8_t>();
  uint32_t* pin_sizes = reinterpret_cast<uint32_t*>(pin + 16);
  uint8_t* pin_first = pin + 16 + 4 * (size_t)nc;
  BOA_TRY(m->total.reserve(16));                   // [0] u64 running payload total, [1] int capacity overflow flag
  BOA_CUDA_TRY(cudaMemsetAsync(m->total.p, 0, 16, st));
  uint64_t launches = 0;

  const bool slab = m->use_slab && chunk_bytes > (size_t)kSlabT;
  const uint64_t W = wave_streams(m, nc, cap, slab ? kSlabT : 1);
  for (uint64_t c0 = 0; c0 < nc; c0 += W) {
    const uint64_t B = std::min(W, nc - c0);
    const uint64_t wave_base = c0 * chunk_bytes;
    const uint64_t n_wave = std::min<uint64_t>(n - wave_base, B * chunk_bytes);
    BOA_TRY(reserve_workspace(m, B, cap, slab ? B * kSlabT : B));
    BOA_TRY(reset_state(m, st));
    StepCtx c{};
    c.m = m; c.st = st; c.B = (int)B; c.mode = 0;
    c.data = const_cast<uint8_t*>(d_in) + wave_base;
    c.chunk_bytes = chunk_bytes;
    c.ca = coder_arrays(m, cap);
    const int g = (int)((B + 255) / 256);
    k_coder_init<0><<<g, 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n_wave, nullptr, nullptr);
    BOA_TRY(mark(c, BOA_K_FINISH));
    k_first_bytes<<<g, 256, 0, st>>>(c.data, chunk_bytes, m->first.as<uint8_t>(), (int)B);
    BOA_TRY(mark(c, BOA_K_FINISH));
    const uint64_t max_len = std::min<uint64_t>(chunk_bytes, n_wave);
    {
      // the bytes are all known: advance kSlabT steps per pass over the state (time slabs), the rest step by step
      const uint64_t steps = max_len - 1;
      const uint64_t n_slabs = slab ? steps / kSlabT : 0;
      BOA_TRY(run_slabs(c, n_slabs));
      const uint64_t rest = steps - n_slabs * kSlabT;
      if (rest) {
        BOA_TRY(launch_embed(c));
        BOA_TRY(run_steps(c, rest));
      }
    }
    m->prof.steps += max_len - 1;
    k_coder_finish<0><<<g, 256, 0, st>>>(c.ca, (int)B);
    BOA_TRY(mark(c, BOA_K_FINISH));
    // S15: sizes -> offsets (exclusive scan on the device, continuing from the waves before), then pack the payloads
    k_wave_offsets<<<1, 1024, 0, st>>>(m->wpos.as<uint32_t>(), m->off.as<uint64_t>(), (int)B, m->total.as<uint64_t>());
    BOA_TRY(mark(c, BOA_K_FINISH));
    k_compact<<<(int)((B * 32 + 255) / 256), 256, 0, st>>>(m->scratch.as<uint8_t>(), cap, m->wpos.as<uint32_t>(),
                                                          m->off.as<uint64_t>(), d_payload, (uint64_t)payload_cap,
                                                          m->total.as<int>() + 2, (int)B);
    BOA_TRY(mark(c, BOA_K_FINISH));
    BOA_CUDA_TRY(cudaMemcpyAsync(pin_sizes + c0, m->wpos.p, B * 4, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(pin_first + c0, m->first.p, B, cudaMemcpyDeviceToHost, st));
    launches += c.launches;
  }
  BOA_CUDA_TRY(cudaMemcpyAsync(pin, m->total.p, 16, cudaMemcpyDeviceToHost, st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));        // the one host synchronisation of the call's device work
  uint64_t total = 0;
  int overflow = 0;
  memcpy(&total, pin, 8);
  memcpy(&overflow, pin + 8, 4);
  if (overflow || total > payload_cap) return BOA_E_CAPACITY;
  memcpy(sizes, pin_sizes, 4 * (size_t)nc);
  memcpy(first, pin_first, (size_t)nc);
  *payload_total = total;
  if (launches_out) *launches_out += launches;
  return BOA_OK;
}

// BOA1 header + first bytes + size index + CRC into index[0 .. index_bytes(nc))
void write_index(uint8_t* index, uint64_t fingerprint, size_t n, size_t chunk_bytes, uint64_t nc, const uint8_t* first,
                 const uint32_t* sizes) {
  const size_t ib = index_bytes(nc);
  memset(index, 0, ib);
  Header h{};
  h.n = n; h.chunk_bytes = (uint32_t)chunk_bytes; h.n_chunks = (uint32_t)nc; h.freq_bits = 16;
  h.last_len = nc ? (uint32_t)(n - (nc - 1) * chunk_bytes) : 0;
  h.fingerprint = fingerprint;
  write_header(index, h);
  if (nc) memcpy(index + kHeaderBytes, first, (size_t)nc);
  uint8_t* sp = index + kHeaderBytes + first_padded(nc);
  for (uint64_t i = 0; i < nc; ++i) put_u32(sp + 4 * i, sizes[i]);
  put_u32(index + ib - 4, crc32_ieee(index, ib - 4));
}

// A validated container index: header, per-chunk sizes and payload offsets.
struct Index {
  Header h{};
  size_t ib = 0;
  std::vector<uint8_t> bytes;
  std::vector<uint32_t> sizes;
  std::vector<uint64_t> offs;
  uint64_t payload_total = 0;
};

// S16: read and validate header, index CRC, fingerprint and total length of a container (host|device pointer).
int read_index(uint64_t fingerprint, const uint8_t* in, size_t in_len, bool in_dev, cudaStream_t st, Index& ix) {
  if (in_len < kHeaderBytes + 4) return BOA_E_FORMAT;
  uint8_t hb[kHeaderBytes];
  if (in_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(hb, in, kHeaderBytes, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
  } else {
    memcpy(hb, in, kHeaderBytes);
  }
  if (!parse_header(hb, ix.h)) return BOA_E_FORMAT;
  const uint64_t nc = ix.h.n_chunks;
  ix.ib = index_bytes(nc);
  if (in_len < ix.ib) return BOA_E_FORMAT;
  ix.bytes.resize(ix.ib);
  if (in_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(ix.bytes.data(), in, ix.ib, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
  } else {
    memcpy(ix.bytes.data(), in, ix.ib);
  }
  if (get_u32(ix.bytes.data() + ix.ib - 4) != crc32_ieee(ix.bytes.data(), ix.ib - 4)) return BOA_E_CRC;
  if (ix.h.fingerprint != fingerprint) return BOA_E_MODEL_MISMATCH;
  const uint8_t* sp = ix.bytes.data() + kHeaderBytes + first_padded(nc);
  ix.sizes.resize((size_t)nc);
  ix.offs.resize((size_t)nc);
  ix.payload_total = 0;
  for (uint64_t i = 0; i < nc; ++i) { ix.sizes[i] = get_u32(sp + 4 * i); ix.offs[i] = ix.payload_total; ix.payload_total += ix.sizes[i]; }
  if (ix.ib + ix.payload_total != in_len) return BOA_E_FORMAT;
  return BOA_OK;
}

// Decode chunks [c_lo, c_hi) of a validated container whose bytes are at d_in (DEVICE) into d_out (DEVICE; byte 0 of
// chunk c_lo at d_out[0]).  Waves of streams, the same step kernels as the encoder.
int decompress_range(boa_model* m, const Index& ix, const uint8_t* d_in, uint64_t c_lo, uint64_t c_hi, uint8_t* d_out,
                     cudaStream_t st, uint64_t* launches_out) {
  const size_t chunk_bytes = ix.h.chunk_bytes;
  const uint64_t n_range = std::min<uint64_t>(ix.h.n, c_hi * chunk_bytes) - c_lo * chunk_bytes;
  uint64_t launches = 0;
  const uint64_t nc = c_hi - c_lo;
  const uint64_t W = wave_streams(m, nc, 0);
  for (uint64_t c0 = 0; c0 < nc; c0 += W) {
    const uint64_t B = std::min(W, nc - c0);
    const uint64_t wave_base = c0 * chunk_bytes;
    const uint64_t n_wave = std::min<uint64_t>(n_range - wave_base, B * chunk_bytes);
    BOA_TRY(reserve_workspace(m, B, 0));
    BOA_TRY(reset_state(m, st));
    if (c0 == 0) BOA_CUDA_TRY(cudaMemsetAsync(m->err.p, 0, 4, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->off.p, ix.offs.data() + c_lo + c0, B * 8, cudaMemcpyHostToDevice, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->size.p, ix.sizes.data() + c_lo + c0, B * 4, cudaMemcpyHostToDevice, st));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->first.p, ix.bytes.data() + kHeaderBytes + c_lo + c0, B, cudaMemcpyHostToDevice, st));
    StepCtx c{};
    c.m = m; c.st = st; c.B = (int)B; c.mode = 1;
    c.data = d_out + wave_base;
    c.chunk_bytes = chunk_bytes;
    c.ca = coder_arrays(m, 0);
    c.ca.payload = d_in + ix.ib;
    const int g = (int)((B + 255) / 256);
    k_coder_init<1><<<g, 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n_wave, m->first.as<uint8_t>(), c.data);
    BOA_TRY(mark(c, BOA_K_FINISH));
    const uint64_t max_len = std::min<uint64_t>(chunk_bytes, n_wave);
    if (max_len > 1) BOA_TRY(launch_embed(c));
    BOA_TRY(run_steps(c, max_len - 1));
    m->prof.steps += max_len - 1;
    k_coder_finish<1><<<g, 256, 0, st>>>(c.ca, (int)B);
    BOA_TRY(mark(c, BOA_K_FINISH));
    launches += c.launches;
  }
  // one host synchronisation: the error flag accumulates over the waves (the index arrays live until the call returns)
  int err = 0;
  BOA_CUDA_TRY(cudaMemcpyAsync(&err, m->err.p, 4, cudaMemcpyDeviceToHost, st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  if (err) return BOA_E_CORRUPT;
  if (launches_out) *launches_out += launches;
  return BOA_OK;
}

}  // namespace

int boa_compress(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, uint8_t* out, size_t* out_len,
                 void* cuda_stream) {
  if (!m || !out || !out_len || chunk_bytes == 0 || chunk_bytes > kMaxChunkBytes || (n && !in)) return BOA_E_ARG;
  cudaStream_t st;
  BOA_TRY(enter(m, cuda_stream, &st));
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  if (nc >= (1ull << 32)) return BOA_E_ARG;
  const size_t ib = index_bytes(nc);
  const size_t capacity = *out_len;
  if (capacity < ib) return BOA_E_CAPACITY;
  prof_begin(m);
  CallTimer timer(st);

  // device views of the user buffers
  const bool in_dev = (n == 0) || is_device_ptr(in), out_dev = is_device_ptr(out);
  const uint8_t* d_in = in;
  if (!in_dev) {
    BOA_TRY(m->stage_in.reserve(n));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->stage_in.p, in, n, cudaMemcpyHostToDevice, st));
    d_in = m->stage_in.as<uint8_t>();
  }
  uint8_t* d_out = out;
  const size_t out_cap = std::min(capacity, boa_compress_bound(n, chunk_bytes));
  if (!out_dev) {
    BOA_TRY(m->stage_out.reserve(out_cap));
    d_out = m->stage_out.as<uint8_t>();
  }

  std::vector<uint8_t> index(ib, 0), first((size_t)nc);
  std::vector<uint32_t> sizes((size_t)nc);
  uint64_t payload_total = 0, launches = 0;
  BOA_TRY(compress_parts(m, d_in, n, chunk_bytes, d_out + ib, out_cap - ib, sizes.data(), first.data(), &payload_total, st, &launches));
  write_index(index.data(), boa_model_fingerprint(m), n, chunk_bytes, nc, first.data(), sizes.data());
  const size_t total = ib + payload_total;
  if (out_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(out, index.data(), ib, cudaMemcpyHostToDevice, st));
  } else {
    memcpy(out, index.data(), ib);
    if (payload_total) BOA_CUDA_TRY(cudaMemcpyAsync(out + ib, d_out + ib, payload_total, cudaMemcpyDeviceToHost, st));
  }
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  *out_len = total;
  m->prof.launches_total = launches;
  m->prof.streams = nc;
  m->prof.total_ms = timer.stop();
  return BOA_OK;
}

int boa_compress_shard(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, uint8_t* payload, size_t* payload_len,
                       uint32_t* sizes, uint8_t* first, void* cuda_stream) {
  if (!m || !payload_len || chunk_bytes == 0 || chunk_bytes > kMaxChunkBytes || (n && (!in || !payload || !sizes || !first)))
    return BOA_E_ARG;
  if (is_device_ptr(sizes) || is_device_ptr(first)) return BOA_E_ARG;
  cudaStream_t st;
  BOA_TRY(enter(m, cuda_stream, &st));
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  if (nc >= (1ull << 32)) return BOA_E_ARG;
  prof_begin(m);
  CallTimer timer(st);
  const size_t capacity = *payload_len;
  const size_t cap_used = std::min(capacity, 2 * n + 4 * (size_t)nc);
  const bool in_dev = (n == 0) || is_device_ptr(in), out_dev = is_device_ptr(payload);
  const uint8_t* d_in = in;
  if (!in_dev) {
    BOA_TRY(m->stage_in.reserve(n));
    BOA_CUDA_TRY(cudaMemcpyAsync(m->stage_in.p, in, n, cudaMemcpyHostToDevice, st));
    d_in = m->stage_in.as<uint8_t>();
  }
  uint8_t* d_pay = payload;
  if (!out_dev && nc) {
    BOA_TRY(m->stage_out.reserve(cap_used));
    d_pay = m->stage_out.as<uint8_t>();
  }
  uint64_t payload_total = 0, launches = 0;
  BOA_TRY(compress_parts(m, d_in, n, chunk_bytes, d_pay, cap_used, sizes, first, &payload_total, st, &launches));
  if (!out_dev && payload_total) {
    BOA_CUDA_TRY(cudaMemcpyAsync(payload, d_pay, payload_total, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
  }
  *payload_len = payload_total;
  m->prof.launches_total = launches;
  m->prof.streams = nc;
  m->prof.total_ms = timer.stop();
  return BOA_OK;
}

size_t boa_container_index_bytes(size_t n, size_t chunk_bytes) {
  return chunk_bytes ? index_bytes(n_chunks_of(n, chunk_bytes)) : 0;
}

int boa_container_assemble(uint64_t fingerprint, size_t n, size_t chunk_bytes, size_t n_parts, const size_t* part_chunks,
                           const uint8_t* const* first, const uint32_t* const* sizes, const uint8_t* const* payload,
                           const size_t* payload_len, uint8_t* out, size_t* out_len, uint64_t* payload_off, void* cuda_stream) {
  if (!out || !out_len || chunk_bytes == 0 || chunk_bytes > kMaxChunkBytes || (n_parts && (!part_chunks || !first || !sizes)))
    return BOA_E_ARG;
  const uint64_t nc = n_chunks_of(n, chunk_bytes);
  uint64_t have = 0;
  for (size_t p = 0; p < n_parts; ++p) have += part_chunks[p];
  if (have != nc || nc >= (1ull << 32)) return BOA_E_ARG;
  const size_t ib = index_bytes(nc);
  std::vector<uint8_t> f((size_t)nc), index(ib);
  std::vector<uint32_t> z((size_t)nc);
  uint64_t c = 0, total = 0;
  std::vector<uint64_t> offs(n_parts + 1, 0);
  for (size_t p = 0; p < n_parts; ++p) {
    if (part_chunks[p] && (!first[p] || !sizes[p])) return BOA_E_ARG;
    uint64_t part_total = 0;
    for (size_t i = 0; i < part_chunks[p]; ++i, ++c) { f[c] = first[p][i]; z[c] = sizes[p][i]; part_total += sizes[p][i]; }
    if (payload_len && payload_len[p] != part_total) return BOA_E_FORMAT;   // a part's payload is the sum of its sizes
    offs[p] = ib + total;
    total += part_total;
  }
  offs[n_parts] = ib + total;
  if (payload_off) memcpy(payload_off, offs.data(), (n_parts + 1) * sizeof(uint64_t));
  if (*out_len < ib + total) return BOA_E_CAPACITY;
  write_index(index.data(), fingerprint, n, chunk_bytes, nc, f.data(), z.data());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const bool out_dev = is_device_ptr(out);
  bool async = false;                              // pure host assembly touches no CUDA call (it also runs without a GPU)
  if (out_dev) { BOA_CUDA_TRY(cudaMemcpyAsync(out, index.data(), ib, cudaMemcpyHostToDevice, st)); async = true; }
  else memcpy(out, index.data(), ib);
  if (payload) {
    for (size_t p = 0; p < n_parts; ++p) {
      const uint64_t len = offs[p + 1] - offs[p];
      if (!len || payload[p] == out + offs[p]) continue;        // already in place (received there)
      if (!payload[p]) return BOA_E_ARG;
      if (!out_dev && !is_device_ptr(payload[p])) memcpy(out + offs[p], payload[p], len);
      else { BOA_CUDA_TRY(cudaMemcpyAsync(out + offs[p], payload[p], len, cudaMemcpyDefault, st)); async = true; }
    }
  }
  if (async) BOA_CUDA_TRY(cudaStreamSynchronize(st));
  *out_len = ib + total;
  return BOA_OK;
}

int boa_decompressed_size(const uint8_t* in, size_t in_len, size_t* n) {
  if (!in || !n || in_len < kHeaderBytes + 4) return in && n ? BOA_E_FORMAT : BOA_E_ARG;
  uint8_t hb[kHeaderBytes];
  if (is_device_ptr(in)) {
    BOA_CUDA_TRY(cudaMemcpy(hb, in, kHeaderBytes, cudaMemcpyDeviceToHost));
  } else {
    memcpy(hb, in, kHeaderBytes);
  }
  Header h;
  if (!parse_header(hb, h)) return BOA_E_FORMAT;
  *n = (size_t)h.n;
  return BOA_OK;
}

namespace {
// boa_decompress and boa_decompress_shard: chunks [c_lo, c_lo + count) of the container (count = SIZE_MAX: all of them)
int decompress_entry(boa_model* m, const uint8_t* in, size_t in_len, uint64_t c_lo, uint64_t count, uint8_t* out,
                     size_t* out_len, void* cuda_stream) {
  if (!m || !in || !out_len) return BOA_E_ARG;
  if (in_len < kHeaderBytes + 4) return BOA_E_FORMAT;
  cudaStream_t st;
  BOA_TRY(enter(m, cuda_stream, &st));
  const bool in_dev = is_device_ptr(in);
  prof_begin(m);
  CallTimer timer(st);
  Index ix;
  BOA_TRY(read_index(boa_model_fingerprint(m), in, in_len, in_dev, st, ix));
  const uint64_t nc = ix.h.n_chunks;
  if (count == SIZE_MAX) count = nc - std::min(nc, c_lo);
  if (c_lo > nc || count > nc - c_lo) return BOA_E_ARG;
  const uint64_t c_hi = c_lo + count;
  const size_t chunk_bytes = ix.h.chunk_bytes;
  const size_t n = count ? (size_t)(std::min<uint64_t>(ix.h.n, c_hi * chunk_bytes) - c_lo * chunk_bytes) : 0;
  if (*out_len < n) return BOA_E_CAPACITY;
  if (n && !out) return BOA_E_ARG;
  if (n == 0) { *out_len = 0; m->prof.total_ms = timer.stop(); return BOA_OK; }

  const uint8_t* d_in = in;
  if (!in_dev) {
    BOA_TRY(m->stage_in.reserve(in_len));
    // only the index and this range's payload bytes are needed on the device
    const uint64_t p_lo = ix.ib + ix.offs[c_lo], p_hi = ix.ib + ix.offs[c_hi - 1] + ix.sizes[c_hi - 1];
    BOA_CUDA_TRY(cudaMemcpyAsync(m->stage_in.as<uint8_t>() + p_lo, in + p_lo, p_hi - p_lo, cudaMemcpyHostToDevice, st));
    d_in = m->stage_in.as<uint8_t>();
  }
  const bool out_dev = is_device_ptr(out);
  uint8_t* d_out = out;
  if (!out_dev) {
    BOA_TRY(m->stage_out.reserve(n));
    d_out = m->stage_out.as<uint8_t>();
  }
  uint64_t launches = 0;
  BOA_TRY(decompress_range(m, ix, d_in, c_lo, c_hi, d_out, st, &launches));
  if (!out_dev) {
    BOA_CUDA_TRY(cudaMemcpyAsync(out, d_out, n, cudaMemcpyDeviceToHost, st));
    BOA_CUDA_TRY(cudaStreamSynchronize(st));
  }
  *out_len = n;
  m->prof.launches_total = launches;
  m->prof.streams = count;
  m->prof.total_ms = timer.stop();
  return BOA_OK;
}
}  // namespace

int boa_decompress(boa_model* m, const uint8_t* in, size_t in_len, uint8_t* out, size_t* out_len, void* cuda_stream) {
  return decompress_entry(m, in, in_len, 0, SIZE_MAX, out, out_len, cuda_stream);
}

int boa_decompress_shard(boa_model* m, const uint8_t* in, size_t in_len, size_t first_chunk, size_t n_chunks_local,
                         uint8_t* out, size_t* out_len, void* cuda_stream) {
  if (n_chunks_local == SIZE_MAX) return BOA_E_ARG;
  return decompress_entry(m, in, in_len, first_chunk, n_chunks_local, out, out_len, cuda_stream);
}

// ------------------------------------------------------------------------------------ test-only
namespace {
struct TmpDev {   // device view of a user buffer for the debug entry points
  void* dev = nullptr;
  void* user = nullptr;
  size_t bytes = 0;
  bool owned = false, back = false;
  int init(const void* p, size_t nbytes, bool copy_in, bool copy_back, cudaStream_t st) {
    user = const_cast<void*>(p); bytes = nbytes; back = false;
    if (!p || nbytes == 0) { dev = nullptr; return BOA_OK; }
    if (is_device_ptr(p)) { dev = user; return BOA_OK; }
    if (cudaMalloc(&dev, nbytes) != cudaSuccess) { (void)cudaGetLastError(); dev = nullptr; return BOA_E_NOMEM; }
    owned = true; back = copy_back;
    if (copy_in) BOA_CUDA_TRY(cudaMemcpyAsync(dev, p, nbytes, cudaMemcpyHostToDevice, st));
    return BOA_OK;
  }
  int finish(cudaStream_t st) {
    if (owned && back) BOA_CUDA_TRY(cudaMemcpyAsync(user, dev, bytes, cudaMemcpyDeviceToHost, st));
    return BOA_OK;
  }
  ~TmpDev() { if (owned && dev) cudaFree(dev); }
};
}  // namespace

int boa_debug_set_slab(boa_model* m, int enabled) {
  if (!m) return BOA_E_ARG;
  m->use_slab = enabled != 0;
  return BOA_OK;
}

int boa_debug_set_pair_tiles(boa_model* m, int min_row_tiles) {
  if (!m || min_row_tiles < 0) return BOA_E_ARG;
  m->pair_min_row_tiles = min_row_tiles;
  return BOA_OK;
}

int boa_debug_set_persist(boa_model* m, size_t max_streams, int cluster_ctas) {
  if (!m || (cluster_ctas != 0 && cluster_ctas != 1 && cluster_ctas != 2 && cluster_ctas != 4 && cluster_ctas != 8 && cluster_ctas != 16))
    return BOA_E_ARG;
  m->persist_max_streams = max_streams;
  if (cluster_ctas) m->persist_cluster = cluster_ctas;
  return BOA_OK;
}

int boa_debug_set_chain(boa_model* m, int enabled) {
  if (!m) return BOA_E_ARG;
  m->use_chain = enabled != 0;
  return BOA_OK;
}

int boa_debug_set_max_wave(boa_model* m, size_t streams) {
  if (!m || streams > kMaxWaveStreams) return BOA_E_ARG;
  m->max_wave = streams;
  return BOA_OK;
}

int boa_debug_step_dump(boa_model* m, const uint8_t* in, size_t n, size_t chunk_bytes, size_t n_steps,
                        float* logits, float* probs, uint32_t* cdf, void* cuda_stream) {
  if (!m || !in || chunk_bytes < 2 || n == 0 || n % chunk_bytes != 0 || n_steps == 0 || n_steps > chunk_bytes - 1)
    return BOA_E_ARG;
  cudaStream_t st;
  BOA_TRY(enter(m, cuda_stream, &st));
  const uint64_t B = n / chunk_bytes;
  if (B > kMaxWaveStreams) return BOA_E_ARG;
  const size_t rows = (size_t)B * n_steps;
  TmpDev tin, tl, tp, tc;
  BOA_TRY(tin.init(in, n, true, false, st));
  BOA_TRY(tl.init(logits, rows * 256 * 4, false, true, st));
  BOA_TRY(tp.init(probs, rows * 256 * 4, false, true, st));
  BOA_TRY(tc.init(cdf, rows * 257 * 4, false, true, st));
  const uint32_t cap = stream_cap(chunk_bytes);
  BOA_TRY(reserve_workspace(m, B, cap));
  BOA_TRY(reset_state(m, st));
  prof_begin(m);
  StepCtx c{};
  c.m = m; c.st = st; c.B = (int)B; c.mode = 0;
  c.data = static_cast<uint8_t*>(tin.dev);
  c.chunk_bytes = chunk_bytes;
  c.ca = coder_arrays(m, cap);
  c.dump = true;
  c.dump_logits = static_cast<float*>(tl.dev);
  c.dump_probs = static_cast<float*>(tp.dev);
  c.dump_cdf = static_cast<uint32_t*>(tc.dev);
  c.dump_steps = (uint32_t)n_steps;
  k_coder_init<0><<<(int)((B + 255) / 256), 256, 0, st>>>(c.ca, (int)B, chunk_bytes, n, nullptr, nullptr);
  BOA_TRY(mark(c, BOA_K_FINISH));
  BOA_TRY(launch_embed(c));
  BOA_TRY(run_steps(c, n_steps));
  BOA_TRY(tl.finish(st));
  BOA_TRY(tp.finish(st));
  BOA_TRY(tc.finish(st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  return BOA_OK;
}

int boa_debug_gemm(const float* A, size_t M, size_t K, const float* W, size_t N, int weight_pieces, int grid_ctas,
                   float* C, void* cuda_stream) {
  if (!A || !W || !C || M == 0 || N == 0 || K == 0 || K % 64 != 0 || (weight_pieces != 1 && weight_pieces != 3) ||
      M >= (1u << 30) || N >= (1u << 20) || K >= (1u << 20))
    return BOA_E_ARG;
  BOA_TRY(check_device());
  BOA_TRY(init_kernels());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const size_t Np = round_up(N, (size_t)tc::BN);
  std::vector<uint16_t> img;
  append_w_image(W, N, K, tc::BN, weight_pieces, img);
  TmpDev ta, tw, tc_;
  BOA_TRY(ta.init(A, M * K * 4, true, false, st));
  BOA_TRY(tw.init(img.data(), img.size() * 2, true, false, st));
  // the kernel stores whole 4-column groups of a row: give it a padded C and copy the valid columns out
  void* cpad = nullptr;
  if (cudaMalloc(&cpad, M * Np * 4) != cudaSuccess) { (void)cudaGetLastError(); return BOA_E_NOMEM; }
  void* aimg = nullptr;
  if (cudaMalloc(&aimg, tc::img_bytes(M, K)) != cudaSuccess) { (void)cudaGetLastError(); cudaFree(cpad); return BOA_E_NOMEM; }
  {
    const size_t total = M * (K / 4);
    tc::k_cut_rows<<<(unsigned)((total + 255) / 256), 256, 0, st>>>(static_cast<const float*>(ta.dev), (int)K, (int)M, (int)K,
                                                                    nullptr, static_cast<uint8_t*>(aimg));
  }
  tc::GemmArgs g{};
  g.A = static_cast<const uint8_t*>(aimg); g.M = (int)M; g.KB = (int)(K / 64);
  g.W = static_cast<const uint16_t*>(tw.dev);
  g.C = static_cast<float*>(cpad); g.ldc = (int)Np; g.n_valid = (int)Np;
  g.NT = (int)(Np / 64); g.KS = 1;
  int n_sm = 148, dev = 0;
  if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) {
    (void)cudaGetLastError();
    n_sm = 148;
  }
  if (grid_ctas > 0) n_sm = std::min(n_sm, grid_ctas);
  int rc = grid_ctas < 0 ? launch_tc2_npw<tc::EPI_STORE>(weight_pieces, g, n_sm, st, grid_ctas == -1 ? 0 : -grid_ctas / 2)
                         : launch_tc_npw<tc::EPI_STORE>(weight_pieces, g, n_sm, st);
  cudaError_t e = cudaGetLastError();
  if (rc == BOA_OK && e != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
  if (rc == BOA_OK) {
    e = cudaMemcpy2DAsync(C, N * 4, cpad, Np * 4, N * 4, M, cudaMemcpyDefault, st);
    if (e == cudaSuccess) e = cudaStreamSynchronize(st);
    if (e != cudaSuccess) rc = note_cuda_error(e, __FILE__, __LINE__);
  }
  cudaFree(cpad);
  cudaFree(aimg);
  return rc;
}

int boa_debug_quantise(const float* logits, size_t rows, uint32_t* cdf, void* cuda_stream) {
  if (!logits || !cdf || rows == 0) return BOA_E_ARG;
  BOA_TRY(check_device());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  TmpDev tl, tc;
  BOA_TRY(tl.init(logits, rows * 256 * 4, true, false, st));
  BOA_TRY(tc.init(cdf, rows * 257 * 4, false, true, st));
  k_debug_quantise<<<(unsigned)((rows * 32 + 255) / 256), 256, 0, st>>>(static_cast<const float*>(tl.dev),
                                                                       static_cast<uint32_t*>(tc.dev), rows);
  BOA_CUDA_TRY(cudaGetLastError());
  BOA_TRY(tc.finish(st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  return BOA_OK;
}

int boa_debug_rc_encode(const uint32_t* cdf, const uint8_t* syms, size_t n_streams, size_t len, uint8_t* out,
                        size_t cap, uint32_t* sizes, void* cuda_stream) {
  if (!cdf || !syms || !out || !sizes || n_streams == 0 || len == 0 || cap < 16 || cap >= (1ull << 32) ||
      len >= (1ull << 31))
    return BOA_E_ARG;
  BOA_TRY(check_device());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  TmpDev tc, ts, to, tz, te;
  int err = 0;
  BOA_TRY(tc.init(cdf, n_streams * len * 257 * 4, true, false, st));
  BOA_TRY(ts.init(syms, n_streams * len, true, false, st));
  BOA_TRY(to.init(out, n_streams * cap, false, true, st));
  BOA_TRY(tz.init(sizes, n_streams * 4, false, true, st));
  BOA_TRY(te.init(&err, 4, true, true, st));
  k_debug_rc_encode<<<(unsigned)((n_streams + 63) / 64), 64, 0, st>>>(
      static_cast<const uint32_t*>(tc.dev), static_cast<const uint8_t*>(ts.dev), (int)n_streams, (uint32_t)len,
      static_cast<uint8_t*>(to.dev), (uint32_t)cap, static_cast<uint32_t*>(tz.dev), static_cast<int*>(te.dev));
  BOA_CUDA_TRY(cudaGetLastError());
  BOA_TRY(to.finish(st));
  BOA_TRY(tz.finish(st));
  BOA_TRY(te.finish(st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  return err ? BOA_E_CAPACITY : BOA_OK;
}

int boa_debug_rc_decode(const uint32_t* cdf, const uint8_t* in, size_t cap, const uint32_t* sizes, size_t n_streams,
                        size_t len, uint8_t* syms, void* cuda_stream) {
  if (!cdf || !syms || !in || !sizes || n_streams == 0 || len == 0 || cap < 16 || cap >= (1ull << 32) ||
      len >= (1ull << 31))
    return BOA_E_ARG;
  BOA_TRY(check_device());
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  TmpDev tc, ts, ti, tz, te;
  int err = 0;
  BOA_TRY(tc.init(cdf, n_streams * len * 257 * 4, true, false, st));
  BOA_TRY(ti.init(in, n_streams * cap, true, false, st));
  BOA_TRY(tz.init(sizes, n_streams * 4, true, false, st));
  BOA_TRY(ts.init(syms, n_streams * len, false, true, st));
  BOA_TRY(te.init(&err, 4, true, true, st));
  k_debug_rc_decode<<<(unsigned)((n_streams + 63) / 64), 64, 0, st>>>(
      static_cast<const uint32_t*>(tc.dev), static_cast<const uint8_t*>(ti.dev), (uint32_t)cap,
      static_cast<const uint32_t*>(tz.dev), (int)n_streams, (uint32_t)len, static_cast<uint8_t*>(ts.dev),
      static_cast<int*>(te.dev));
  BOA_CUDA_TRY(cudaGetLastError());
  BOA_TRY(ts.finish(st));
  BOA_TRY(te.finish(st));
  BOA_CUDA_TRY(cudaStreamSynchronize(st));
  return err ? BOA_E_CORRUPT : BOA_OK;
}

}  // extern "C"

// ===================================================================================== allocation-free entry point
// boa_rc_encode_packed_noalloc (include/boa.h): S13e-S15 on given tables - one thread per stream codes into a scratch
// row, a device-side exclusive scan of the sizes, a compaction pass - for callers that must not allocate (CUDA graph
// capture, serving loops).  Everything the existing path keeps in a model's cudaMalloc'ed workspace (per-stream scratch
// rows, offsets, running total and flags) lives in ONE file-scope device array of fixed size; every GPU that loads the
// library holds it until exit.  Its name is a host-side stand-in in host code: the kernels get the device address
// that cudaGetSymbolAddress returns for the current device (looked up once per device, below).
// Every call shares the array: calls that overlap on the GPU (two streams, two threads) race.
#include <mutex>

constexpr size_t kNoAllocScratchBytes = 4u << 20;                      // 4 MiB
constexpr size_t kNoAllocCtrlBytes = 256;                              // [0] u64 payload total, [8] int flags payload / row
static __device__ __align__(256) uint8_t g_noalloc_scratch[kNoAllocScratchBytes];

namespace {

constexpr int kNoAllocMaxDevices = 64;
std::mutex g_noalloc_mu;
uint8_t* g_noalloc_dev[kNoAllocMaxDevices] = {};

// device address of the array on the CURRENT device (set-up: first call on that device)
int noalloc_scratch(uint8_t** out) {
  int dev = 0;
  BOA_CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kNoAllocMaxDevices) return BOA_E_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_noalloc_mu);
  if (!g_noalloc_dev[dev]) {
    void* p = nullptr;
    BOA_CUDA_TRY(cudaGetSymbolAddress(&p, g_noalloc_scratch));
    if (!p) return BOA_E_CUDA;
    g_noalloc_dev[dev] = static_cast<uint8_t*>(p);
  }
  *out = g_noalloc_dev[dev];
  return BOA_OK;
}

size_t noalloc_need(size_t n_streams, size_t cap) { return kNoAllocCtrlBytes + round_up(8 * n_streams, 256) + n_streams * cap; }

// the control words of the shared array start every call at zero (they keep the last call's values otherwise)
__global__ void k_noalloc_clear(uint64_t* ctrl) {
  if (threadIdx.x < kNoAllocCtrlBytes / 8) ctrl[threadIdx.x] = 0;
}
// k_debug_rc_encode with the rows in the scratch array: stream i -> rows + i * cap, its size -> sizes[i] (caller's)
__global__ void k_noalloc_rc_encode(const uint32_t* __restrict__ cdf, const uint8_t* __restrict__ syms, int B, uint32_t len,
                                    uint8_t* rows, uint32_t cap, uint32_t* __restrict__ sizes, int* row_overflow) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= B) return;
  EncState st;
  st.low = 0; st.range = 0xFFFFFFFFu; st.pending = 0; st.wpos = 0; st.cache = 0; st.started = 0;
  ByteSink o;
  o.begin(rows + (size_t)i * cap, 0u);
  for (uint32_t t = 0; t < len; ++t) {
    if (st.wpos + st.pending + 8u > cap) { *row_overflow = 1; sizes[i] = 0; return; }
    const uint32_t* C = cdf + ((size_t)i * len + t) * 257;
    const uint32_t s = syms[(size_t)i * len + t];
    enc_symbol(st, C[s], C[s + 1], o);
  }
  if (st.wpos + st.pending + 8u > cap) { *row_overflow = 1; sizes[i] = 0; return; }
  for (int k = 0; k < 5; ++k) enc_shift_low(st, o);
  sizes[i] = st.wpos;
}
// status[0] = payload bytes, status[1] = flags (bit 0: payload_cap too small, bit 1: a scratch row overflowed)
__global__ void k_noalloc_status(const uint8_t* ctrl, uint64_t* status) {
  status[0] = *reinterpret_cast<const uint64_t*>(ctrl);
  const int* f = reinterpret_cast<const int*>(ctrl + 8);
  status[1] = (f[0] ? 1u : 0u) | (f[1] ? 2u : 0u);
}

}  // namespace

extern "C" {

size_t boa_noalloc_scratch_bytes(void) { return kNoAllocScratchBytes; }

size_t boa_noalloc_max_streams(size_t len) {
  if (len == 0 || len >= (1ull << 30)) return 0;
  const size_t cap = stream_cap(len);
  size_t n = (kNoAllocScratchBytes - kNoAllocCtrlBytes) / (cap + 8);
  while (n > 0 && noalloc_need(n, cap) > kNoAllocScratchBytes) --n;
  return std::min<size_t>(n, kMaxWaveStreams);
}

// No cudaMalloc / cudaFree / allocating routine below: pointer queries, one symbol look-up per device, five launches.
int boa_rc_encode_packed_noalloc(const uint32_t* cdf, const uint8_t* syms, size_t n_streams, size_t len, uint8_t* payload,
                                 size_t payload_cap, uint32_t* sizes, uint64_t* status, void* cuda_stream) {
  if (!cdf || !syms || !payload || !sizes || !status || n_streams == 0 || len == 0) return BOA_E_ARG;
  if (n_streams > boa_noalloc_max_streams(len)) {
    snprintf(last_cuda_error_buf(), 256, "boa_rc_encode_packed_noalloc: %zu streams x %zu symbols need more than the %zu-byte static scratch (at most %zu streams of this length)",
             n_streams, len, kNoAllocScratchBytes, boa_noalloc_max_streams(len));
    return BOA_E_CAPACITY;
  }
  BOA_TRY(check_device());
  // staging a host buffer would need an allocation: every pointer is a device pointer
  if (!is_device_ptr(cdf) || !is_device_ptr(syms) || !is_device_ptr(payload) || !is_device_ptr(sizes) || !is_device_ptr(status))
    return BOA_E_ARG;
  uint8_t* scratch = nullptr;
  BOA_TRY(noalloc_scratch(&scratch));
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const uint32_t cap = stream_cap(len);
  const int B = (int)n_streams;
  uint64_t* total = reinterpret_cast<uint64_t*>(scratch);
  int* flags = reinterpret_cast<int*>(scratch + 8);                 // [0] payload_cap too small, [1] a row overflowed
  uint64_t* off = reinterpret_cast<uint64_t*>(scratch + kNoAllocCtrlBytes);
  uint8_t* rows = scratch + kNoAllocCtrlBytes + round_up(8 * n_streams, 256);
  k_noalloc_clear<<<1, 32, 0, st>>>(total);
  k_noalloc_rc_encode<<<(unsigned)((n_streams + 63) / 64), 64, 0, st>>>(cdf, syms, B, (uint32_t)len, rows, cap, sizes, flags + 1);
  k_wave_offsets<<<1, 1024, 0, st>>>(sizes, off, B, total);
  k_compact<<<(unsigned)((n_streams * 32 + 255) / 256), 256, 0, st>>>(rows, cap, sizes, off, payload, (uint64_t)payload_cap, flags, B);
  k_noalloc_status<<<1, 1, 0, st>>>(scratch, status);
  BOA_CUDA_TRY(cudaPeekAtLastError());
  return BOA_OK;
}

}  // extern "C"

#include "boa_fx.cuh"   // FX1, the deterministic fixed-point pipeline (same translation unit: it reuses the helpers above)
