// common.cuh — constants and small helpers shared by the CUDA translation unit.
// Product code: nothing here (or anywhere under csrc/) includes or links anything from oracle/.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace boa {

constexpr int kNState = 16;          // d_state N; the scan kernel holds 16 h values per thread
constexpr int kDConv = 4;            // d_conv K
constexpr int kFreqBits = 16;        // M = 2^16 (eq. 7; BASELINE.json)
constexpr uint32_t kM = 1u << kFreqBits;
constexpr uint32_t kGOne = 1u << 23; // quantiser scale (R#5)
constexpr uint32_t kRcTop = 1u << 24;// renormalise while range < 2^24 (R#6)
constexpr float kEps = 1e-5f;        // RMSNorm epsilon (R#10)

// Arithmetic generation of the step kernels: part of the container fingerprint because the tables
// are only reproducible with the same per-step floating-point arithmetic.
// 'B2' + generation number.  Bump whenever any kernel upstream of the quantiser changes its
// arithmetic (operation order, fusion, precision).
constexpr uint32_t kArithVersion = 0x42320008u;

// Programmatic dependent launch (PDL): a kernel launched with the programmatic-serialization attribute may start
// while its predecessor in the stream is still draining; pdl_wait() blocks until the predecessor grid has completed
// and its memory is visible (every thread that touches data produced upstream calls it first); pdl_launch() lets the
// successor's CTAs be scheduled as soon as SMs free up.  Without the attribute both are no-ops.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }

// Last CUDA failure seen by this thread ("file:line: cudaErrorName"), for boa_last_cuda_error().
inline char* last_cuda_error_buf() {
  static thread_local char buf[256] = "";
  return buf;
}
inline int note_cuda_error(cudaError_t e, const char* file, int line);

#define BOA_CUDA_TRY(expr)                      \
  do {                                          \
    cudaError_t _e = (expr);                    \
    if (_e != cudaSuccess) return boa::note_cuda_error(_e, __FILE__, __LINE__); \
  } while (0)

#define BOA_TRY(expr)            \
  do {                           \
    int _r = (expr);             \
    if (_r != BOA_OK) return _r; \
  } while (0)

}  // namespace boa
#include <stdio.h>
#include "../../include/boa.h"
namespace boa {
inline int note_cuda_error(cudaError_t e, const char* file, int line) {
  const char* slash = file;
  for (const char* c = file; *c; ++c) if (*c == '/') slash = c + 1;
  snprintf(last_cuda_error_buf(), 256, "%s:%d: %s", slash, line, cudaGetErrorName(e));
  (void)cudaGetLastError();
  return (e == cudaErrorMemoryAllocation) ? BOA_E_NOMEM : BOA_E_CUDA;
}

__host__ __device__ inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace boa
