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
constexpr uint32_t kArithVersion = 0x42320001u;

#define BOA_CUDA_TRY(expr)                      \
  do {                                          \
    cudaError_t _e = (expr);                    \
    if (_e != cudaSuccess) {                    \
      (void)cudaGetLastError();                 \
      return (_e == cudaErrorMemoryAllocation) ? BOA_E_NOMEM : BOA_E_CUDA; \
    }                                           \
  } while (0)

#define BOA_TRY(expr)            \
  do {                           \
    int _r = (expr);             \
    if (_r != BOA_OK) return _r; \
  } while (0)

__host__ __device__ inline size_t round_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

}  // namespace boa
