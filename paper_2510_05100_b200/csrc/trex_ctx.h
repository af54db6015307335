// trex_ctx.h -- process-global context shared by the translation units of librex_trex.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>

#include "../../include/rex_trex.h"

namespace trex {

struct Context {
  cudaStream_t stream = nullptr;
  int precision = 0;
  int table_min_n = 3;               // gluon multiplicities >= this use the fused current-table kernel (trex_set_algorithm)
  int nsm = 0;                       // multiprocessors of the device
  int64_t launches = 0;
  char err[512] = {0};
  // rex_bucket scratch (device) and results of the last call (host)
  void* bucket_scratch = nullptr;
  size_t bucket_scratch_bytes = 0;
  void* bucket_host = nullptr;       // pinned
  uint64_t last_keys[REX_MAX_BUCKETS];
  int last_nbuckets = 0;
  // trex_run / trex_run_host scratch (device)
  void* run_perm = nullptr; size_t run_perm_bytes = 0;
  void* run_blocks = nullptr; size_t run_blocks_bytes = 0;
  void* host_io = nullptr; size_t host_io_bytes = 0;
  void* probe_out = nullptr;
  // colour matrices on the device
  bool colour_ready = false;
  double* C120 = nullptr;            // 120 x 120, global memory
  double* Cfold[3] = {nullptr, nullptr, nullptr};   // folded upper-triangular colour matrices of N = 3, 4, 5 (trex_table_tu.cu)
  int* table_meta[3] = {nullptr, nullptr, nullptr}; // tuple / entry index tables of the current-table kernels
};

Context& ctx();

inline int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(ctx().err, sizeof ctx().err, fmt, ap);
  va_end(ap);
  return code;
}

#define TREX_CUDA_CHECK(expr)                                                                      \
  do {                                                                                             \
    cudaError_t e_ = (expr);                                                                       \
    if (e_ != cudaSuccess)                                                                         \
      return ::trex::fail(e_ == cudaErrorMemoryAllocation ? TREX_ENOMEM : TREX_ECUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
  } while (0)

}  // namespace trex
