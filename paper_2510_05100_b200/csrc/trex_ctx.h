// trex_ctx.h -- process-global context shared by the translation units of librex_trex.so (not part of the ABI).
#pragma once
#include <cuda_runtime.h>

#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <vector>

#include "../../include/rex_trex.h"
#include "../../include/rex_trex_diag.h"

namespace trex {

// Device-resident plan of one trex_run: where every compiled-in subprocess finds its events in bucketed order. Written
// by the last kernel of rex_bucket's chain, read by every later kernel of the run -- the host never waits for it.
struct DevPlan {
  long long off[TREX_NSUBPROC];   // first event of the subprocess's bucket in bucketed order
  long long cnt[TREX_NSUBPROC];   // events of that bucket (0: subprocess absent from the sample, or leg count mismatch)
  int single;                     // 1: the sample is ONE known class -> kernels work on the caller's arrays, no transposition
  int nb;
};

struct Context {
  cudaStream_t stream = nullptr;
  int precision = 0;
  int table_min_n = 3;               // gluon multiplicities >= this use the fused current-table kernel (trex_set_algorithm)
  int nsm = 0;                       // multiprocessors of the device
  int64_t launches = 0;
  // diagnostics: CUDA events around every |M|^2 launch (trex_kernel_timing); implies no graph replay
  double* dbg_out = nullptr;         // device buffer of trex_debug_xtile while it runs, else nullptr
  bool ktiming = false;
  std::vector<cudaEvent_t> kev;      // start/stop pairs recorded since the last trex_kernel_time
  std::vector<cudaEvent_t> kev_pool; // events free for reuse
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
  void* poly_tmp = nullptr; size_t poly_tmp_bytes = 0;   // trex_run_multi: |M|^2 at three kappa values + the u_k
  bool poly_multi = true;
  bool hel_sym = true;               // trex_set_helicity_symmetry
  void* xsec_scratch = nullptr; void* xsec_host = nullptr;   // trex_xsec_moments: block partials (device), result (pinned)
  // trex_run replayed as a CUDA graph when it is called again with the same buffers, sizes and parameter points
  struct RunKey {
    const void* ptr[6]; int64_t n, ld; int npar, precision, table_min_n, hel_sym; double th[2 * TREX_NTHETA];
  };
  bool in_host_run = false;
  // trex_run_alphas: its passes run the path at g_s = 1 with these kappa / g_s in the theta_old / theta_new slots
  bool unit_gs = false; double unit_gs_kq[2] = {0.0, 0.0};
  RunKey last_key{}; bool last_key_valid = false;
  RunKey exec_key{}; bool exec_valid = false; bool graphs_ok = true;
  cudaGraphExec_t run_exec = nullptr; int64_t exec_launches = 0; int64_t graph_replays = 0;
  cudaStream_t cap_stream = nullptr;
  cudaStream_t copy_stream = nullptr; cudaEvent_t copy_ev[2] = {nullptr, nullptr};   // trex_run_host: transfers beside the kernels
  DevPlan* plan = nullptr;           // device
  void* plan_keys = nullptr;         // device: key, leg count [2 NSUB] and process string [NSUB][8] of every compiled-in subprocess
  const int8_t* legmap = nullptr;    // trex_run_pdg: per-event leg order (device [npar][n]); forces the transposition
  void* pdg_tmp = nullptr; size_t pdg_tmp_bytes = 0;   // trex_run_pdg: keys + leg maps
  // colour matrices on the device
  bool colour_ready = false;
  double* C120 = nullptr;            // 120 x 120, global memory
  double* Cfold[3][3] = {};          // folded upper-triangular colour matrices of N = 3, 4, 5 per precision mode (trex_table_tu.cu)
  int* table_meta[3] = {nullptr, nullptr, nullptr}; // tuple / entry index tables of the current-table kernels
};

Context& ctx();

// rex_bucket in two halves (rex_bucket.cu): enqueue the kernel chain (+ the device plan for a run over `npar`-leg events,
// if sub_keys != nullptr), then fetch sizes and keys -- the only point where the host waits for the device
int bucket_reserve(int64_t n);          // (re)allocates the scratch of bucket_enqueue; never called while capturing
int bucket_enqueue(const uint64_t* keys, int64_t n, int32_t* perm, int npar, int32_t* inv);   // inv (nullable): inverse permutation
int ensure_plan();                      // uploads the subprocess registry the device plan and rex_keys need (trex_api.cu)
int bucket_finish(int64_t* offsets);
// transposition kernels of trex_run driven by the device plan (both are no-ops for a single-class sample)
int run_gather(const double* mom, int64_t ld, const double* w_in, int64_t n, int nrows, const int32_t* inv, double* blk, double* res);   // ld: row stride of mom
int run_scatter(const double* res, int64_t n, const int32_t* perm, double* w_out, double* me2_old, double* me2_new);

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
