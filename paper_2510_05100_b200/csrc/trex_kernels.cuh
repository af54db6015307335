// trex_kernels.cuh -- launch geometry shared by every |M|^2 kernel.
//
// A block is 32 consecutive events (one per lane, so every momentum component is one coalesced 256-byte row read per
// warp) times WARPS warps; the warps split the helicity units of those events between them, each thread accumulating
// its units' J^dagger C J for theta_old and theta_new. A fixed-order shared-memory reduction over the warps and the
// epilogue (normalisation, zero guard, ratio) finish inside the same launch: one launch per
// trex_reweight call, deterministic results.
#pragma once
#include <cuda_runtime.h>

#include "trex_ctx.h"
#include "trex_proc.cuh"

namespace trex {

constexpr int WARPS = 8;

struct EvIO {
  const double* mom; long n; long ld;   // ld = row stride of the SoA block (== n for a caller-provided block)
  const double* w_in; double* w_out; double* me2_old; double* me2_new;
};
struct ReweightArgs {
  EvIO io;                 // the caller's arrays (trex_reweight; single-class samples in trex_run)
  EvIO alt;                // trex_run's scratch in bucketed order (mom, w_in, results), ld = sample size
  const DevPlan* plan;     // trex_run: device-resident bucket ranges; nullptr for trex_reweight
  int sid;
  int hsym;                // 1: sum one helicity configuration of every parity pair {h, -h} and double (valid for Gamma_t = 0 at
                           // both parameter points: DESIGN.md R-21); honoured by k_gg_tt, k_table<3>, k_table4w<., ., 1>, k_table<5>, k_qq and k_qq2
  int qfamily;             // k_qq inside trex_run: one launch serves every quark-channel class of the plan
  const double* C120;
  ThetaPair T;
  QLineLegs q;
  // diagnostics (trex_debug_xtile): when set, the production kernels copy the colour-flow amplitudes of event 0 here
  // before the colour sum -- [iteration][flow][column][re, im]; nullptr in every product call
  double* dbg;
};

// which events this launch works on: decided on the device for trex_run (the host has not seen the bucket sizes)
__device__ __forceinline__ EvIO resolve_io(const ReweightArgs& a, int sid = -1) {
  EvIO io = a.io;
  if (sid < 0) sid = a.sid;
  if (a.plan) {
    const long off = a.plan->off[sid], cnt = a.plan->cnt[sid];
    if (!a.plan->single) {
      io = a.alt;
      io.mom += off; io.w_in += off; io.w_out += off; io.me2_old += off; io.me2_new += off;
    }
    io.n = cnt;
  }
  return io;
}

// fixed-order reduction over the warps of a block + epilogue by warp 0
template <class RC, int NW = WARPS> __device__ __forceinline__ void reduce_and_finish(const ReweightArgs& a, const EvIO& io, RC acc0, RC acc1, long e) {
  __shared__ double red[2][NW][32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  red[0][warp][lane] = (double)acc0; red[1][warp][lane] = (double)acc1;
  __syncthreads();
  if (warp == 0 && e < io.n) {
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) { s0 += red[0][w][lane]; s1 += red[1][w][lane]; }
    const double mo = s0 * a.T.pref[0], mn = s1 * a.T.pref[1];
    const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
    io.w_out[e] = io.w_in[e] * norm * mn;                        // evaluate + append_wgts
    if (io.me2_old) io.me2_old[e] = mo;
    if (io.me2_new) io.me2_new[e] = mn;
  }
}

// warps per block and resident blocks per SM the register allocation is sized for
#ifndef TREX_N2_WARPS
#define TREX_N2_WARPS 2
#endif
#ifndef TREX_N2_MINB
#define TREX_N2_MINB 4
#endif
template <int N> struct TtngGeom { static constexpr int NW = N == 2 ? TREX_N2_WARPS : WARPS, MINB = N == 2 ? TREX_N2_MINB : 1; };

template <class R, class RC, int N, int NPASS>
__global__ void __launch_bounds__(TtngGeom<N>::NW * 32, TtngGeom<N>::MINB) k_ttng(const ReweightArgs a) {
  constexpr int NU = 1 << (N + 1), WARPS = TtngGeom<N>::NW;
  const EvIO io = resolve_io(a);
  if ((long)blockIdx.x * 32 >= io.n) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long e = (long)blockIdx.x * 32 + lane;
  const long ev = e < io.n ? e : io.n - 1;
  RC acc[2] = {RC(0), RC(0)};
  for (int u = warp; u < NU; u += WARPS) {
    RC out[2];
    ttng_unit<R, RC, N, NPASS>(io.mom, io.ld, ev, u >> 1, (u & 1) ? 1 : -1, a.T, a.C120, out);
    acc[0] += out[0]; acc[1] += out[1];
  }
  reduce_and_finish<RC, WARPS>(a, io, acc[0], acc[1], e);
}

// one translation unit per (N, precision mode): trex_ttng_tu.cu compiled with -DTREX_TU_N=.. -DTREX_TU_MODE=..
using TtngLaunchFn = int (*)(const ReweightArgs&, int npass, unsigned grid, cudaStream_t stream);
using TtngUploadFn = int (*)(const double* C, int count);
#define TREX_TU_DECL(N, M)                                                                   \
  int trex_tu_launch_n##N##_m##M(const ReweightArgs&, int npass, unsigned grid, cudaStream_t); \
  int trex_tu_upload_n##N##_m##M(const double* C, int count);
TREX_TU_DECL(2, 0) TREX_TU_DECL(2, 1) TREX_TU_DECL(2, 2)
TREX_TU_DECL(3, 0) TREX_TU_DECL(3, 1) TREX_TU_DECL(3, 2)
TREX_TU_DECL(4, 0) TREX_TU_DECL(4, 1) TREX_TU_DECL(4, 2)
TREX_TU_DECL(5, 0) TREX_TU_DECL(5, 1) TREX_TU_DECL(5, 2)
#undef TREX_TU_DECL

// one light line + two gluons (trex_qq2_tu.cu): tables (legs, 1 / N_avg per id, 12 x 12 colour matrix) and launch
int trex_tu_qq2_setup(const QLineLegs* legs, const double* invnavg, const double* C144);
int trex_tu_qq2_launch(const ReweightArgs& a, int mode, unsigned grid, cudaStream_t stream);

// fused current-table kernels (trex_table_tu.cu), one translation unit per (N = 3, 4, 5; precision mode)
using TableLaunchFn = int (*)(const ReweightArgs&, int npass, long nmax, const int* meta, const double* Cfold, int nsm, cudaStream_t);
using TableMetaFn = int (*)(int* meta);                       // fills the meta block (if non-null), returns its size in ints
using TableFoldFn = int (*)(const double* C, double* f);      // fills the folded colour matrix (if non-null), returns its size
using TableGeomFn = int (*)(int* out);                        // {NFIX, iterations, lambda_t passes, flows, columns} of the X-tile dump
#define TREX_TABLE_DECL(N, M)                                                                                       \
  int trex_tu_table_launch_n##N##_m##M(const ReweightArgs&, int npass, long nmax, const int* meta, const double* Cfold, int nsm, cudaStream_t); \
  int trex_tu_table_meta_n##N##_m##M(int* meta);                                                                    \
  int trex_tu_table_fold_n##N##_m##M(const double* C, double* f);                                                   \
  int trex_tu_table_geom_n##N##_m##M(int* out);
TREX_TABLE_DECL(3, 0) TREX_TABLE_DECL(3, 1) TREX_TABLE_DECL(3, 2)
TREX_TABLE_DECL(4, 0) TREX_TABLE_DECL(4, 1) TREX_TABLE_DECL(4, 2)
TREX_TABLE_DECL(5, 0) TREX_TABLE_DECL(5, 1) TREX_TABLE_DECL(5, 2)
#undef TREX_TABLE_DECL

}  // namespace trex
