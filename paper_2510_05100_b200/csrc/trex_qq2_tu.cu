// trex_qq2_tu.cu -- kernel of the one-light-line channels with two gluons (trex_qq2.cuh; ids TREX_SP_UUX_TTGG ..).
//
// A block is 32 consecutive events x 4 warps. On the massless light line only two helicity combinations c survive (see
// k_qq in trex_api.cu), so the sum runs over (c, lambda_a, lambda_b) x lambda_t x lambda_tbar = 8 x 2 x 2: a warp takes two
// of the eight (c, lambda_a, lambda_b) one after the other, with the top helicity looped inside and both antitop helicities
// closed at the leaves. The 96 flow amplitudes of a thread live in shared memory (96 KB per block in fp64: two blocks per
// SM). Fixed-order reduction over the warps and the epilogue of PAPER.md:785-808 finish inside the launch. Inside trex_run
// ONE launch serves every two-gluon quark class of the plan.
#include "trex_kernels.cuh"
#include "trex_qq2.cuh"

namespace trex {
namespace {

__constant__ QLineLegs c_q2legs[TREX_NSUBPROC];
__constant__ double c_q2invnavg[TREX_NSUBPROC];      // 1 / N_avg; 0 for ids that are not two-gluon quark channels

#ifndef TREX_QQ2_MINB
#define TREX_QQ2_MINB 2
#endif
constexpr int Q2_WARPS = 4, Q2_TB = Q2_WARPS * 32;
template <class R> constexpr size_t q2_smem() { return sizeof(R) * Qq2Acc<R>::NEL * Q2_TB; }

// DBG: the instantiation trex_debug_helicity_me2 launches -- the same code with the per-helicity dump compiled in
template <class R, class RC, bool DBG = false>
__global__ void __launch_bounds__(Q2_TB, TREX_QQ2_MINB) k_qq2(const ReweightArgs a) {
  extern __shared__ __align__(16) unsigned char q2_raw[];
  __shared__ double red[2][Q2_WARPS][32];
  int sid = a.sid;
  long blk = blockIdx.x;
  if (a.plan && a.qfamily) {
    sid = -1;
    for (int s = 0; s < TREX_NSUBPROC; ++s) {
      if (c_q2invnavg[s] == 0.0) continue;
      const long nb = (a.plan->cnt[s] + 31) >> 5;
      if (blk < nb) { sid = s; break; }
      blk -= nb;
    }
    if (sid < 0) return;
  }
  const EvIO io = resolve_io(a, sid);
  if (blk * 32 >= io.n) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long e = blk * 32 + lane;
  const long ev = e < io.n ? e : io.n - 1;
  double pm[6][4];
#pragma unroll
  for (int l = 0; l < 6; ++l)
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) pm[l][mu] = io.mom[(long)(l * 4 + mu) * io.ld + ev];
  const Qq2Acc<R> fl{reinterpret_cast<R*>(q2_raw) + threadIdx.x, Q2_TB};
  RC acc[2] = {RC(0), RC(0)};
  // helicity symmetry (a.hsym): the four choices with light-line combination c = 0 stand for their parity partners
  const int nhalf = (a.hsym && !DBG) ? 1 : 2;
#pragma unroll 1
  for (int half = 0; half < nhalf; ++half) {
    const int u = nhalf == 1 ? 2 * warp : warp + Q2_WARPS * half;        // (c, lambda_a, lambda_b)
    RC o[2];
    qq2_unit<R, RC>(pm, c_q2legs[sid], u & 1, (u >> 1) & 1, (u >> 2) & 1, a.T, fl, o, (DBG && a.dbg && e == 0) ? a.dbg + u * 8 : nullptr);
    acc[0] += o[0]; acc[1] += o[1];
  }
  red[0][warp][lane] = (double)acc[0]; red[1][warp][lane] = (double)acc[1];
  __syncthreads();
  if (warp == 0 && e < io.n) {
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int w = 0; w < Q2_WARPS; ++w) { s0 += red[0][w][lane]; s1 += red[1][w][lane]; }
    const double hs = nhalf == 1 ? 2.0 : 1.0;
    const double mo = s0 * (a.T.gs2nv[0] * c_q2invnavg[sid] * hs), mn = s1 * (a.T.gs2nv[1] * c_q2invnavg[sid] * hs);
    const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
    io.w_out[e] = io.w_in[e] * norm * mn;                      // evaluate + append_wgts
    if (io.me2_old) io.me2_old[e] = mo;
    if (io.me2_new) io.me2_new[e] = mn;
  }
}

}  // namespace

int trex_tu_qq2_setup(const QLineLegs* legs, const double* invnavg, const double* C144) {
  if (cudaMemcpyToSymbol(c_q2legs, legs, sizeof(QLineLegs) * TREX_NSUBPROC) != cudaSuccess) return 1;
  if (cudaMemcpyToSymbol(c_q2invnavg, invnavg, sizeof(double) * TREX_NSUBPROC) != cudaSuccess) return 1;
  if (cudaMemcpyToSymbol(c_Ctab, C144, sizeof(double) * 144) != cudaSuccess) return 1;
  return 0;
}

int trex_tu_qq2_launch(const ReweightArgs& a, int mode, unsigned grid, cudaStream_t stream) {
  static bool ready = false;
  if (!ready) {
    if (cudaFuncSetAttribute(k_qq2<double, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q2_smem<double>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_qq2<double, double, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q2_smem<double>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_qq2<double, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q2_smem<double>()) != cudaSuccess ||
        cudaFuncSetAttribute(k_qq2<float, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)q2_smem<float>()) != cudaSuccess)
      return 1;
    ready = true;
  }
  if (mode == 0 && a.dbg) k_qq2<double, double, true><<<grid, Q2_TB, q2_smem<double>(), stream>>>(a);
  else if (mode == 0) k_qq2<double, double><<<grid, Q2_TB, q2_smem<double>(), stream>>>(a);
  else if (mode == 1) k_qq2<double, float><<<grid, Q2_TB, q2_smem<double>(), stream>>>(a);
  else k_qq2<float, float><<<grid, Q2_TB, q2_smem<float>(), stream>>>(a);
  return cudaGetLastError() == cudaSuccess ? 0 : 1;
}

}  // namespace trex
