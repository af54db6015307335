// trex_ttng_tu.cu -- g g -> t t~ + (N-2) g reweighting kernels for ONE (N, precision mode); compiled once per pair with
// -DTREX_TU_N={2,3,4,5} -DTREX_TU_MODE={0 fp64, 1 mixed: amplitudes fp64 + colour sum fp32, 2 fp32} (PAPER.md:1209 fptype d/m/f).
#include "trex_kernels.cuh"

#if TREX_TU_MODE == 0
using TuR = double; using TuRC = double;
#elif TREX_TU_MODE == 1
using TuR = double; using TuRC = float;
#else
using TuR = float; using TuRC = float;
#endif

#define TREX_CAT3(a, b, c, d) a##b##c##d
#define TREX_TU_NAME(stem, n, m) TREX_CAT3(stem, n, _m, m)

namespace trex {

int TREX_TU_NAME(trex_tu_launch_n, TREX_TU_N, TREX_TU_MODE)(const ReweightArgs& a, int npass, unsigned grid, cudaStream_t s) {
  if (npass == 1) k_ttng<TuR, TuRC, TREX_TU_N, 1><<<grid, WARPS * 32, 0, s>>>(a);
  else k_ttng<TuR, TuRC, TREX_TU_N, 2><<<grid, WARPS * 32, 0, s>>>(a);
  return (int)cudaGetLastError();
}

int TREX_TU_NAME(trex_tu_upload_n, TREX_TU_N, TREX_TU_MODE)(const double* C, int count) {
  if (count > 576) return 0;            // ncol = 120 is read from global memory
  return (int)cudaMemcpyToSymbol(c_Ctab, C, sizeof(double) * count);
}

}  // namespace trex
