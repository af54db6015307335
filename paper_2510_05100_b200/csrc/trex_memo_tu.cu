// trex_memo_tu.cu -- g g -> t t~ + (N-2) g, current-table kernels for ONE (N, precision mode); compiled once per pair
// with -DTREX_TU_N={4,5} -DTREX_TU_MODE={0 fp64, 1 mixed, 2 fp32}. See trex_memo.cuh for the method.
//   k_memo_amps  : one block per event. Phase 1 builds the gluon-current table in shared memory level by level;
//                  phase 2 walks the top line (one thread per helicities x first gluon [x parameter point]) and writes
//                  the colour-flow amplitudes of theta_old / theta_new to the scratch matrix X.
//   k_memo_colour: one block per event. Stages X tiles and the (symmetry-folded) colour matrix in shared memory,
//                  evaluates x^dagger C x per column with 8-row register blocks, sums helicities in a fixed order and
//                  applies the epilogue (normalisation, zero guard, ratio).
#include "trex_kernels.cuh"
#include "trex_memo.cuh"

#if TREX_TU_MODE == 0
using TuR = double; using TuRC = double;
#elif TREX_TU_MODE == 1
using TuR = double; using TuRC = float;
#else
using TuR = float; using TuRC = float;
#endif

#define TREX_CAT4(a, b, c, d) a##b##c##d
#define TREX_TU_NAME(stem, n, m) TREX_CAT4(stem, n, _m, m)

namespace trex {
namespace {

template <int N> struct MemoGeom {
  static constexpr int NC = MemoIdx<N>::falling(N, N);
  static constexpr int NCOLS = (1 << N) * 8;                 // (h, lt, ltb, theta)
  static constexpr int TASKS = N * (2 << N);                 // (first gluon, h, lt)
  static constexpr int PT = N <= 4 ? 2 : 1;                  // parameter points walked by parallel threads (if NPASS = 2)
};

template <class R, int N, int K> __device__ __forceinline__ void build_levels(R* tab, const rvec4<double>* pset) {
  if constexpr (K <= N) {
    constexpr int items = MemoIdx<N>::ncanon(K) << K;
    for (int item = threadIdx.x; item < items; item += blockDim.x) memo_build_item<R, N, K>(tab, pset, item);
    __syncthreads();
    build_levels<R, N, K + 1>(tab, pset);
  }
}

template <class R, int N, int NPASS>
__global__ void __launch_bounds__(MemoGeom<N>::TASKS * (NPASS == 2 ? MemoGeom<N>::PT : 1), 1)
k_memo_amps(const ReweightArgs a, double* __restrict__ X, long ev0) {
  using G = MemoGeom<N>;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  rvec4<double>* pset = reinterpret_cast<rvec4<double>*>(smem_raw);
  R* tab = reinterpret_cast<R*>(smem_raw + sizeof(rvec4<double>) * (1 << N));
  const long e = ev0 + blockIdx.x;
  const int tid = threadIdx.x;
  for (int s = tid; s < (1 << N); s += blockDim.x) memo_pset_item<N>(a.mom, a.ld, e, (unsigned)s, pset);
  for (int it = tid; it < 2 * N; it += blockDim.x) memo_level1_item<R, N>(a.mom, a.ld, e, it, tab);
  __syncthreads();
  build_levels<R, N, 2>(tab, pset);
  // walk: lanes of a warp share (pass, first gluon) and differ in (h, lt) only -> uniform control flow
  constexpr int NHL = 2 << N;
  const int hl = tid % NHL, g1 = (tid / NHL) % N, ppar = tid / G::TASKS;
  double* Xev = X + (long)blockIdx.x * G::NCOLS * G::NC * 2;
  constexpr int PSTEP = NPASS == 2 ? G::PT : 1;
  for (int pass = ppar; pass < NPASS; pass += PSTEP)
    memo_walk_task<R, N>(tab, pset, a.mom, a.ld, e, a.T.mt, a.T.mGt, a.T.kq, (unsigned)(hl >> 1), hl & 1, g1, pass, NPASS, Xev);
}

// folded colour matrix C'(i,j) = 0 (j < i), C_ii (j == i), 2 C_ij (j > i), stored by rows i for j >= 8 floor(i/8)
template <int NC> struct FoldedC {
  static constexpr int NB = NC / 8;
  __host__ __device__ static constexpr int row_len(int i) { return NC - 8 * (i / 8); }
  __host__ __device__ static constexpr int size() { int s = 0; for (int i = 0; i < NC; ++i) s += row_len(i); return s; }
};

template <class RC, int NC, int COLS, int TPC>
__global__ void __launch_bounds__(COLS * TPC) k_memo_colour(const ReweightArgs a, const double* __restrict__ X, const double* __restrict__ Cfold, long ev0, int ncols) {
  using F = FoldedC<NC>;
  constexpr int NB = F::NB, XS = COLS + 1;
  extern __shared__ __align__(16) unsigned char smem_raw[];
  RC* Cp = reinterpret_cast<RC*>(smem_raw);
  cx<RC>* xs = reinterpret_cast<cx<RC>*>(smem_raw + ((sizeof(RC) * F::size() + 15) / 16) * 16);
  __shared__ double red[COLS * TPC / 32][2];
  const int tid = threadIdx.x, c = tid % COLS, q = tid / COLS;
  for (int i = tid; i < F::size(); i += blockDim.x) Cp[i] = RC(Cfold[i]);
  const double* Xev = X + (long)blockIdx.x * ncols * NC * 2;
  RC acc = RC(0);
  for (int tile = 0; tile < ncols; tile += COLS) {
    __syncthreads();
    for (int idx = tid; idx < COLS * NC; idx += blockDim.x) {
      const int col = idx / NC, sg = idx - col * NC;
      const double2 v = *reinterpret_cast<const double2*>(Xev + ((long)(tile + col) * NC + sg) * 2);
      xs[sg * XS + col] = cx<RC>(RC(v.x), RC(v.y));
    }
    __syncthreads();
    // row blocks of this thread: pairs (p, NB-1-p) with p % TPC == q, plus the middle block
    for (int p = q; 2 * p < NB; p += TPC) {
      for (int side = 0; side < 2; ++side) {
        const int b = side == 0 ? p : NB - 1 - p;
        if (side == 1 && b == p) break;
        cx<RC> t[8];
#pragma unroll
        for (int r = 0; r < 8; ++r) t[r] = cx<RC>(RC(0), RC(0));
        const RC* row = Cp;                       // start of row i
        const int iend = 8 * b + 8;
#pragma unroll 2
        for (int i = 0; i < iend; ++i) {
          const cx<RC> xi = xs[i * XS + c];
          const RC* cr = row + (8 * b - 8 * (i >> 3));
#pragma unroll
          for (int r = 0; r < 8; ++r) cfma(t[r], xi, cr[r]);
          row += F::row_len(i);
        }
#pragma unroll
        for (int r = 0; r < 8; ++r) { const cx<RC> xj = xs[(8 * b + r) * XS + c]; acc += xj.re * t[r].re + xj.im * t[r].im; }
      }
    }
  }
  // fixed-order reduction: column parity = theta; xor-shuffles by even offsets keep the parity
  double v = (double)acc;
#pragma unroll
  for (int off = 16; off >= 2; off >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, off);
  if ((tid & 31) < 2) red[tid >> 5][tid & 1] = v;
  __syncthreads();
  if (tid == 0) {
    double s0 = 0.0, s1 = 0.0;
    for (int w = 0; w < COLS * TPC / 32; ++w) { s0 += red[w][0]; s1 += red[w][1]; }
    const long e = ev0 + blockIdx.x;
    const double mo = s0 * a.T.pref[0], mn = s1 * a.T.pref[1];
    const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
    a.w_out[e] = a.w_in[e] * norm * mn;                        // evaluate + append_wgts
    if (a.me2_old) a.me2_old[e] = mo;
    if (a.me2_new) a.me2_new[e] = mn;
  }
}

template <int N> struct ColourGeom;
template <> struct ColourGeom<4> { static constexpr int COLS = 128, TPC = 1; };
template <> struct ColourGeom<5> { static constexpr int COLS = 64, TPC = 4; };

}  // namespace

// scratch bytes per event of X
size_t TREX_TU_NAME(trex_tu_memo_xbytes_n, TREX_TU_N, TREX_TU_MODE)() {
  return sizeof(double) * 2 * MemoGeom<TREX_TU_N>::NCOLS * MemoGeom<TREX_TU_N>::NC;
}

// amplitudes + colour sum + epilogue for events [ev0, ev0 + nev) of the block described by `a`; X holds nev events
int TREX_TU_NAME(trex_tu_memo_launch_n, TREX_TU_N, TREX_TU_MODE)(const ReweightArgs& a, int npass, double* X, const double* Cfold,
                                                                 long ev0, long nev, cudaStream_t s) {
  constexpr int N = TREX_TU_N;
  using G = MemoGeom<N>;
  using CG = ColourGeom<N>;
  const size_t smemA = sizeof(rvec4<double>) * (1 << N) + sizeof(TuR) * 8 * MemoIdx<N>::NE;
  const size_t smemB = ((sizeof(TuRC) * FoldedC<G::NC>::size() + 15) / 16) * 16 + sizeof(cx<TuRC>) * G::NC * (CG::COLS + 1);
  static bool configured = false;
  if (!configured) {
    cudaFuncSetAttribute(k_memo_amps<TuR, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemA);
    cudaFuncSetAttribute(k_memo_amps<TuR, N, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemA);
    cudaFuncSetAttribute(k_memo_colour<TuRC, G::NC, CG::COLS, CG::TPC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smemB);
    configured = true;
  }
  if (npass == 1) k_memo_amps<TuR, N, 1><<<(unsigned)nev, G::TASKS, smemA, s>>>(a, X, ev0);
  else k_memo_amps<TuR, N, 2><<<(unsigned)nev, G::TASKS * G::PT, smemA, s>>>(a, X, ev0);
  k_memo_colour<TuRC, G::NC, CG::COLS, CG::TPC><<<(unsigned)nev, CG::COLS * CG::TPC, smemB, s>>>(a, X, Cfold, ev0, G::NCOLS);
  return (int)cudaGetLastError();
}

}  // namespace trex
