// trex_table_tu.cu -- g g -> t t~ + (N-2) g, fused current-table kernel for ONE (N, precision mode); compiled once per
// pair with -DTREX_TU_N={3,4,5} -DTREX_TU_MODE={0 fp64, 1 mixed, 2 fp32}. See trex_table.cuh for the method.
//   k_table: persistent blocks, one event at a time per block. Per event and per outer helicity iteration:
//     phase 1  gluon-current table, level by level, in shared memory               (a6, a7)
//     phase 2  top-line walk, one thread per (ordering prefix, free helicities, lambda_t [, theta]); colour-flow
//              amplitudes x_sigma(theta_old), x_sigma(theta_new) of both antitop helicities -> X tile in shared memory (a7)
//     phase 3  x^dagger C x per X column with the symmetry-folded colour matrix held in shared memory,
//              8-row register blocks                                                (a8)
//   then a fixed-order block reduction and the epilogue (normalisation, zero guard, ratio)  (a9).
// Nothing but the momenta is read from, and nothing but the three results is written to, global memory.
#include "trex_kernels.cuh"
#include "trex_table.cuh"

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

template <int N> struct TabCfg;
template <> struct TabCfg<3> { static constexpr int NFIX = 0, D = 2, TB = 96; };
template <> struct TabCfg<4> { static constexpr int NFIX = 0, D = 2, TB = 256; };
template <> struct TabCfg<5> { static constexpr int NFIX = 3, D = 3, TB = 256; };

template <int NC> struct FoldedC {
  // C'(i,j) = 0 (j < i), C_ii (j == i), 2 C_ij (j > i), stored by rows i for j >= RB floor(i/RB)
  static constexpr int RB = NC % 8 == 0 ? 8 : NC;            // rows per register block (NC = 6: one block)
  static constexpr int NB = NC / RB;
  __host__ __device__ static constexpr int row_len(int i) { return NC - RB * (i / RB); }
  __host__ __device__ static constexpr int size() { int s = 0; for (int i = 0; i < NC; ++i) s += row_len(i); return s; }
};

template <class R, class RC, int N> struct TabGeom {
  using Cfg = TabCfg<N>;
  using I = TabIdx<N, Cfg::NFIX>;
  static constexpr int NFIX = Cfg::NFIX, D = Cfg::D, TB = Cfg::TB;
  static constexpr int NE = I::NE;
  static constexpr int NC = I::falling(N, N);
  static constexpr int NIT = 1 << NFIX;
  static constexpr int NHL = 2 << I::NFREE;                  // (free helicities, lambda_t)
  static constexpr int NPREF = I::falling(N, D);
  static constexpr int NTASK = NPREF * NHL;
  static constexpr int NCOLT = NHL * 4;                      // X tile columns: (hfree, lt, ltb, theta)
  static constexpr int XS = NCOLT + 1;
  static constexpr int NSUB = 1 << N;
  // shared-memory carve-up (bytes, every region 16-byte aligned)
  static constexpr size_t al(size_t x) { return (x + 15) / 16 * 16; }
  static constexpr size_t o_tab = 0;
  static constexpr size_t o_x = o_tab + al(sizeof(R) * TAB_NCOMP * NE);
  static constexpr size_t o_c = o_x + al(sizeof(cx<RC>) * NC * XS);
  static constexpr size_t o_pset = o_c + al(sizeof(RC) * FoldedC<NC>::size());
  static constexpr size_t o_eps = o_pset + al(sizeof(rvec4<double>) * NSUB);
  static constexpr size_t o_spin = o_eps + al(sizeof(double) * 16 * N);
  static constexpr size_t o_meta = o_spin + al(sizeof(double) * 8 * 4);
  static constexpr size_t o_red = o_meta + al(sizeof(int) * I::M_SIZE);
  static constexpr size_t bytes = o_red + al(sizeof(double) * 2 * (TB / 32));
};

// leaf sink of the walk: x_sigma = A0 + (kappa/g_s) A1 for both antitop helicities -> X tile
template <class R, class RC, int XS> struct TabLeafStore {
  cx<RC>* xs;
  const double* vsp;         // v(p_tbar, -), v(p_tbar, +): 2 x 4 complex
  int colbase;               // ((hfree * 2 + lt) * 2 + 0) * 2 + 0
  int leaf0;                 // rank of the first ordering below this task's prefix
  int th_lo, th_hi;          // parameter points this task writes
  R kq[2];
  __device__ __forceinline__ void operator()(int leaf, const spinor<R>& b0, const spinor<R>& b1) {
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) {
      spinor<R> v;
#pragma unroll
      for (int i = 0; i < 4; ++i) v.c[i] = cx<R>(R(vsp[iv * 8 + 2 * i]), R(vsp[iv * 8 + 2 * i + 1]));
      const cx<R> a0 = row_col(b0, v), a1 = row_col(b1, v);
      for (int th = th_lo; th < th_hi; ++th) {
        cx<R> x = a0; cfma(x, a1, kq[th]);
        xs[(leaf0 + leaf) * XS + colbase + iv * 2 + th] = cx<RC>(RC(x.re), RC(x.im));
      }
    }
  }
};

template <class R, int N, int NFIX, int K> __device__ __forceinline__ void build_levels(R* tab, const int* meta, const rvec4<double>* pset) {
  using I = TabIdx<N, NFIX>;
  if constexpr (K <= N) {
    const int e1 = meta[I::M_LVL + K + 1];
    for (int e = meta[I::M_LVL + K] + threadIdx.x; e < e1; e += blockDim.x) tab_build_entry<R, N, NFIX, K>(tab, meta, pset, e);
    __syncthreads();
    build_levels<R, N, NFIX, K + 1>(tab, meta, pset);
  }
}

template <class R, class RC, int N, int NPASS>
__global__ void __launch_bounds__(TabCfg<N>::TB, 1) k_table(const ReweightArgs a, const int* __restrict__ gmeta, const double* __restrict__ Cfold) {
  using G = TabGeom<R, RC, N>;
  using I = typename G::I;
  using F = FoldedC<G::NC>;
  constexpr int NFIX = G::NFIX, D = G::D, TB = G::TB, XS = G::XS;
  extern __shared__ __align__(16) unsigned char smem[];
  R* tab = reinterpret_cast<R*>(smem + G::o_tab);
  cx<RC>* xs = reinterpret_cast<cx<RC>*>(smem + G::o_x);
  RC* Cs = reinterpret_cast<RC*>(smem + G::o_c);
  rvec4<double>* pset = reinterpret_cast<rvec4<double>*>(smem + G::o_pset);
  double* eps_all = reinterpret_cast<double*>(smem + G::o_eps);
  double* spin = reinterpret_cast<double*>(smem + G::o_spin);
  int* meta = reinterpret_cast<int*>(smem + G::o_meta);
  double* red = reinterpret_cast<double*>(smem + G::o_red);
  const int tid = threadIdx.x;

  for (int i = tid; i < I::M_SIZE; i += TB) meta[i] = gmeta[i];
  for (int i = tid; i < F::size(); i += TB) Cs[i] = RC(Cfold[i]);
  __syncthreads();

  for (long e = blockIdx.x; e < a.n; e += gridDim.x) {
    // ---- per-event set-up: momentum of every gluon subset (incoming convention), polarisation vectors, t / t~ spinors
    for (int sset = tid; sset < G::NSUB; sset += TB) {
      rvec4<double> P;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) P.c[mu] = 0.0;
      for (int g = 0; g < N; ++g) {
        if (!((sset >> g) & 1)) continue;
        const int leg = g < 2 ? g : g + 2;
        const double sg = g < 2 ? 1.0 : -1.0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) P.c[mu] += sg * a.mom[(long)(leg * 4 + mu) * a.ld + e];
      }
      pset[sset] = P;
    }
    for (int it = tid; it < 2 * N + 4; it += TB) {
      double p[4];
      if (it < 2 * N) {
        const int g = it >> 1, leg = g < 2 ? g : g + 2;
        load_leg<double>(a.mom, a.ld, e, leg, p);
        const vec4<double> ev = polvec<double>(p, (it & 1) ? 1 : -1, g >= 2);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) { eps_all[it * 8 + 2 * mu] = ev.c[mu].re; eps_all[it * 8 + 2 * mu + 1] = ev.c[mu].im; }
      } else {
        const int k = it - 2 * N;                          // 0, 1: ubar(p_t, -/+); 2, 3: v(p_tbar, -/+)
        load_leg<double>(a.mom, a.ld, e, k < 2 ? 2 : 3, p);
        const spinor<double> sp = k < 2 ? bar(spinor_u<double>(p, (k & 1) ? 1 : -1, false)) : spinor_v<double>(p, (k & 1) ? 1 : -1, false);
#pragma unroll
        for (int i = 0; i < 4; ++i) { spin[k * 8 + 2 * i] = sp.c[i].re; spin[k * 8 + 2 * i + 1] = sp.c[i].im; }
      }
    }
    __syncthreads();

    RC acc0 = RC(0), acc1 = RC(0);
    for (unsigned itb = 0; itb < (unsigned)G::NIT; ++itb) {
      // ---- phase 1: current table of this helicity iteration
      for (int e1 = tid; e1 < meta[I::M_LVL + 2]; e1 += TB) tab_build_level1<R, N, NFIX>(tab, meta, pset, eps_all, itb, e1);
      __syncthreads();
      build_levels<R, N, NFIX, 2>(tab, meta, pset);

      // ---- phase 2: top-line walk
      for (int task = tid; task < G::NTASK * NPASS; task += TB) {
        const int pass = task / G::NTASK, r = task - pass * G::NTASK;
        const int hl = r % G::NHL, prank = r / G::NHL;
        using Store = TabLeafStore<R, RC, XS>;
        Store st;
        TabWalk<R, N, NFIX, D, Store> w;
        prefix_of_rank<N, D>(prank, w.pref);
        const int lt = hl & 1;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) w.pt.c[mu] = a.mom[(long)(2 * 4 + mu) * a.ld + e];
#pragma unroll
        for (int i = 0; i < 4; ++i) w.ubar_t.c[i] = cx<R>(R(spin[lt * 8 + 2 * i]), R(spin[lt * 8 + 2 * i + 1]));
        w.tab = tab; w.off = meta + I::M_OFF; w.pset = pset;
        w.hfree = (unsigned)(hl >> 1);
        w.line.mt = a.T.mt[pass]; w.line.mGt = a.T.mGt[pass];
        st.xs = xs; st.vsp = spin + 16;
        st.colbase = hl * 4;
        st.leaf0 = prank * I::falling(N - D, N - D);
        st.th_lo = NPASS == 1 ? 0 : pass; st.th_hi = NPASS == 1 ? 2 : pass + 1;
        st.kq[0] = R(a.T.kq[0]); st.kq[1] = R(a.T.kq[1]);
        w.run(&st);
      }
      __syncthreads();

      // ---- phase 3: x^dagger C x of every X column; row blocks paired (p, NB-1-p) for balance
      constexpr int RB = F::RB, NB = F::NB, NPAIR = (NB + 1) / 2;
      for (int item = tid; item < G::NCOLT * NPAIR; item += TB) {
        const int c = item % G::NCOLT, p = item / G::NCOLT;
        RC accl = RC(0);
        for (int side = 0; side < 2; ++side) {
          const int b = side == 0 ? p : NB - 1 - p;
          if (side == 1 && b == p) break;
          cx<RC> t[RB];
#pragma unroll
          for (int r = 0; r < RB; ++r) t[r] = cx<RC>(RC(0), RC(0));
          const RC* row = Cs;
          const int iend = RB * b + RB;
#pragma unroll 2
          for (int i = 0; i < iend; ++i) {
            const cx<RC> xi = xs[i * XS + c];
            const RC* cr = row + (RB * b - RB * (i / RB));
#pragma unroll
            for (int r = 0; r < RB; ++r) cfma(t[r], xi, cr[r]);
            row += F::row_len(i);
          }
#pragma unroll
          for (int r = 0; r < RB; ++r) { const cx<RC> xj = xs[(RB * b + r) * XS + c]; accl += xj.re * t[r].re + xj.im * t[r].im; }
        }
        if (c & 1) acc1 += accl; else acc0 += accl;
      }
      // no barrier needed here: the next writes to X happen after the barriers of the next iteration's phase 1
    }

    // ---- fixed-order block reduction + epilogue
    double v0 = (double)acc0, v1 = (double)acc1;
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) { v0 += __shfl_xor_sync(0xFFFFFFFFu, v0, o); v1 += __shfl_xor_sync(0xFFFFFFFFu, v1, o); }
    if ((tid & 31) == 0) { red[(tid >> 5) * 2] = v0; red[(tid >> 5) * 2 + 1] = v1; }
    __syncthreads();
    if (tid == 0) {
      double s0 = 0.0, s1 = 0.0;
      for (int w = 0; w < TB / 32; ++w) { s0 += red[2 * w]; s1 += red[2 * w + 1]; }
      const double mo = s0 * a.T.pref[0], mn = s1 * a.T.pref[1];
      const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
      a.w_out[e] = a.w_in[e] * norm * mn;                        // evaluate + append_wgts
      if (a.me2_old) a.me2_old[e] = mo;
      if (a.me2_new) a.me2_new[e] = mn;
    }
  }
}

}  // namespace

// meta block and folded colour matrix sizes (host allocates and fills them once)
int TREX_TU_NAME(trex_tu_table_meta_n, TREX_TU_N, TREX_TU_MODE)(int* meta) {
  using I = TabIdx<TREX_TU_N, TabCfg<TREX_TU_N>::NFIX>;
  if (meta) I::build_meta(meta);
  return I::M_SIZE;
}
int TREX_TU_NAME(trex_tu_table_fold_n, TREX_TU_N, TREX_TU_MODE)(const double* C, double* f) {
  using F = FoldedC<TabIdx<TREX_TU_N, 0>::falling(TREX_TU_N, TREX_TU_N)>;
  constexpr int NC = TabIdx<TREX_TU_N, 0>::falling(TREX_TU_N, TREX_TU_N);
  if (f) {
    int k = 0;
    for (int i = 0; i < NC; ++i)
      for (int j = F::RB * (i / F::RB); j < NC; ++j) f[k++] = j < i ? 0.0 : (j == i ? C[i * NC + i] : 2.0 * C[i * NC + j]);
  }
  return F::size();
}

int TREX_TU_NAME(trex_tu_table_launch_n, TREX_TU_N, TREX_TU_MODE)(const ReweightArgs& a, int npass, const int* meta, const double* Cfold,
                                                                  int nsm, cudaStream_t s) {
  constexpr int N = TREX_TU_N;
  using G = TabGeom<TuR, TuRC, N>;
  static int blocks_per_sm = 0;
  if (!blocks_per_sm) {
    cudaFuncSetAttribute(k_table<TuR, TuRC, N, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::bytes);
    cudaFuncSetAttribute(k_table<TuR, TuRC, N, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)G::bytes);
    int b1 = 0, b2 = 0;
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b1, k_table<TuR, TuRC, N, 1>, G::TB, G::bytes);
    cudaOccupancyMaxActiveBlocksPerMultiprocessor(&b2, k_table<TuR, TuRC, N, 2>, G::TB, G::bytes);
    blocks_per_sm = b1 < b2 ? b1 : b2;
    if (blocks_per_sm < 1) return (int)cudaErrorLaunchOutOfResources;
  }
  const long want = (long)nsm * blocks_per_sm;
  const unsigned grid = (unsigned)(a.n < want ? a.n : want);
  if (npass == 1) k_table<TuR, TuRC, N, 1><<<grid, G::TB, G::bytes, s>>>(a, meta, Cfold);
  else k_table<TuR, TuRC, N, 2><<<grid, G::TB, G::bytes, s>>>(a, meta, Cfold);
  return (int)cudaGetLastError();
}

}  // namespace trex
