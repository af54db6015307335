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

#ifndef TREX_T3_TB
#define TREX_T3_TB 128
#endif
#ifndef TREX_T3_EPB
#define TREX_T3_EPB 4
#endif
#ifndef TREX_T3_MINB
#define TREX_T3_MINB 3
#endif
#ifndef TREX_T3_UT
#define TREX_T3_UT 1
#endif
#ifndef TREX_T5_UT
#define TREX_T5_UT 1
#endif
#ifndef TREX_T5_DMMA
#define TREX_T5_DMMA 1
#endif
#ifndef TREX_T4_TB
#define TREX_T4_TB 384
#endif
#ifndef TREX_T4_MINB
#define TREX_T4_MINB 1
#endif
#ifndef TREX_T4_UT
#define TREX_T4_UT 2
#endif
#ifndef TREX_T4_LTSPLIT
#define TREX_T4_LTSPLIT 0
#endif
#ifndef TREX_T4_WFORM
#define TREX_T4_WFORM 1
#endif
#ifndef TREX_TF32_COLOUR
#define TREX_TF32_COLOUR 1
#endif
#ifndef TREX_T4_DMMA
#define TREX_T4_DMMA 1
#endif
// NFIX: gluons whose helicity the outer loop fixes; D: depth of the ordering prefix that defines a walk task;
// TB: threads per block; EPB: events a block works on at the same time, each by its own group of TB / EPB threads
// (a group of 32 = one warp synchronises with __syncwarp and runs free of the other warps); MINB: blocks per SM;
// UT: the top-line states of ordering prefixes up to this length are tabulated per event instead of being carried by
// every walk thread (fewer registers per thread -> more warps, and no recomputation across tasks)
template <int N> struct TabCfg;
// (N = 4 runs the W-form event pipeline of trex_table4.cuh unless TREX_T4_WFORM = 0 selects the kernel of this file)
// LTSPLIT: walk + colour sum run once per top helicity, the X tile holds the columns of one lambda_t only (half the tile:
// room for a second resident block per SM)
template <> struct TabCfg<3> { static constexpr int NFIX = 0, D = TREX_T3_UT == 2 ? 3 : 2, TB = TREX_T3_TB, EPB = TREX_T3_EPB, MINB = TREX_T3_MINB, UT = TREX_T3_UT, LTSPLIT = 0; };
template <> struct TabCfg<4> { static constexpr int NFIX = 0, D = TREX_T4_UT ? 4 : 2, TB = TREX_T4_TB, EPB = 1, MINB = TREX_T4_MINB, UT = TREX_T4_UT, LTSPLIT = TREX_T4_LTSPLIT; };
template <> struct TabCfg<5> { static constexpr int NFIX = 3, D = 3, TB = 256, EPB = 1, MINB = 1, UT = TREX_T5_UT, LTSPLIT = 0; };

template <int NC> struct FoldedC {
  // C'(i,j) = 0 (j < i), C_ii (j == i), 2 C_ij (j > i), stored by rows i for j >= RB floor(i/RB)
  static constexpr int RB = NC % 8 == 0 ? 8 : NC;            // rows per register block (NC = 6: one block)
  static constexpr int NB = NC / RB;
  static constexpr int NPAIR = (NB + 1) / 2;                 // row blocks are paired (p, NB-1-p) for balance
  __host__ __device__ static constexpr int row_len(int i) { return NC - RB * (i / RB); }
  __host__ __device__ static constexpr int size() { int s = 0; for (int i = 0; i < NC; ++i) s += row_len(i); return s; }
};

template <class R, class RC, int N> struct TabGeom {
  using Cfg = TabCfg<N>;
  using I = TabIdx<N, Cfg::NFIX>;
  static constexpr int NFIX = Cfg::NFIX, D = Cfg::D, TB = Cfg::TB, EPB = Cfg::EPB, GS = TB / EPB, UT = Cfg::UT;
  using UI = UTabIdx<N, Cfg::NFIX>;
  static constexpr int NU = UI::N1 + (UT == 2 ? UI::N2 : 0), NUT = 2 * NU;   // line-state table entries per parameter point / in all
  static_assert(GS * EPB == TB && (GS == TB || GS == 32), "an event group is one warp or the whole block");
  static constexpr int NE = I::NE;
  static constexpr int NC = I::falling(N, N);
  static constexpr int NIT = 1 << NFIX;
  static constexpr int NLT = Cfg::LTSPLIT ? 2 : 1;           // walk + colour passes per helicity iteration (one per lambda_t)
  static constexpr int NHL = (2 << I::NFREE) / NLT;          // (free helicities [, lambda_t]) of one pass
  static constexpr int NPREF = I::falling(N, D);
  static constexpr int NTASK = NPREF * NHL;
  static constexpr int NCOLT = NHL * 4;                      // X tile columns: (hfree [, lt], ltb, theta)
  // row stride of the X tile in complex numbers: odd for the vector colour sum; = 4 mod 8 for the tensor-core one, so
  // that the four k rows of an mma fragment (stride 2 XS doubles = 8 mod 16) land in disjoint banks
  static constexpr bool DMMA_CFG = sizeof(RC) == 8 && EPB == 1 && ((TREX_T5_DMMA && NC == 120) || (TREX_T4_DMMA && NC == 24));
  // fp32 colour arithmetic (mixed / fp32 modes) on the tensor cores: mma.sync.m16n8k8 with TF32 operands.
  // The folded colour matrix times 54 (ncol = 24) / 324 (ncol = 120) consists of integers with at most 11 significant
  // bits: exact in TF32; X is split into two TF32 numbers (hi + lo), so the products keep fp32 accuracy.
  // Measured (profiles/r02_kernels.md): wins for ncol = 120 (+2.4 % mixed, +5.8 % fp32 on the kernel), loses for ncol = 24
  // (-9 %: the FMA form there is a fraction of one pipelined phase) -> ncol = 120 only.
  static constexpr bool TF32 = TREX_TF32_COLOUR && sizeof(RC) == 4 && EPB == 1 && NC == 120;
  static constexpr int TF32_DEN = NC == 24 ? 54 : 324;
  static constexpr int NMT = (NC + 15) / 16, NKB = NC / 8;   // 16-row tiles of T = C'^T X, 8-flow k blocks
  __host__ __device__ static constexpr int tf32_kb(int J) { return 2 * J + 2 < NKB ? 2 * J + 2 : NKB; }   // k blocks with i <= 16 J + 15
  __host__ __device__ static constexpr int tf32_frag0(int J) { int f = 0; for (int j = 0; j < J; ++j) f += tf32_kb(j); return f; }
  static constexpr int CN = TF32 ? tf32_frag0(NMT) * 128 : FoldedC<NC>::size();       // numbers in the colour-matrix block
  static constexpr int XS = (DMMA_CFG || TF32) ? NCOLT + 4 : NCOLT + 1;
  static constexpr int NSUB = 1 << N;
  // colour sum on the FP64 tensor cores: fp64 colour arithmetic, ncol = 120 (and 24), one partial-sum slot per thread
  static constexpr bool DMMA = DMMA_CFG;
  static constexpr int NCI0 = NCOLT * FoldedC<NC>::NPAIR;    // colour-sum work items of the FMA form
  static constexpr int NCI = ((DMMA || TF32) && NCI0 < TB) ? TB : NCI0;  // partial-sum slots per event
  // shared-memory carve-up (bytes, every region 16-byte aligned): EPB event slots, then the block-wide constants
  static constexpr size_t al(size_t x) { return (x + 15) / 16 * 16; }
  static constexpr size_t o_tab = 0;
  static constexpr size_t o_x = o_tab + al(sizeof(R) * TAB_NCOMP * NE);
  static constexpr size_t o_pset = o_x + al(sizeof(cx<RC>) * NC * XS);
  static constexpr size_t o_eps = o_pset + al(sizeof(rvec4<double>) * NSUB);
  static constexpr size_t o_spin = o_eps + al(sizeof(double) * 16 * N);
  static constexpr size_t o_part = o_spin + al(sizeof(double) * 8 * 4);
  static constexpr size_t o_utab = o_part + al(sizeof(double) * NCI);
  static constexpr size_t o_pm = o_utab + (UT ? al(sizeof(R) * 16 * NUT) : 0);
  static constexpr int NROW = 4 * (N + 2);                   // momentum rows of one event
  static constexpr size_t slot = o_pm + al(sizeof(double) * NROW);
  static constexpr size_t o_c = slot * EPB;
  static constexpr size_t o_meta = o_c + al(sizeof(RC) * CN);
  static constexpr size_t bytes = o_meta + al(sizeof(int) * I::M_SIZE);
  static_assert(bytes <= 232448, "one SM has 227 KB of shared memory");
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

template <int GS> __device__ __forceinline__ void group_sync() {
  if constexpr (GS == 32) __syncwarp(); else __syncthreads();
}

struct NoSink {
  template <class S> __device__ __forceinline__ void operator()(int, const S&, const S&) {}
};

// line state of one ordering prefix of length L (item = UTabIdx level-L index, pass) -> utab
template <class R, class RC, int N, int L>
__device__ __forceinline__ void build_ustate(unsigned char* sb, const int* meta, const ReweightArgs& a, const rvec4<double>& pt, int item, int pass) {
  using G = TabGeom<R, RC, N>;
  using I = typename G::I;
  TabWalk<R, N, G::NFIX, L, NoSink, L - 1, L> w;
  NoSink none;
  const int lt = item & 1;
  unsigned bits;
  if constexpr (L == 1) {
    G::UI::level1_decode(item >> 1, w.pref[0], bits);
    w.hfree = w.pref[0] >= G::NFIX ? bits << (w.pref[0] - G::NFIX) : 0u;
  }
  else {
    bits = (item >> 1) & 3u;
    const int pr = item >> 3, g1 = pr / (N - 1), r = pr - g1 * (N - 1), g2 = r + (r >= g1 ? 1 : 0);
    w.pref[0] = g1; w.pref[1] = g2;
    w.hfree = ((bits & 1u) << g1) | (((bits >> 1) & 1u) << g2);
  }
  const double* spin = reinterpret_cast<const double*>(sb + G::o_spin);
#pragma unroll
  for (int i = 0; i < 4; ++i) w.ubar_t.c[i] = cx<R>(R(spin[lt * 8 + 2 * i]), R(spin[lt * 8 + 2 * i + 1]));
  w.pt = pt;
  w.tab = reinterpret_cast<const R*>(sb + G::o_tab); w.off = meta + I::M_OFF;
  w.pset = reinterpret_cast<const rvec4<double>*>(sb + G::o_pset);
  w.utab = reinterpret_cast<R*>(sb + G::o_utab); w.nut = G::NUT; w.ubase = pass * G::NU; w.lt = lt;
  w.line.mt = a.T.mt[pass]; w.line.mGt = a.T.mGt[pass];
  w.run(&none);
}

template <class R, class RC, int N, int NPASS, int K>
__device__ __forceinline__ void build_levels(unsigned char* sb, const int* meta, int gtid, const ReweightArgs& a, const rvec4<double>& pt) {
  using G = TabGeom<R, RC, N>;
  using I = typename G::I;
  if constexpr (K <= N) {
    const int e0 = meta[I::M_LVL + K], ntab = meta[I::M_LVL + K + 1] - e0;
    // the line states of the prefixes of length K - 1 need the table levels < K and the states of length K - 2: same phase
    constexpr int L = K - 1;
    constexpr int nus = L <= G::UT ? (L == 1 ? G::UI::N1 : G::UI::N2) : 0;
    for (int it = gtid; it < ntab + nus * NPASS; it += G::GS) {
      if (it < ntab) {
        tab_build_entry<R, N, G::NFIX, K>(reinterpret_cast<R*>(sb + G::o_tab), meta, reinterpret_cast<const rvec4<double>*>(sb + G::o_pset), e0 + it);
      } else if constexpr (nus > 0) {
        const int u = it - ntab, pass = u / nus;
        build_ustate<R, RC, N, L>(sb, meta, a, pt, u - pass * nus, pass);
      }
    }
    group_sync<G::GS>();
    build_levels<R, RC, N, NPASS, K + 1>(sb, meta, gtid, a, pt);
  }
}

// ---- phase 3 of k_table: x^dagger C x of every X column added into the event's partial-sum slots
template <class R, class RC, int N>
// ncw > 0 (tensor-core form only): the first ncw warps of the group share the column blocks, the others do not take part
__device__ __forceinline__ void colour_phase(const cx<RC>* __restrict__ xs, const RC* __restrict__ Cs, double* __restrict__ part, int tid, int gtid, int ncw = 0,
                                             bool half_lt = false) {
  using G = TabGeom<R, RC, N>;
  using F = FoldedC<G::NC>;
  constexpr int XS = G::XS, GS = G::GS;
  // ---- phase 3: x^dagger C x of every X column, 8-row register blocks, row blocks paired (p, NB-1-p) for balance.
  // A work item is always handled by the same thread, so its partial sum accumulates race-free in shared memory.
  constexpr int RB = F::RB, NB = F::NB;
  if constexpr (G::DMMA) {
    // FP64 tensor cores (mma.sync m8n8k4, measured 37 TFLOP/s against 24.7 for register-operand DFMA): the tile is a
    // real [NC x 2 NCOLT] matrix X (re/im interleaved); T = C'^T X is formed in 8 x 8 tiles (row block J of 8 flows,
    // column block of 4 complex columns), k runs over the flows i < 8 J + 8 in steps of 4; the accumulator layout
    // (lane: row lane/4, columns 2 (lane%4), +1) puts (Re, Im) of t_j for one complex column into one lane, which
    // closes it with x_j. A warp owns one column block and walks the row-block pairs (p, NB-1-p).
    const int lane = tid & 31, wrp = tid >> 5;
    const int fr = lane >> 2, fc = lane & 3;
    const double* xr = reinterpret_cast<const double*>(xs);
    constexpr int XR = 2 * XS, NCB = G::NCOLT / 4;
    double accl = 0.0;
    // a warp owns one column block; row blocks go four at a time (J0 .. J0+3) so that one X fragment feeds four
    // independent accumulator chains
    const int cstep = ncw > 0 ? ncw : GS / 32;
    if (wrp >= cstep) return;
    // half_lt: the column blocks of lambda_t = + (odd ones) are not in use (helicity symmetry)
    for (int kb = wrp; kb < (half_lt ? NCB / 2 : NCB); kb += cstep) {
      const int cb = half_lt ? 2 * kb : kb;
      for (int J0 = 0; J0 < NB; J0 += 4) {
        double d[4][2];
#pragma unroll
        for (int q = 0; q < 4; ++q) { d[q][0] = 0.0; d[q][1] = 0.0; }
        const int Jm = min(J0 + 3, NB - 1);
        for (int ks = 0; ks < 2 * (Jm + 1); ++ks) {
          const int i = 4 * ks + fc, bi = i >> 3;
          const double bv = xr[i * XR + 8 * cb + fr];
#pragma unroll
          for (int q = 0; q < 4; ++q) {
            const int J = J0 + q;
            if (J < NB && bi <= J) {
              // C' is stored in fragment order: fragment (J, ks) = the 8 x 4 block C'(4 ks + fc, 8 J + fr), lane-major
              const double av = Cs[(J * (J + 1) + ks) * 32 + lane];
              asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};"
                           : "+d"(d[q][0]), "+d"(d[q][1]) : "d"(av), "d"(bv));
            }
          }
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
          const int J = J0 + q;
          if (J < NB) { const cx<RC> xj = xs[(8 * J + fr) * XS + 4 * cb + fc]; accl += xj.re * d[q][0] + xj.im * d[q][1]; }
        }
      }
    }
    part[tid] += accl;                                  // slot parity = lane parity = column parity = theta
  } else if constexpr (G::TF32) {
    // TF32 tensor cores (mma.sync m16n8k8, fp32 accumulators): T = C'^T X in 16 x 8 tiles (16 flows j, 4 complex columns),
    // k over the flows i <= 16 J + 15 in blocks of 8; A = the integer colour matrix (exact in TF32), B = X as hi + lo.
    // Accumulator layout: rows g = lane / 4 and g + 8, columns 2 (lane % 4), + 1 = (Re, Im) of t_j for one complex column.
    const int lane = tid & 31, wrp = tid >> 5;
    const int g = lane >> 2, t = lane & 3;
    const float* xr = reinterpret_cast<const float*>(xs);
    constexpr int XR = 2 * XS, NCB = G::NCOLT / 4;
    const int cstep = ncw > 0 ? ncw : GS / 32;
    if (wrp >= cstep) return;
    float accl = 0.f;
    const auto tf32 = [](float x) { unsigned r; asm("cvt.rna.tf32.f32 %0, %1;" : "=r"(r) : "f"(x)); return r; };
    for (int cb = wrp; cb < NCB; cb += cstep) {
#pragma unroll 1
      for (int J = 0; J < G::NMT; ++J) {
        float d0 = 0.f, d1 = 0.f, d2 = 0.f, d3 = 0.f;
        const int nkb = G::tf32_kb(J);
        const float4* af = reinterpret_cast<const float4*>(Cs) + (size_t)G::tf32_frag0(J) * 32 + lane;
        for (int kb = 0; kb < nkb; ++kb) {
          const float4 av = af[kb * 32];
          const unsigned a0 = __float_as_uint(av.x), a1 = __float_as_uint(av.y), a2 = __float_as_uint(av.z), a3 = __float_as_uint(av.w);
          const float x0 = xr[(8 * kb + t) * XR + 8 * cb + g], x1 = xr[(8 * kb + t + 4) * XR + 8 * cb + g];
          const unsigned h0 = tf32(x0), h1 = tf32(x1);
          const unsigned l0 = tf32(x0 - __uint_as_float(h0)), l1 = tf32(x1 - __uint_as_float(h1));
          asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                       : "+f"(d0), "+f"(d1), "+f"(d2), "+f"(d3) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(h0), "r"(h1));
          asm volatile("mma.sync.aligned.m16n8k8.row.col.f32.tf32.tf32.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
                       : "+f"(d0), "+f"(d1), "+f"(d2), "+f"(d3) : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(l0), "r"(l1));
        }
        const int j0 = 16 * J + g;
        if (j0 < G::NC) { const cx<RC> xj = xs[j0 * XS + 4 * cb + t]; accl += xj.re * d0 + xj.im * d1; }
        if (j0 + 8 < G::NC) { const cx<RC> xj = xs[(j0 + 8) * XS + 4 * cb + t]; accl += xj.re * d2 + xj.im * d3; }
      }
    }
    part[tid] += (double)accl * (1.0 / G::TF32_DEN);        // slot parity = lane parity = column parity = theta
  } else
  // half_lt (FMA form only): the columns of lambda_t = + [bit 2 of the column index] are not in use (helicity symmetry)
  for (int item = gtid; item < (half_lt ? G::NCI0 / 2 : G::NCI0); item += GS) {
    const int ncolt = half_lt ? G::NCOLT / 2 : G::NCOLT;
    const int cc = item % ncolt, p = item / ncolt;
    const int c = half_lt ? (((cc >> 2) << 3) | (cc & 3)) : cc;
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
    part[item] += (double)accl;
  }
}

template <class R, class RC, int N, int NPASS>
__global__ void __launch_bounds__(TabCfg<N>::TB, TabCfg<N>::MINB) k_table(const ReweightArgs a, const int* __restrict__ gmeta, const double* __restrict__ Cfold) {
  using G = TabGeom<R, RC, N>;
  using I = typename G::I;
  using F = FoldedC<G::NC>;
  constexpr int NFIX = G::NFIX, D = G::D, TB = G::TB, XS = G::XS, EPB = G::EPB, GS = G::GS, UT = G::UT;
  extern __shared__ __align__(16) unsigned char smem[];
  RC* Cs = reinterpret_cast<RC*>(smem + G::o_c);
  int* meta = reinterpret_cast<int*>(smem + G::o_meta);
  const int tid = threadIdx.x, sl = tid / GS, gtid = tid - sl * GS;
  unsigned char* sb = smem + sl * G::slot;                    // this group's event slot
  R* tab = reinterpret_cast<R*>(sb + G::o_tab);
  cx<RC>* xs = reinterpret_cast<cx<RC>*>(sb + G::o_x);
  rvec4<double>* pset = reinterpret_cast<rvec4<double>*>(sb + G::o_pset);
  double* eps_all = reinterpret_cast<double*>(sb + G::o_eps);
  double* spin = reinterpret_cast<double*>(sb + G::o_spin);
  double* part = reinterpret_cast<double*>(sb + G::o_part);
  double* pm = reinterpret_cast<double*>(sb + G::o_pm);

  const EvIO io = resolve_io(a);
  for (int i = tid; i < I::M_SIZE; i += TB) meta[i] = gmeta[i];
  for (int i = tid; i < G::CN; i += TB) Cs[i] = RC(Cfold[i]);
  for (int i = gtid; i < G::NCI; i += GS) part[i] = 0.0;
  // helicity symmetry (a.hsym, R-21) without a helicity loop to halve (N = 3): the walk tasks with lambda_t = -
  // stand for their parity partners; the X columns of lambda_t = + are neither written nor read
  constexpr bool HS_LT = G::NIT == 1 && G::NLT == 1 && !G::DMMA && !G::TF32;
  const bool hs_lt = HS_LT && a.hsym && !a.dbg;
  __syncthreads();

#ifdef TREX_PHASE_CLOCKS
  long long pc[5] = {0, 0, 0, 0, 0}, t0;
#define PHASE_TICK(k) do { if (tid == 0) { const long long t1 = clock64(); pc[k] += t1 - t0; t0 = t1; } } while (0)
#else
#define PHASE_TICK(k) do { } while (0)
#endif
  // the momenta of the group's NEXT event are loaded (one row per thread) while the current one is worked on: the DRAM
  // latency of the only global read of the kernel is paid once per block, not once per event
  const long e_first = (long)blockIdx.x * EPB + sl, e_step = (long)gridDim.x * EPB;
  double nxt = (gtid < G::NROW && e_first < io.n) ? io.mom[(long)gtid * io.ld + e_first] : 0.0;
  for (long e = e_first; e < io.n; e += e_step) {
#ifdef TREX_PHASE_CLOCKS
    if (tid == 0) t0 = clock64();
#endif
    if (gtid < G::NROW) pm[gtid] = nxt;
    group_sync<GS>();
    if (gtid < G::NROW && e + e_step < io.n) nxt = io.mom[(long)gtid * io.ld + e + e_step];
    // ---- per-event set-up: momentum of every gluon subset (incoming convention), polarisation vectors, t / t~ spinors
    // (subset momenta and wavefunctions are independent: different lanes, one pass, one latency)
    for (int item = gtid; item < G::NSUB + 2 * N + 4; item += GS) {
     if (item < G::NSUB) {
      const int sset = item;
      rvec4<double> P;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) P.c[mu] = 0.0;
      for (int g = 0; g < N; ++g) {
        if (!((sset >> g) & 1)) continue;
        const int leg = g < 2 ? g : g + 2;
        const double sg = g < 2 ? 1.0 : -1.0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) P.c[mu] += sg * pm[leg * 4 + mu];
      }
      pset[sset] = P;
     } else {
      const int it = item - G::NSUB;
      double p[4];
      if (it < 2 * N) {
        const int g = it >> 1, leg = g < 2 ? g : g + 2;
        for (int mu = 0; mu < 4; ++mu) p[mu] = pm[leg * 4 + mu];
        const vec4<double> ev = polvec<double>(p, (it & 1) ? 1 : -1, g >= 2);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) { eps_all[it * 8 + 2 * mu] = ev.c[mu].re; eps_all[it * 8 + 2 * mu + 1] = ev.c[mu].im; }
      } else {
        const int k = it - 2 * N;                          // 0, 1: ubar(p_t, -/+); 2, 3: v(p_tbar, -/+)
        for (int mu = 0; mu < 4; ++mu) p[mu] = pm[(k < 2 ? 2 : 3) * 4 + mu];
        const spinor<double> sp = k < 2 ? bar(spinor_u<double>(p, (k & 1) ? 1 : -1, false)) : spinor_v<double>(p, (k & 1) ? 1 : -1, false);
#pragma unroll
        for (int i = 0; i < 4; ++i) { spin[k * 8 + 2 * i] = sp.c[i].re; spin[k * 8 + 2 * i + 1] = sp.c[i].im; }
      }
     }
    }
    group_sync<GS>();
    PHASE_TICK(0);

    rvec4<double> ptop;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) ptop.c[mu] = pm[2 * 4 + mu];
    // helicity symmetry (a.hsym): the iterations with the last fixed gluon at helicity - stand for their parity partners
    const unsigned nit = (a.hsym && G::NIT >= 2 && !(a.dbg)) ? (unsigned)G::NIT / 2 : (unsigned)G::NIT;
    const double hscale = (nit < (unsigned)G::NIT || hs_lt) ? 2.0 : 1.0;
    for (unsigned itb = 0; itb < nit; ++itb) {
      // ---- phase 1: current table of this helicity iteration (+ line states of short prefixes, if tabulated)
      for (int e1 = gtid; e1 < meta[I::M_LVL + 2]; e1 += GS) tab_build_level1<R, N, NFIX>(tab, meta, pset, eps_all, itb, e1);
      group_sync<GS>();
      build_levels<R, RC, N, NPASS, 2>(sb, meta, gtid, a, ptop);
      PHASE_TICK(1);

      for (int lti = 0; lti < G::NLT; ++lti) {
      // ---- phase 2: top-line walk
      const int nhl = hs_lt ? G::NHL / 2 : G::NHL, ntask = G::NPREF * nhl;
      for (int task = gtid; task < ntask * NPASS; task += GS) {
        const int pass = task / ntask, r = task - pass * ntask;
        const int hli = hs_lt ? 2 * (r % nhl) : r % nhl, prank = r / nhl;
        const int hl = G::NLT == 2 ? hli * 2 + lti : hli;
        using Store = TabLeafStore<R, RC, XS>;
        Store st;
        TabWalk<R, N, NFIX, D, Store, UT> w;
        prefix_of_rank<N, D>(prank, w.pref);
        const int lt = hl & 1;
        w.pt = ptop;
        w.utab = reinterpret_cast<R*>(sb + G::o_utab); w.nut = G::NUT; w.ubase = pass * G::NU; w.lt = lt;
#pragma unroll
        for (int i = 0; i < 4; ++i) w.ubar_t.c[i] = cx<R>(R(spin[lt * 8 + 2 * i]), R(spin[lt * 8 + 2 * i + 1]));
        w.tab = tab; w.off = meta + I::M_OFF; w.pset = pset;
        w.hfree = (unsigned)(hl >> 1);
        w.line.mt = a.T.mt[pass]; w.line.mGt = a.T.mGt[pass];
        st.xs = xs; st.vsp = spin + 16;
        st.colbase = hli * 4;
        st.leaf0 = prank * I::falling(N - D, N - D);
        st.th_lo = NPASS == 1 ? 0 : pass; st.th_hi = NPASS == 1 ? 2 : pass + 1;
        st.kq[0] = R(a.T.kq[0]); st.kq[1] = R(a.T.kq[1]);
        w.run(&st);
      }
      group_sync<GS>();
      PHASE_TICK(2);
      if (a.dbg && e == 0)                                  // diagnostics only (trex_debug_xtile)
        for (int i = gtid; i < G::NC * G::NCOLT; i += GS) {
          const int row = i / G::NCOLT, col = i - row * G::NCOLT;
          const cx<RC> x = xs[row * XS + col];
          double* d = a.dbg + 2 * ((((long)itb * G::NLT + lti) * G::NC + row) * G::NCOLT + col);
          d[0] = (double)x.re; d[1] = (double)x.im;
        }

      colour_phase<R, RC, N>(xs, Cs, part, tid, gtid, 0, hs_lt);
#ifdef TREX_PHASE_CLOCKS
      group_sync<GS>();
      PHASE_TICK(3);
#else
      if (lti + 1 < G::NLT) group_sync<GS>();                // the next walk pass overwrites X
#endif
      }
      // no barrier needed here: the next writes to X happen after the barriers of the next iteration's phase 1
    }
    group_sync<GS>();

    // ---- fixed-order reduction of the partial sums (column parity = theta) + epilogue by the group's first warp, which
    // clears what it has read; the other warps of the group may already set up the next event
    if (gtid < 32) {
      double v = 0.0;
      for (int i = gtid; i < G::NCI; i += 32) { v += part[i]; part[i] = 0.0; }
#pragma unroll
      for (int o = 16; o >= 2; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
      const double s1 = __shfl_sync(0xFFFFFFFFu, v, 1);
      if (gtid == 0) {
        const double mo = v * (a.T.pref[0] * hscale), mn = s1 * (a.T.pref[1] * hscale);
        const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
        io.w_out[e] = io.w_in[e] * norm * mn;                        // evaluate + append_wgts
        if (io.me2_old) io.me2_old[e] = mo;
        if (io.me2_new) io.me2_new[e] = mn;
      }
    }
    PHASE_TICK(4);
  }
#ifdef TREX_PHASE_CLOCKS
  if (tid == 0 && blockIdx.x == 0) printf("k_table N=%d phases [cycles of block 0]: setup %lld  table %lld  walk %lld  colour %lld  epilogue %lld\n", N, pc[0], pc[1], pc[2], pc[3], pc[4]);
#endif
}

#if TREX_TU_N == 4
#include "trex_table4.cuh"
#endif

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
  const auto folded = [&](int i, int j) { return j < i ? 0.0 : (j == i ? C[i * NC + i] : 2.0 * C[i * NC + j]); };
  if (f) {
    int k = 0;
    using G = TabGeom<TuR, TuRC, TREX_TU_N>;
    if (G::TF32) {
      // mma.m16n8k8 A fragments (row-major 16 x 8, A[m = j][k = i] = C'(i, j) x TF32_DEN, integers): per (J, kb) 32 lanes x
      // (a0, a1, a2, a3) = rows g / g + 8, columns t / t + 4 with g = lane / 4, t = lane % 4; flows beyond ncol are zero
      const auto A = [&](int i, int j) { return (i < NC && j < NC) ? folded(i, j) * G::TF32_DEN : 0.0; };
      for (int J = 0; J < G::NMT; ++J)
        for (int kb = 0; kb < G::tf32_kb(J); ++kb)
          for (int lane = 0; lane < 32; ++lane) {
            const int g = lane >> 2, t = lane & 3;
            f[k++] = std::nearbyint(A(8 * kb + t, 16 * J + g));     f[k++] = std::nearbyint(A(8 * kb + t, 16 * J + g + 8));
            f[k++] = std::nearbyint(A(8 * kb + t + 4, 16 * J + g)); f[k++] = std::nearbyint(A(8 * kb + t + 4, 16 * J + g + 8));
          }
    } else if (TabGeom<TuR, TuRC, TREX_TU_N>::DMMA) {
      // tensor-core colour sum: mma A fragments in the order the kernel consumes them, (J, ks) -> 32 lanes
      // (lane = 4 fr + fc holds C'(4 ks + fc, 8 J + fr)); sum_J 2 (J + 1) fragments of 32 = F::size() numbers again
      for (int J = 0; J < F::NB; ++J)
        for (int ks = 0; ks < 2 * (J + 1); ++ks)
          for (int lane = 0; lane < 32; ++lane) f[k++] = folded(4 * ks + (lane & 3), 8 * J + (lane >> 2));
    } else {
      for (int i = 0; i < NC; ++i)
        for (int j = F::RB * (i / F::RB); j < NC; ++j) f[k++] = folded(i, j);
    }
  }
  return TabGeom<TuR, TuRC, TREX_TU_N>::CN;
}

// layout of the diagnostic X-tile dump: {NFIX, iterations, lambda_t passes per iteration, flows, columns per pass}
int TREX_TU_NAME(trex_tu_table_geom_n, TREX_TU_N, TREX_TU_MODE)(int* out) {
  using G = TabGeom<TuR, TuRC, TREX_TU_N>;
  out[0] = G::NFIX; out[1] = G::NIT; out[2] = G::NLT; out[3] = G::NC; out[4] = G::NCOLT;
  return 0;
}

int TREX_TU_NAME(trex_tu_table_launch_n, TREX_TU_N, TREX_TU_MODE)(const ReweightArgs& a, int npass, long nmax, const int* meta, const double* Cfold,
                                                                  int nsm, cudaStream_t s) {
  constexpr int N = TREX_TU_N;
  using G = TabGeom<TuR, TuRC, N>;
#if TREX_TU_N == 4 && TREX_T4_WFORM
  {
    // software-pipelined W-form kernel (trex_table4.cuh): one persistent 384-thread block per SM
    using W = W4<TuR, TuRC>;
    static bool ready = false;
    if (!ready) {
      if (cudaFuncSetAttribute(k_table4w<TuR, TuRC, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)W::bytes) != cudaSuccess ||
          cudaFuncSetAttribute(k_table4w<TuR, TuRC, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)W::bytes) != cudaSuccess)
        return (int)cudaGetLastError();
      ready = true;
    }
    const unsigned grid = (unsigned)(nmax < (long)nsm ? nmax : (long)nsm);
    if (npass == 1) k_table4w<TuR, TuRC, 1><<<grid, W::TB, W::bytes, s>>>(a, meta, Cfold);
    else k_table4w<TuR, TuRC, 2><<<grid, W::TB, W::bytes, s>>>(a, meta, Cfold);
    return (int)cudaGetLastError();
  }
#else
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
  const long want = (long)nsm * blocks_per_sm, have = (nmax + G::EPB - 1) / G::EPB;
  const unsigned grid = (unsigned)(have < want ? have : want);
  if (npass == 1) k_table<TuR, TuRC, N, 1><<<grid, G::TB, G::bytes, s>>>(a, meta, Cfold);
  else k_table<TuR, TuRC, N, 2><<<grid, G::TB, G::bytes, s>>>(a, meta, Cfold);
  return (int)cudaGetLastError();
#endif
}

}  // namespace trex
