// trex_ttng_tu.cu -- g g -> t t~ + (N-2) g reweighting kernels for ONE (N, precision mode); compiled once per pair with
// -DTREX_TU_N={2,3,4,5} -DTREX_TU_MODE={0 fp64, 1 mixed: amplitudes fp64 + colour sum fp32, 2 fp32} (PAPER.md:1209 fptype d/m/f).
#include "trex_kernels.cuh"

#ifndef TREX_GGTT_UNROLL
#define TREX_GGTT_UNROLL 2
#endif
#ifndef TREX_GGTT_NW
#define TREX_GGTT_NW 8
#endif
#ifndef TREX_GGTT_MINB
#define TREX_GGTT_MINB 2
#endif

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

#if TREX_TU_N == 2
// ---------------------------------------------------------------- g g -> t t~ : external wavefunctions shared by a block
// A block is 32 consecutive events x 8 warps. Phase A: warp w evaluates ONE of the eight external wavefunctions of the
// process (eps(g1,-/+), eps(g2,-/+), ubar(t,-/+), v(t~,-/+)) for the 32 events and parks it in shared
// memory -- the generic unit kernel re-derives five of them in each of its eight units. Phase B: warp = helicity unit
// (gluon helicities, lambda_t); the thread reads its wavefunctions back (lane = event: conflict-free), forms the
// two-gluon current and field-strength bracket once (J_21 = -J_12), walks the two orderings one after the other and
// closes the 2 x 2 colour sum. Same recursion and the same operation order per amplitude as TTNGS<R, 2, 1, .>
// (SURVEY.md C-4); parameter points with equal top mass and width only (otherwise the generic kernel runs).
// HS (helicity symmetry, R-21; Gamma_t = 0): only the four units with lambda_t = - are evaluated (and doubled):
// four warps per block, one unit each, and twice as many blocks per SM.
template <class R, class RC, bool HS = false>
__global__ void __launch_bounds__(32 * (HS ? 4 : TREX_GGTT_NW), HS ? 2 * TREX_GGTT_MINB : TREX_GGTT_MINB) k_gg_tt(const ReweightArgs a) {
  constexpr int NW = HS ? 4 : TREX_GGTT_NW;                   // warps per block: 8 (one unit each) or 4 (two units each; HS: one each)
  __shared__ double wf[8][8][32];
  __shared__ double red[2][NW][32];
  extern __shared__ __align__(16) double u1t_raw[];              // [8][16][32]: line state after ONE gluon, see phase A2
  double (*u1t)[16][32] = reinterpret_cast<double (*)[16][32]>(u1t_raw);
  const EvIO io = resolve_io(a);
  if ((long)blockIdx.x * 32 >= io.n) return;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long e = (long)blockIdx.x * 32 + lane;
  const long ev = e < io.n ? e : io.n - 1;
  // all 16 momentum rows of the block's 32 events: one coalesced pass, one DRAM latency; later reads come from here
  __shared__ double pm[16][32];
  for (int r = warp; r < 16; r += NW) pm[r][lane] = io.mom[(long)r * io.ld + ev];
  __syncthreads();
  for (int item = warp; item < 8; item += NW) {
    double p[4];
    const int leg = item >> 1, lam = (item & 1) ? 1 : -1;      // legs in process order: g g t t~
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) p[mu] = pm[leg * 4 + mu][lane];
    if (leg < 2) {
      const vec4<double> w = polvec<double>(p, lam, false);
#pragma unroll
      for (int i = 0; i < 4; ++i) { wf[item][2 * i][lane] = w.c[i].re; wf[item][2 * i + 1][lane] = w.c[i].im; }
    } else {
      const spinor<double> w = leg == 2 ? bar(spinor_u<double>(p, lam, false)) : spinor_v<double>(p, lam, false);
#pragma unroll
      for (int i = 0; i < 4; ++i) { wf[item][2 * i][lane] = w.c[i].re; wf[item][2 * i + 1][lane] = w.c[i].im; }
    }
  }
  __syncthreads();
  // ---- phase A2: U(a) = ubar Gamma(eps_a) S(p_t - K_a) depends on (gluon a, its helicity, lambda_t) only: 8 states per
  // event where the 8 units x 2 orderings would form 16; one per warp, parked in shared memory
  for (int item = warp; item < 8; item += NW) {
    const int ga = item >> 2, ha = (item >> 1) & 1, lt = item & 1;
    if (HS && lt) continue;                                    // only lambda_t = - is walked
    vec4<R> ea;
    spinor<R> ubar;
    rvec4<double> Ka, pt;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      ea.c[i] = cx<R>(R(wf[2 * ga + ha][2 * i][lane]), R(wf[2 * ga + ha][2 * i + 1][lane]));
      ubar.c[i] = cx<R>(R(wf[4 + lt][2 * i][lane]), R(wf[4 + lt][2 * i + 1][lane]));
      Ka.c[i] = pm[ga * 4 + i][lane]; pt.c[i] = pm[8 + i][lane];
    }
    spinor<R> c0, c1 = szero<R>();
    ften<R> F = fzero<R>();
    wedge_acc(F, cast<R>(Ka), ea);
    const spinor<R> t0 = row_slash(ubar, ea);
#pragma unroll
    for (int i = 0; i < 4; ++i) c0.c[i] = mul_i(t0.c[i]);
    row_sigma_acc(c1, ubar, F);
    const rvec4<double> qd = rsub(pt, Ka);
    const double q2 = rdot(qd, qd);
    const rvec4<R> q = cast<R>(qd);
    const cx<double> den(q2 - a.T.mt[0] * a.T.mt[0], a.T.mGt[0]);
    const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
    const spinor<R> s0 = row_slash(c0, q), s1 = row_slash(c1, q);
    const R mtr = R(a.T.mt[0]);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      cx<R> n0 = s0.c[i]; cfma(n0, c0.c[i], mtr);
      cx<R> n1 = s1.c[i]; cfma(n1, c1.c[i], mtr);
      const cx<R> o0 = n0 * pr, o1 = n1 * pr;
      u1t[item][2 * i][lane] = (double)o0.re; u1t[item][2 * i + 1][lane] = (double)o0.im;
      u1t[item][8 + 2 * i][lane] = (double)o1.re; u1t[item][9 + 2 * i][lane] = (double)o1.im;
    }
  }
  __syncthreads();
  RC acc[2] = {RC(0), RC(0)};
#pragma unroll 1
 for (int uu = warp; uu < (HS ? 4 : 8); uu += NW) {
  const int unit = HS ? 2 * uu : uu;
  const int gh = unit >> 1, lt = unit & 1;
  const int wsel[2] = {gh & 1, 2 + ((gh >> 1) & 1)};           // wavefunction slots of eps(g1), eps(g2) for this unit
  spinor<R> ubar;
  rvec4<double> pt;
#pragma unroll
  for (int i = 0; i < 4; ++i) ubar.c[i] = cx<R>(R(wf[4 + lt][2 * i][lane]), R(wf[4 + lt][2 * i + 1][lane]));
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) pt.c[mu] = pm[8 + mu][lane];
  // ---- tuple (1,2) attached to the line at once: i ubar Jslash_12 and ubar sigma.F_12; ordering (2,1) takes the opposite sign
  spinor<R> d0, d1 = szero<R>();
  {
    vec4<R> e1, e2;
    rvec4<double> K1, K2;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      e1.c[i] = cx<R>(R(wf[wsel[0]][2 * i][lane]), R(wf[wsel[0]][2 * i + 1][lane]));
      e2.c[i] = cx<R>(R(wf[wsel[1]][2 * i][lane]), R(wf[wsel[1]][2 * i + 1][lane]));
      K1.c[i] = pm[i][lane]; K2.c[i] = pm[4 + i][lane];
    }
    const rvec4<double> P12 = radd(K1, K2);
    vec4<R> acc = vzero<R>();
    v3_acc(acc, K1, e1, K2, e2);
    const R sc = R(-1.0 / rdot(P12, P12));
    vec4<R> J12;
#pragma unroll
    for (int i = 0; i < 4; ++i) J12.c[i] = acc.c[i] * sc;
    ften<R> F = fzero<R>();
    wedge_acc(F, cast<R>(P12), J12);
    wedge_acc(F, e1, e2);
    const spinor<R> t0 = row_slash(ubar, J12);
#pragma unroll
    for (int i = 0; i < 4; ++i) d0.c[i] = mul_i(t0.c[i]);
    row_sigma_acc(d1, ubar, F);
  }
  const R mt = R(a.T.mt[0]);
  const RC cd = RC(c_Ctab[0]), co = RC(2.0 * c_Ctab[1]);
  const R kq[2] = {R(a.T.kq[0]), R(a.T.kq[1])};
  cx<RC> xprev[2][2];                                         // [lambda_tbar][theta] of the previous ordering
#pragma unroll
  for (int k = 0; k < 4; ++k) xprev[k >> 1][k & 1] = cx<RC>(RC(0), RC(0));
  constexpr int kOrdUnroll = TREX_GGTT_UNROLL;
#pragma unroll kOrdUnroll
  for (int ord = 0; ord < 2; ++ord) {
    // operands of this ordering (g_a next to the top, then g_b) come from shared memory / L1, not from register arrays
    const int ga = ord, gb = 1 - ord;
    vec4<R> eb;
    rvec4<double> Kb;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      eb.c[i] = cx<R>(R(wf[wsel[gb]][2 * i][lane]), R(wf[wsel[gb]][2 * i + 1][lane]));
      Kb.c[i] = pm[gb * 4 + i][lane];
    }
    // U(a) from phase A2
    dspinor<R> U1;
    {
      const int it = (ga << 2) | (((gh >> ga) & 1) << 1) | lt;
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        U1.o0.c[i] = cx<R>(R(u1t[it][2 * i][lane]), R(u1t[it][2 * i + 1][lane]));
        U1.o1.c[i] = cx<R>(R(u1t[it][8 + 2 * i][lane]), R(u1t[it][9 + 2 * i][lane]));
      }
    }
    // bracket = +- (tuple term) + U(a) Gamma(eps_b)
    spinor<R> b0, b1;
#pragma unroll
    for (int i = 0; i < 4; ++i) { b0.c[i] = ord ? -d0.c[i] : d0.c[i]; b1.c[i] = ord ? -d1.c[i] : d1.c[i]; }
    {
      ften<R> F = fzero<R>();
      wedge_acc(F, cast<R>(Kb), eb);
      const spinor<R> t0 = row_slash(U1.o0, eb);
#pragma unroll
      for (int i = 0; i < 4; ++i) b0.c[i] += mul_i(t0.c[i]);
      const spinor<R> t1 = row_slash(U1.o1, eb);
#pragma unroll
      for (int i = 0; i < 4; ++i) b1.c[i] += mul_i(t1.c[i]);
      row_sigma_acc(b1, U1.o0, F);
    }
    // close with both antitop helicities; 2 x 2 colour sum: C_11 |x_1|^2 + C_22 |x_2|^2 + 2 C_12 Re(conj(x_2) x_1)
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) {
      spinor<R> v;
#pragma unroll
      for (int i = 0; i < 4; ++i) v.c[i] = cx<R>(R(wf[6 + iv][2 * i][lane]), R(wf[6 + iv][2 * i + 1][lane]));
      const cx<R> a0 = row_col(b0, v), a1 = row_col(b1, v);
#pragma unroll
      for (int th = 0; th < 2; ++th) {
        cx<R> x = a0; cfma(x, a1, kq[th]);
        const cx<RC> y(RC(x.re), RC(x.im));
        acc[th] += cd * norm2(y) + co * (y.re * xprev[iv][th].re + y.im * xprev[iv][th].im);
        xprev[iv][th] = y;
        if (a.dbg && e == 0) {                              // diagnostics only (trex_debug_xtile): [unit][ordering][ltb][theta]
          double* d = a.dbg + 2 * (((unit * 2 + ord) * 2 + iv) * 2 + th);
          d[0] = (double)y.re; d[1] = (double)y.im;
        }
      }
    }
  }
 }
  red[0][warp][lane] = (double)acc[0]; red[1][warp][lane] = (double)acc[1];
  __syncthreads();
  if (warp == 0 && e < io.n) {
    double s0 = 0.0, s1 = 0.0;
#pragma unroll
    for (int w = 0; w < NW; ++w) { s0 += red[0][w][lane]; s1 += red[1][w][lane]; }
    const double hs = HS ? 2.0 : 1.0;
    const double mo = s0 * (a.T.pref[0] * hs), mn = s1 * (a.T.pref[1] * hs);
    const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
    io.w_out[e] = io.w_in[e] * norm * mn;                        // evaluate + append_wgts
    if (io.me2_old) io.me2_old[e] = mo;
    if (io.me2_new) io.me2_new[e] = mn;
  }
}
#endif

int TREX_TU_NAME(trex_tu_launch_n, TREX_TU_N, TREX_TU_MODE)(const ReweightArgs& a, int npass, unsigned grid, cudaStream_t s) {
#if TREX_TU_N == 2
  if (npass == 1) {                                   // equal top mass and width at both parameter points
    constexpr int kU1Bytes = 8 * 16 * 32 * (int)sizeof(double);
    static bool configured = false;
    if (!configured) {
      cudaFuncSetAttribute(k_gg_tt<TuR, TuRC>, cudaFuncAttributeMaxDynamicSharedMemorySize, kU1Bytes);
      cudaFuncSetAttribute(k_gg_tt<TuR, TuRC, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, kU1Bytes);
      configured = true;
    }
    if (a.hsym && !a.dbg) k_gg_tt<TuR, TuRC, true><<<grid, 32 * 4, kU1Bytes, s>>>(a);
    else k_gg_tt<TuR, TuRC><<<grid, 32 * TREX_GGTT_NW, kU1Bytes, s>>>(a);
    return (int)cudaGetLastError();
  }
#endif
  if (npass == 1) k_ttng<TuR, TuRC, TREX_TU_N, 1><<<grid, TtngGeom<TREX_TU_N>::NW * 32, 0, s>>>(a);
  else k_ttng<TuR, TuRC, TREX_TU_N, 2><<<grid, TtngGeom<TREX_TU_N>::NW * 32, 0, s>>>(a);
  return (int)cudaGetLastError();
}

int TREX_TU_NAME(trex_tu_upload_n, TREX_TU_N, TREX_TU_MODE)(const double* C, int count) {
  if (count > 576) return 0;            // ncol = 120 is read from global memory
  return (int)cudaMemcpyToSymbol(c_Ctab, C, sizeof(double) * count);
}

}  // namespace trex
