// trex_qq2.cuh -- one light-quark line + t t~ + TWO gluons (q q~ -> t t~ g g, q g -> t t~ q g, g q~ -> t t~ q~ g;
// SURVEY.md NEXT-4; R-8b).
//
// Decomposition. Remove the light line from a diagram: what is left falls into pieces attached to the line at one vertex
// each, exactly one of which holds the top line. Call S_L the gluons (a, b) in the other pieces. The piece with the top
// line is a top-line amplitude whose sources are the gluons NOT in S_L plus ONE off-shell source c: the current the light
// line emits after absorbing S_L in a given colour order,
//     Q(L | R) = (R_L gamma^mu C_R) / P^2,   R_L = row spinor after the ordered tuple L, C_R = column spinor after R,
// (vertices i gamma, propagators i qslash / q^2, tuples with their merged three-gluon currents -- the same colour-ordered
// rules as on the top line, trex_ttng.cuh, with m = 0 and no dipole). Colour: (L T^c R)_light x (L_T T^c R_T)_top summed over
// c; the Fierz identity turns every term into two of the twelve flows
//     type I : (S1)_{t k} (S2)_{r tb}      +1/2 A      with S1 = L_T R, S2 = L R_T
//     type II: (S1)_{t tb} (S2)_{r k}      -1/6 A      with S1 = L_T R_T, S2 = L R
// (t, tb: colour of top / antitop; r, k: row / column end of the light line; S1, S2: ordered strings of T^a, T^b). The pair
// (S1, S2) is numbered 0 (ab, -), 1 (ba, -), 2 (a, b), 3 (b, a), 4 (-, ab), 5 (-, ba); type II adds 6. Terms:
//     S_L = {}     : six orderings of (a, b, Q) on the top line                      (three_source_path)
//     S_L = {x}    : Q(x|) and Q(|x), two orderings of (y, Q) each                    (two_source_line)
//     S_L = {a, b} : Q(ab|) Q(ba|) Q(a|b) Q(b|a) Q(|ab) Q(|ba), single source        (one bracket each)
// The 12 x 12 colour matrix comes from trex_colour.h (traces of the strings, exact rationals).
//
// Live state. The 12 x 2 x 2 complex flow amplitudes of a thread (96 numbers) are accumulated in SHARED memory (element i
// of thread t at s[i * stride + t]: conflict-free), and the eleven light-line currents are formed right where they are used
// instead of being kept (they cost a few hundred operations each, the top-line walks tens of thousands): what stays in
// registers is the external wavefunctions and the walk itself.
#pragma once
#include "trex_proc.cuh"

namespace trex {

constexpr int QQ2_NFLOW = 12;

// flow amplitudes of one (light-line, gluon, top) helicity choice, both antitop helicities: element
// ((flow * 2 + order in kappa) * 2 + v) * 2 + (re, im) of this thread at s[element * stride]
template <class R> struct Qq2Acc {
  R* s; int stride;
  static constexpr int NEL = QQ2_NFLOW * 8;
  TREX_HD R& at(int f, int o, int iv, int ri) const { return s[(((f * 2 + o) * 2 + iv) * 2 + ri) * stride]; }
  TREX_HD void clear() const {
#pragma unroll 8
    for (int i = 0; i < NEL; ++i) s[i * stride] = R(0);
  }
  // one term: +1/2 to its type-I flow, -1/6 to its type-II flow
  TREX_HD void add(int f1, int f2, const cx<R> A[2][2]) const {
#pragma unroll
    for (int o = 0; o < 2; ++o)
#pragma unroll
      for (int iv = 0; iv < 2; ++iv) {
        at(f1, o, iv, 0) += R(0.5) * A[o][iv].re; at(f1, o, iv, 1) += R(0.5) * A[o][iv].im;
        at(6 + f2, o, iv, 0) += R(-1.0 / 6.0) * A[o][iv].re; at(6 + f2, o, iv, 1) += R(-1.0 / 6.0) * A[o][iv].im;
      }
  }
  TREX_HD cx<R> get(int f, int o, int iv) const { return cx<R>(at(f, o, iv, 0), at(f, o, iv, 1)); }
};

template <class R> TREX_HD vec4<R> qq2_scaled(const vec4<R>& j, double s) {
  vec4<R> o; const R sr = R(s);
#pragma unroll
  for (int i = 0; i < 4; ++i) o.c[i] = j.c[i] * sr;
  return o;
}

// light line after ONE gluon (e, K) at its row end / column end:
//   R_x = w (i eslash)(i qslash)/q^2 = -w eslash qslash / q^2, q = -(Kr + K);   C_x = -qslash eslash x / q^2, q = Kc + K
template <class R>
TREX_HD spinor<R> qq2_row1(const spinor<R>& w, const rvec4<double>& Kr, const vec4<R>& e, const rvec4<double>& K) {
  rvec4<double> q;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) q.c[mu] = -(Kr.c[mu] + K.c[mu]);
  const R s = R(-1.0 / rdot(q, q));
  spinor<R> o = row_slash(row_slash(w, e), cast<R>(q));
#pragma unroll
  for (int i = 0; i < 4; ++i) o.c[i] = o.c[i] * s;
  return o;
}
template <class R>
TREX_HD spinor<R> qq2_col1(const spinor<R>& x, const rvec4<double>& Kc, const vec4<R>& e, const rvec4<double>& K) {
  const rvec4<double> q = radd(Kc, K);
  const R s = R(-1.0 / rdot(q, q));
  spinor<R> o = slash_col(cast<R>(q), slash_col(e, x));
#pragma unroll
  for (int i = 0; i < 4; ++i) o.c[i] = o.c[i] * s;
  return o;
}

// external wavefunctions and momenta of one (light-line combination, gluon helicities) choice
template <class R> struct Qq2Ext {
  spinor<R> w, x;                 // row / column spinor of the light line
  vec4<R> e[2];                   // gluon polarisations
  rvec4<double> Kr, Kc, K[2], pt; // incoming-convention momenta of the light-line ends and the gluons; top momentum
};

// single-source top-line amplitude of the current Q (momentum P into the line): A[order][v]
template <class R>
TREX_HD void qq2_single(const spinor<R>& ubar_t, const spinor<R> vtb[2], const vec4<R>& Q, const rvec4<R>& P, cx<R> A[2][2]) {
  const spinor<R> c0 = row_slash(ubar_t, Q);
  spinor<R> c1 = szero<R>();
  ften<R> F = fzero<R>();
  wedge_acc(F, P, Q);
  row_sigma_acc(c1, ubar_t, F);
#pragma unroll
  for (int iv = 0; iv < 2; ++iv) { A[0][iv] = mul_i(row_col(c0, vtb[iv])); A[1][iv] = row_col(c1, vtb[iv]); }
}

// the three groups of terms for one top helicity and one parameter point's top line. On the device they are separate
// functions (not inlined): each gets the whole register file for its walk, and the caller's state is saved once around
// the call instead of being spilled and reloaded piecemeal inside it.
#if defined(__CUDA_ARCH__) && !defined(TREX_QQ2_INLINE)
#define TREX_QQ2_FN __device__ __noinline__
#else
#define TREX_QQ2_FN TREX_HD
#endif

// Top line with THREE ordered sources (e[i], K[i]: current and momentum into the line), ONE ordering (0, 1, 2): the path
// (0), (0 1), (0 1 2) of the prefix walk of trex_ttng.cuh written out -- merged currents J02 = (0 1), J13 = (1 2),
// J03 = (0 1 2), line states U1, U2 -- and closed with both antitop spinors: A[order in kappa][v]. The caller loops over
// the six orderings (rolled), so that only one path is alive at a time.
template <class R>
TREX_HD void three_source_path(const spinor<R>& ubar, const rvec4<double>& pt, const vec4<R>& e0, const rvec4<double>& K0,
                               const vec4<R>& e1, const rvec4<double>& K1, const vec4<R>& e2, const rvec4<double>& K2, double mt_d,
                               double mGt, const spinor<R> v[2], cx<R> A[2][2]) {
  const R mt = R(mt_d);
  auto propagate = [&](const spinor<R>& b0, const spinor<R>& b1, const rvec4<double>& qd, dspinor<R>& U) {
    const double q2 = rdot(qd, qd);
    const rvec4<R> q = cast<R>(qd);
    const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), cx<double>(q2 - mt_d * mt_d, mGt)));
    const spinor<R> s0 = row_slash(b0, q), s1 = row_slash(b1, q);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      cx<R> n0 = s0.c[i]; cfma(n0, b0.c[i], mt);
      cx<R> n1 = s1.c[i]; cfma(n1, b1.c[i], mt);
      U.o0.c[i] = n0 * pr; U.o1.c[i] = n1 * pr;
    }
  };
  auto scale = [](const vec4<R>& a, double s) { vec4<R> o; const R sr = R(s);
#pragma unroll
    for (int i = 0; i < 4; ++i) o.c[i] = a.c[i] * sr;
    return o; };
  // term of a bracket: b0 += i U.o0 Jslash, b1 += i U.o1 Jslash + U.o0 sigma.F
  auto absorb = [](spinor<R>& b0, spinor<R>& b1, const dspinor<R>& U, const vec4<R>& J, const ften<R>& F) {
    const spinor<R> t0 = row_slash(U.o0, J), t1 = row_slash(U.o1, J);
#pragma unroll
    for (int i = 0; i < 4; ++i) { b0.c[i] += mul_i(t0.c[i]); b1.c[i] += mul_i(t1.c[i]); }
    row_sigma_acc(b1, U.o0, F);
  };
  auto absorb0 = [&](spinor<R>& b0, spinor<R>& b1, const vec4<R>& J, const ften<R>& F) {      // at the external spinor
    const spinor<R> t0 = row_slash(ubar, J);
#pragma unroll
    for (int i = 0; i < 4; ++i) b0.c[i] += mul_i(t0.c[i]);
    row_sigma_acc(b1, ubar, F);
  };
  // level 1
  dspinor<R> U1, U2;
  {
    spinor<R> b0 = szero<R>(), b1 = szero<R>();
    ften<R> F = fzero<R>();
    wedge_acc(F, cast<R>(K0), e0);
    absorb0(b0, b1, e0, F);
    propagate(b0, b1, rsub(pt, K0), U1);
  }
  // level 2
  const rvec4<double> P02 = radd(K0, K1);
  vec4<R> J02;
  {
    vec4<R> acc = vzero<R>();
    v3_acc(acc, K0, e0, K1, e1);
    J02 = scale(acc, -1.0 / rdot(P02, P02));
  }
  {
    spinor<R> b0 = szero<R>(), b1 = szero<R>();
    ften<R> F = fzero<R>();
    wedge_acc(F, cast<R>(P02), J02); wedge_acc(F, e0, e1);
    absorb0(b0, b1, J02, F);
    F = fzero<R>();
    wedge_acc(F, cast<R>(K1), e1);
    absorb(b0, b1, U1, e1, F);
    propagate(b0, b1, rsub(pt, P02), U2);
  }
  // level 3
  const rvec4<double> P13 = radd(K1, K2), P03 = radd(P02, K2);
  vec4<R> J13, J03;
  {
    vec4<R> acc = vzero<R>();
    v3_acc(acc, K1, e1, K2, e2);
    J13 = scale(acc, -1.0 / rdot(P13, P13));
    acc = vzero<R>();
    v3_acc(acc, K0, e0, P13, J13);
    v3_acc(acc, P02, J02, K2, e2);
    v4_acc(acc, e0, e1, e2);
    J03 = scale(acc, -1.0 / rdot(P03, P03));
  }
  spinor<R> b0 = szero<R>(), b1 = szero<R>();
  {
    ften<R> F = fzero<R>();
    wedge_acc(F, cast<R>(P03), J03); wedge_acc(F, e0, J13); wedge_acc(F, J02, e2);
    absorb0(b0, b1, J03, F);
    F = fzero<R>();
    wedge_acc(F, cast<R>(P13), J13); wedge_acc(F, e1, e2);
    absorb(b0, b1, U1, J13, F);
    F = fzero<R>();
    wedge_acc(F, cast<R>(K2), e2);
    absorb(b0, b1, U2, e2, F);
  }
#pragma unroll
  for (int iv = 0; iv < 2; ++iv) { A[0][iv] = row_col(b0, v[iv]); A[1][iv] = row_col(b1, v[iv]); }
}

// S_L = {}: three sources (a, b, Q0), Q0 = (w gamma x) / Kq^2, six orderings
template <class R>
TREX_QQ2_FN void qq2_group0(const Qq2Ext<R>& X, const spinor<R>& ubar_t, const spinor<R> vtb[2], double mt, double mGt, const Qq2Acc<R>& fl) {
  const rvec4<double> Kq = radd(X.Kr, X.Kc);
  const vec4<R> Q0 = qq2_scaled(bilinear(X.w, X.x), 1.0 / rdot(Kq, Kq));
  auto src_e = [&](int i) { return i == 0 ? X.e[0] : (i == 1 ? X.e[1] : Q0); };
  auto src_K = [&](int i) { return i == 0 ? X.K[0] : (i == 1 ? X.K[1] : Kq); };
  // orderings in lexicographic order of (a, b, Q) = (0, 1, 2): (a,b,Q) (a,Q,b) (b,a,Q) (b,Q,a) (Q,a,b) (Q,b,a);
  // type I pair = (gluons before Q; gluons after Q), type II pair = (all gluons in order; -)
#pragma unroll 1
  for (int o = 0; o < 6; ++o) {
    const int i0 = o >> 1, r = o & 1;
    const int i1 = i0 == 0 ? 1 + r : (i0 == 1 ? 2 * r : r), i2 = 3 - i0 - i1;
    cx<R> A[2][2];
    three_source_path<R>(ubar_t, X.pt, src_e(i0), src_K(i0), src_e(i1), src_K(i1), src_e(i2), src_K(i2), mt, mGt, vtb, A);
    const int f1 = o == 0 ? 0 : o == 1 ? 2 : o == 2 ? 1 : o == 3 ? 3 : o == 4 ? 4 : 5;
    const int f2 = (o == 0 || o == 1 || o == 4) ? 0 : 1;
    fl.add(f1, f2, A);
  }
}

// S_L = {x}: the other gluon y and Q(x|) / Q(|x)
template <class R>
TREX_QQ2_FN void qq2_group1(const Qq2Ext<R>& X, const spinor<R>& ubar_t, const spinor<R> vtb[2], double mt, double mGt, const Qq2Acc<R>& fl) {
  const rvec4<double> Kq = radd(X.Kr, X.Kc);
#pragma unroll 1
  for (int k = 0; k < 4; ++k) {
    const int xg = k >> 1, yg = 1 - xg, col_end = k & 1;
    const rvec4<double> Kqx = radd(Kq, X.K[xg]);
    const double iP2 = 1.0 / rdot(Kqx, Kqx);
    const vec4<R> ex = xg ? X.e[1] : X.e[0], ey = yg ? X.e[1] : X.e[0];
    const rvec4<double> Kx = xg ? X.K[1] : X.K[0], Ky = yg ? X.K[1] : X.K[0];
    const vec4<R> Q = col_end ? qq2_scaled(bilinear(X.w, qq2_col1(X.x, X.Kc, ex, Kx)), iP2)
                              : qq2_scaled(bilinear(qq2_row1(X.w, X.Kr, ex, Kx), X.x), iP2);
    cx<R> A12[2][2], A21[2][2];                            // (y, Q'), (Q', y)
    two_source_line<R>(ubar_t, X.pt, ey, Ky, Q, Kqx, mt, mGt, vtb, A12, A21);
    // pair numbers: (a; b) = 2, (b; a) = 3, (-; x y) = 4 + xg, (y x; -) = yg
    const int p_yx = 2 + yg, p_xy = 2 + xg;
    fl.add(col_end ? yg : p_yx, p_yx, A12);
    fl.add(col_end ? p_xy : 4 + xg, p_yx, A21);
  }
}

// S_L = {a, b}: single source; (ab|) (ba|) (a|b) (b|a) (|ab) (|ba) -> type I pairs 4 5 3 2 0 1, type II pairs 4 5 4 5 4 5
template <class R>
TREX_QQ2_FN void qq2_group2(const Qq2Ext<R>& X, const spinor<R>& ubar_t, const spinor<R> vtb[2], const Qq2Acc<R>& fl) {
  const rvec4<double> Kq = radd(X.Kr, X.Kc);
  {
    const rvec4<double> Kab = radd(X.K[0], X.K[1]);
    const rvec4<double> Ptot = radd(Kq, Kab);
    const rvec4<R> Pr = cast<R>(Ptot);
    const double iP2 = 1.0 / rdot(Ptot, Ptot);
    vec4<R> Jab;                                           // merged current of the tuple (a, b); (b, a) has the opposite sign
    {
      vec4<R> acc = vzero<R>();
      v3_acc(acc, X.K[0], X.e[0], X.K[1], X.e[1]);
      Jab = qq2_scaled(acc, -1.0 / rdot(Kab, Kab));
    }
    rvec4<double> qr, qc;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) { qr.c[mu] = -(X.Kr.c[mu] + Kab.c[mu]); qc.c[mu] = X.Kc.c[mu] + Kab.c[mu]; }
    const R sr = R(-1.0 / rdot(qr, qr)), sc = R(-1.0 / rdot(qc, qc));
#pragma unroll 1
    for (int ord = 0; ord < 2; ++ord) {                    // ord 0: strings (a, b); 1: (b, a)
      const vec4<R> e1 = ord ? X.e[1] : X.e[0], e2 = ord ? X.e[0] : X.e[1];
      const rvec4<double> K1 = ord ? X.K[1] : X.K[0], K2 = ord ? X.K[0] : X.K[1];
      const R sg = ord ? R(-1) : R(1);
      const spinor<R> R1 = qq2_row1(X.w, X.Kr, e1, K1), C2 = qq2_col1(X.x, X.Kc, e2, K2);
      cx<R> A[2][2];
      // (g1 g2 |): R_2 = -[ R_g1 eslash_g2 + w Jslash ] qslash / q^2
      {
        spinor<R> t = row_slash(R1, e2);
        const spinor<R> wJ = row_slash(X.w, Jab);
#pragma unroll
        for (int i = 0; i < 4; ++i) cfma(t.c[i], wJ.c[i], sg);
        spinor<R> R2 = row_slash(t, cast<R>(qr));
#pragma unroll
        for (int i = 0; i < 4; ++i) R2.c[i] = R2.c[i] * sr;
        qq2_single(ubar_t, vtb, qq2_scaled(bilinear(R2, X.x), iP2), Pr, A);
        fl.add(4 + ord, 4 + ord, A);
      }
      // (g1 | g2)
      qq2_single(ubar_t, vtb, qq2_scaled(bilinear(R1, C2), iP2), Pr, A);
      fl.add(3 - ord, 4 + ord, A);
      // (| g1 g2), g2 next to the column end: C = -qslash [ eslash_g1 C_g2 + Jslash x ] / q^2
      {
        spinor<R> u = slash_col(e1, C2);
        const spinor<R> Jx = slash_col(Jab, X.x);
#pragma unroll
        for (int i = 0; i < 4; ++i) cfma(u.c[i], Jx.c[i], sg);
        spinor<R> Cc = slash_col(cast<R>(qc), u);
#pragma unroll
        for (int i = 0; i < 4; ++i) Cc.c[i] = Cc.c[i] * sc;
        qq2_single(ubar_t, vtb, qq2_scaled(bilinear(X.w, Cc), iP2), Pr, A);
        fl.add(ord, 4 + ord, A);
      }
    }
  }
}

// all twelve flows
template <class R>
TREX_HD void qq2_flows(const Qq2Ext<R>& X, const spinor<R>& ubar_t, const spinor<R> vtb[2], double mt, double mGt, const Qq2Acc<R>& fl) {
  fl.clear();
  qq2_group0<R>(X, ubar_t, vtb, mt, mGt, fl);
  qq2_group1<R>(X, ubar_t, vtb, mt, mGt, fl);
  qq2_group2<R>(X, ubar_t, vtb, fl);
}

// sum over the top helicity (and both antitop helicities) of x^dagger C x at theta_old and theta_new for one choice of the
// light-line combination c and the gluon helicities; pm = momenta of the event [leg][mu]; fl = this thread's flow storage
template <class R, class RC>
TREX_HD void qq2_unit(const double (*pm)[4], const QLineLegs& L, int c, int la, int lb, const ThetaPair& T, const Qq2Acc<R>& fl, RC out[2],
                      double* dbg = nullptr) {
  const bool row_in = L.lrow < 2, col_in = L.lcol < 2;
  // row spinor in the upper block for c = 1 (see k_qq)
  const bool row_upper = c != 0, col_upper = !row_upper;
  Qq2Ext<R> X;
  {
    const int lam = (row_in ? !row_upper : row_upper) ? 1 : -1;
    X.w = cast<R>(row_in ? bar(spinor_v<double>(pm[L.lrow], lam, true)) : bar(spinor_u<double>(pm[L.lrow], lam, true)));
    const int lamc = (col_in ? !col_upper : col_upper) ? 1 : -1;
    X.x = cast<R>(col_in ? spinor_u<double>(pm[L.lcol], lamc, true) : spinor_v<double>(pm[L.lcol], lamc, true));
  }
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    X.Kr.c[mu] = row_in ? pm[L.lrow][mu] : -pm[L.lrow][mu];
    X.Kc.c[mu] = col_in ? pm[L.lcol][mu] : -pm[L.lcol][mu];
    X.pt.c[mu] = pm[2][mu];
  }
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    const int lg = g == 0 ? L.lg : L.lg2;
    const bool g_in = lg < 2;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) X.K[g].c[mu] = g_in ? pm[lg][mu] : -pm[lg][mu];
    X.e[g] = cast<R>(polvec<double>(pm[lg], (g == 0 ? la : lb) ? 1 : -1, !g_in));
  }
  const spinor<R> vtb[2] = {cast<R>(spinor_v<double>(pm[3], -1, false)), cast<R>(spinor_v<double>(pm[3], +1, false))};
  const bool same_line = (T.mt[0] == T.mt[1]) && (T.mGt[0] == T.mGt[1]);
  RC acc[2] = {RC(0), RC(0)};
#pragma unroll 1
  for (int lt = 0; lt < 2; ++lt) {
    const spinor<R> ubar_t = cast<R>(bar(spinor_u<double>(pm[2], lt ? 1 : -1, false)));
#pragma unroll 1
    for (int th = 0; th < 2; ++th) {
      if (th == 0 || !same_line) qq2_flows<R>(X, ubar_t, vtb, T.mt[th], T.mGt[th], fl);
      const R kq = R(T.kq[th]);
#pragma unroll 1
      for (int iv = 0; iv < 2; ++iv) {
        cx<RC> xf[QQ2_NFLOW];
#pragma unroll
        for (int f = 0; f < QQ2_NFLOW; ++f) {
          cx<R> a = fl.get(f, 0, iv);
          cfma(a, fl.get(f, 1, iv), kq);
          xf[f] = cx<RC>(RC(a.re), RC(a.im));
        }
        const RC q = colour_quadform<RC, QQ2_NFLOW, 1>(xf, nullptr);
        if (dbg) dbg[(lt * 2 + iv) * 2 + th] = (double)q;     // diagnostics only (trex_debug_helicity_me2)
        acc[th] += q;
      }
    }
  }
  out[0] = acc[0]; out[1] = acc[1];
}

}  // namespace trex
