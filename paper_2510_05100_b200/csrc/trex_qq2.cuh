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
//     S_L = {}     : six orderings of (a, b, Q) on the top line                      (TTNGS<3>)
//     S_L = {x}    : Q(x|) and Q(|x), two orderings of (y, Q) each                    (two_source_line)
//     S_L = {a, b} : Q(ab|) Q(ba|) Q(a|b) Q(b|a) Q(|ab) Q(|ba), single source        (one bracket each)
// The 12 x 12 colour matrix comes from trex_colour.h (traces of the strings, exact rationals).
#pragma once
#include "trex_proc.cuh"

namespace trex {

constexpr int QQ2_NFLOW = 12;

// amplitudes of one (light-line, gluon, top) helicity choice, both antitop helicities: F[flow][order in kappa][v]
template <class R> struct Qq2Flows {
  cx<R> F[QQ2_NFLOW][2][2];
  TREX_HD void clear() {
#pragma unroll
    for (int f = 0; f < QQ2_NFLOW; ++f)
#pragma unroll
      for (int o = 0; o < 2; ++o) { F[f][o][0] = cx<R>(0, 0); F[f][o][1] = cx<R>(0, 0); }
  }
  // one term: +1/2 to its type-I flow, -1/6 to its type-II flow
  TREX_HD void add(int f1, int f2, const cx<R> A[2][2]) {
#pragma unroll
    for (int o = 0; o < 2; ++o)
#pragma unroll
      for (int iv = 0; iv < 2; ++iv) {
        cfma(F[f1][o][iv], A[o][iv], R(0.5));
        cfma(F[6 + f2][o][iv], A[o][iv], R(-1.0 / 6.0));
      }
  }
};

// sink of the three-source walk (sources 0 = a, 1 = b, 2 = Q; leaves in lexicographic order)
template <class R> struct Qq2Sink3 {
  Qq2Flows<R>* fl;
  const spinor<R>* v;
  template <int LEAF> TREX_HD void put(const spinor<R>* b0, const spinor<R>* b1) {
    // leaf: 0 (a,b,Q) 1 (a,Q,b) 2 (b,a,Q) 3 (b,Q,a) 4 (Q,a,b) 5 (Q,b,a)
    constexpr int f1 = LEAF == 0 ? 0 : LEAF == 1 ? 2 : LEAF == 2 ? 1 : LEAF == 3 ? 3 : LEAF == 4 ? 4 : 5;
    constexpr int f2 = (LEAF == 0 || LEAF == 1 || LEAF == 4) ? 0 : 1;
    cx<R> A[2][2];
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) { A[0][iv] = row_col(b0[0], v[iv]); A[1][iv] = row_col(b1[0], v[iv]); }
    fl->add(f1, f2, A);
  }
};

// the eleven currents of the light line for one choice of its helicity combination and of the gluon helicities
template <class R> struct Qq2Currents {
  vec4<R> Q0;            // no gluon absorbed
  vec4<R> Qr[2], Qc[2];  // gluon x (0 = a, 1 = b) absorbed at the row / column end
  vec4<R> Q2[6];         // both: (ab|) (ba|) (a|b) (b|a) (|ab) (|ba)
};

template <class R>
TREX_HD void qq2_light_line(const spinor<R>& w, const spinor<R>& x, const rvec4<double>& Kr, const rvec4<double>& Kc, const vec4<R> e[2],
                            const rvec4<double> K[2], Qq2Currents<R>& out) {
  const rvec4<double> Kq = radd(Kr, Kc);
  auto scaled = [](const vec4<R>& j, double s) { vec4<R> o; const R sr = R(s);
#pragma unroll
    for (int i = 0; i < 4; ++i) o.c[i] = j.c[i] * sr; return o; };
  out.Q0 = scaled(bilinear(w, x), 1.0 / rdot(Kq, Kq));
  // one gluon: R_x = w (i eslash)(i qslash)/q^2 = -w eslash qslash / q^2, q = -(Kr + Kx);  C_x = -qslash eslash x / q^2, q = Kc + Kx
  spinor<R> Rx[2], Cx[2];
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    rvec4<double> qr, qc;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) { qr.c[mu] = -(Kr.c[mu] + K[g].c[mu]); qc.c[mu] = Kc.c[mu] + K[g].c[mu]; }
    const R sr = R(-1.0 / rdot(qr, qr)), sc = R(-1.0 / rdot(qc, qc));
    Rx[g] = row_slash(row_slash(w, e[g]), cast<R>(qr));
    Cx[g] = slash_col(cast<R>(qc), slash_col(e[g], x));
#pragma unroll
    for (int i = 0; i < 4; ++i) { Rx[g].c[i] = Rx[g].c[i] * sr; Cx[g].c[i] = Cx[g].c[i] * sc; }
    const rvec4<double> P = radd(Kq, K[g]);
    const double iP2 = 1.0 / rdot(P, P);
    out.Qr[g] = scaled(bilinear(Rx[g], x), iP2);
    out.Qc[g] = scaled(bilinear(w, Cx[g]), iP2);
  }
  // both gluons: merged current of the tuple (a, b); the tuple (b, a) has the opposite sign
  const rvec4<double> Kab = radd(K[0], K[1]);
  vec4<R> Jab;
  {
    vec4<R> acc = vzero<R>();
    v3_acc(acc, K[0], e[0], K[1], e[1]);
    Jab = scaled(acc, -1.0 / rdot(Kab, Kab));
  }
  rvec4<double> qr, qc;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) { qr.c[mu] = -(Kr.c[mu] + Kab.c[mu]); qc.c[mu] = Kc.c[mu] + Kab.c[mu]; }
  const R sr = R(-1.0 / rdot(qr, qr)), sc = R(-1.0 / rdot(qc, qc));
  const rvec4<double> P = radd(Kq, Kab);
  const double iP2 = 1.0 / rdot(P, P);
  const spinor<R> wJ = row_slash(w, Jab), Jx = slash_col(Jab, x);
#pragma unroll
  for (int ord = 0; ord < 2; ++ord) {                       // ord 0: (a, b); 1: (b, a)
    const int g1 = ord, g2 = 1 - ord;
    const R sg = ord ? R(-1) : R(1);
    // R_2 = -[ R_g1 eslash_g2 + w Jslash ] qslash / q^2
    spinor<R> t = row_slash(Rx[g1], e[g2]);
#pragma unroll
    for (int i = 0; i < 4; ++i) cfma(t.c[i], wJ.c[i], sg);
    spinor<R> R2 = row_slash(t, cast<R>(qr));
#pragma unroll
    for (int i = 0; i < 4; ++i) R2.c[i] = R2.c[i] * sr;
    out.Q2[ord] = scaled(bilinear(R2, x), iP2);
    // (g1 | g2)
    out.Q2[2 + ord] = scaled(bilinear(Rx[g1], Cx[g2]), iP2);
    // C_2 (string g1 g2, g2 next to the column end) = -qslash [ eslash_g1 C_g2 + Jslash x ] / q^2
    spinor<R> u = slash_col(e[g1], Cx[g2]);
#pragma unroll
    for (int i = 0; i < 4; ++i) cfma(u.c[i], Jx.c[i], sg);
    spinor<R> C2 = slash_col(cast<R>(qc), u);
#pragma unroll
    for (int i = 0; i < 4; ++i) C2.c[i] = C2.c[i] * sc;
    out.Q2[4 + ord] = scaled(bilinear(w, C2), iP2);
  }
}

// all twelve flows for one top helicity and one parameter point's top line
template <class R>
TREX_HD void qq2_flows(const Qq2Currents<R>& Q, const vec4<R> e[2], const rvec4<double> K[2], const rvec4<double>& Kq, const spinor<R>& ubar_t,
                       const spinor<R> vtb[2], const rvec4<double>& pt, double mt, double mGt, Qq2Flows<R>& fl) {
  fl.clear();
  // S_L = {}: three sources
  {
    Qq2Sink3<R> sink{&fl, vtb};
    TTNGS<R, 3, 1, Qq2Sink3<R>> t;
    t.K[0] = K[0]; t.K[1] = K[1]; t.K[2] = Kq;
    t.eps[0] = e[0]; t.eps[1] = e[1]; t.eps[2] = Q.Q0;
    t.pt = pt; t.ubar_t = ubar_t;
    t.line[0].mt = mt; t.line[0].mGt = mGt;
    t.run(&sink);
  }
  // S_L = {x}: the other gluon y and Q(x|) / Q(|x)
#pragma unroll
  for (int xg = 0; xg < 2; ++xg) {
    const int yg = 1 - xg;
    const rvec4<double> Kqx = radd(Kq, K[xg]);
    cx<R> A12[2][2], A21[2][2];                            // (y, Q'), (Q', y)
    // pair numbers: (y; x) = 3 - ... : (a; b) = 2, (b; a) = 3
    const int p_yx = yg == 0 ? 2 : 3, p_xy = xg == 0 ? 2 : 3;
    const int p_0_xy = xg == 0 ? 4 : 5;                    // (-; x y)
    const int p_yx_0 = yg == 0 ? 0 : 1;                    // (y x; -)
    two_source_line<R>(ubar_t, pt, e[yg], K[yg], Q.Qr[xg], Kqx, mt, mGt, vtb, A12, A21);
    fl.add(p_yx, p_yx, A12);
    fl.add(p_0_xy, p_yx, A21);
    two_source_line<R>(ubar_t, pt, e[yg], K[yg], Q.Qc[xg], Kqx, mt, mGt, vtb, A12, A21);
    fl.add(p_yx_0, p_yx, A12);
    fl.add(p_xy, p_yx, A21);
  }
  // S_L = {a, b}: single source
  {
    const rvec4<double> Ptot = radd(Kq, radd(K[0], K[1]));
    const rvec4<R> Pr = cast<R>(Ptot);
    // (ab|) (ba|) (a|b) (b|a) (|ab) (|ba): type I pair, type II pair
    const int f1[6] = {4, 5, 3, 2, 0, 1}, f2[6] = {4, 5, 4, 5, 4, 5};
#pragma unroll
    for (int k = 0; k < 6; ++k) {
      const spinor<R> c0 = row_slash(ubar_t, Q.Q2[k]);
      spinor<R> c1 = szero<R>();
      ften<R> F = fzero<R>();
      wedge_acc(F, Pr, Q.Q2[k]);
      row_sigma_acc(c1, ubar_t, F);
      cx<R> A[2][2];
#pragma unroll
      for (int iv = 0; iv < 2; ++iv) { A[0][iv] = mul_i(row_col(c0, vtb[iv])); A[1][iv] = row_col(c1, vtb[iv]); }
      fl.add(f1[k], f2[k], A);
    }
  }
}

// sum over the top helicity (and both antitop helicities) of x^dagger C x at theta_old and theta_new for one choice of the
// light-line combination c and the gluon helicities; pm = momenta of the event [leg][mu]
template <class R, class RC>
TREX_HD void qq2_unit(const double (*pm)[4], const QLineLegs& L, int c, int la, int lb, const ThetaPair& T, RC out[2]) {
  const bool row_in = L.lrow < 2, col_in = L.lcol < 2;
  // row spinor in the upper block for c = 1 (see k_qq)
  const bool row_upper = c != 0, col_upper = !row_upper;
  spinor<R> w, x;
  {
    const int lam = (row_in ? !row_upper : row_upper) ? 1 : -1;
    w = cast<R>(row_in ? bar(spinor_v<double>(pm[L.lrow], lam, true)) : bar(spinor_u<double>(pm[L.lrow], lam, true)));
    const int lamc = (col_in ? !col_upper : col_upper) ? 1 : -1;
    x = cast<R>(col_in ? spinor_u<double>(pm[L.lcol], lamc, true) : spinor_v<double>(pm[L.lcol], lamc, true));
  }
  rvec4<double> Kr, Kc, K[2], pt;
  vec4<R> e[2];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) {
    Kr.c[mu] = row_in ? pm[L.lrow][mu] : -pm[L.lrow][mu];
    Kc.c[mu] = col_in ? pm[L.lcol][mu] : -pm[L.lcol][mu];
    pt.c[mu] = pm[2][mu];
  }
#pragma unroll
  for (int g = 0; g < 2; ++g) {
    const int lg = g == 0 ? L.lg : L.lg2;
    const bool g_in = lg < 2;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) K[g].c[mu] = g_in ? pm[lg][mu] : -pm[lg][mu];
    e[g] = cast<R>(polvec<double>(pm[lg], (g == 0 ? la : lb) ? 1 : -1, !g_in));
  }
  Qq2Currents<R> Q;
  qq2_light_line<R>(w, x, Kr, Kc, e, K, Q);
  const rvec4<double> Kq = radd(Kr, Kc);
  const spinor<R> vtb[2] = {cast<R>(spinor_v<double>(pm[3], -1, false)), cast<R>(spinor_v<double>(pm[3], +1, false))};
  const bool same_line = (T.mt[0] == T.mt[1]) && (T.mGt[0] == T.mGt[1]);
  RC acc[2] = {RC(0), RC(0)};
#pragma unroll 1
  for (int lt = 0; lt < 2; ++lt) {
    const spinor<R> ubar_t = cast<R>(bar(spinor_u<double>(pm[2], lt ? 1 : -1, false)));
    Qq2Flows<R> fl;
#pragma unroll 1
    for (int th = 0; th < 2; ++th) {
      if (th == 0 || !same_line) qq2_flows<R>(Q, e, K, Kq, ubar_t, vtb, pt, T.mt[th], T.mGt[th], fl);
      const R kq = R(T.kq[th]);
#pragma unroll
      for (int iv = 0; iv < 2; ++iv) {
        cx<RC> xf[QQ2_NFLOW];
#pragma unroll
        for (int f = 0; f < QQ2_NFLOW; ++f) {
          cx<R> a = fl.F[f][0][iv];
          cfma(a, fl.F[f][1][iv], kq);
          xf[f] = cx<RC>(RC(a.re), RC(a.im));
        }
        acc[th] += colour_quadform<RC, QQ2_NFLOW, 1>(xf, nullptr);
      }
    }
  }
  out[0] = acc[0]; out[1] = acc[1];
}

}  // namespace trex
