// trex_proc.cuh -- per-thread evaluation of one helicity "unit" of one event for every compiled-in subprocess
// (SURVEY.md 8(a) a6-a8): external wavefunctions, colour-flow amplitudes, colour sum J^dagger C J.
//
// A unit fixes the helicities of every leg except the antitop (gluons / light quarks and the top); both antitop
// helicities are closed inside the unit because they only differ in the final contraction with v(p_tbar, lambda).
// All functions return sum over the unit's helicities of  x^dagger C x  for theta_old and theta_new at g_s = 1;
// the caller multiplies by g_s^(2 n_vertices) / N_avg.
#pragma once
#include <type_traits>

#include "trex_ttng.cuh"

namespace trex {

// ---------------------------------------------------------------- per-call parameters (uniform over the grid)
struct ThetaPair {           // index 0 = theta_old, 1 = theta_new
  double mt[2], mGt[2];      // top mass, m_t * Gamma_t
  double kq[2];              // kappa / g_s
  double pref[2];            // g_s^(2 nv) / N_avg
  double gs2nv[2];           // g_s^(2 nv) alone (the quark-channel family kernel divides by its class's N_avg itself)
  // electroweak (e- e+ -> mu- mu+)
  double e2[2], gL[2], gR[2], mZ2[2], mZGZ[2];
};

// ---------------------------------------------------------------- colour matrices
// t t~ + n gluons: C_{sigma sigma'} = sum_a tr(T^{a_s1}..T^{a_sn} T^{a_s'n}..T^{a_s'1}), built by the host at first use
// (trex_colour.h: Fierz reduction in exact rational arithmetic). Every translation unit that instantiates the
// g g -> t t~ + gluons kernel for one N owns one constant-memory table holding that N's matrix (ncol = 2, 6, 24), so
// that the fully unrolled colour sums read the entries as instruction operands; ncol = 120 lives in global memory.
#if defined(__CUDACC__)
static __constant__ double c_Ctab[576];
#else
static double c_Ctab[576];
#endif

template <int NC> TREX_HD double colour_entry(const double* __restrict__ Cg, int i, int j) {
  if constexpr (NC <= 24) return c_Ctab[i * NC + j];
  else {
#if defined(__CUDA_ARCH__)
    return __ldg(Cg + i * NC + j);
#else
    return Cg[i * NC + j];
#endif
  }
}

// x^dagger C x for real symmetric C: sum_j [ C_jj |x_j|^2 + 2 Re(conj(x_j) sum_{i<j} C_ji x_i) ]
template <class RC, int NC, int STRIDE> TREX_HD RC colour_quadform(const cx<RC>* x, const double* __restrict__ Cg) {
  RC tot = RC(0);
  if constexpr (NC <= 24) {
#pragma unroll
    for (int j = 0; j < NC; ++j) {
      cx<RC> t(RC(0), RC(0));
#pragma unroll
      for (int i = 0; i < j; ++i) cfma(t, x[i * STRIDE], RC(colour_entry<NC>(Cg, j, i)));
      cx<RC> xj = x[j * STRIDE];
      cfma(t, xj, RC(0.5 * colour_entry<NC>(Cg, j, j)));
      tot += RC(2) * (xj.re * t.re + xj.im * t.im);
    }
  } else {
    // rolled, 4 rows of C at a time so that every x_i loaded from local memory feeds 8 FMAs
    static_assert(NC % 4 == 0, "ncolor must be a multiple of 4");
    for (int j0 = 0; j0 < NC; j0 += 4) {
      cx<RC> t[4];
#pragma unroll
      for (int r = 0; r < 4; ++r) t[r] = cx<RC>(RC(0), RC(0));
      for (int i = 0; i < j0; ++i) {
        cx<RC> xi = x[i * STRIDE];
#pragma unroll
        for (int r = 0; r < 4; ++r) cfma(t[r], xi, RC(colour_entry<NC>(Cg, j0 + r, i)));
      }
#pragma unroll
      for (int r = 0; r < 4; ++r) {
#pragma unroll
        for (int i = 0; i < r; ++i) cfma(t[r], x[(j0 + i) * STRIDE], RC(colour_entry<NC>(Cg, j0 + r, j0 + i)));
        cx<RC> xj = x[(j0 + r) * STRIDE];
        cfma(t[r], xj, RC(0.5 * colour_entry<NC>(Cg, j0 + r, j0 + r)));
        tot += RC(2) * (xj.re * t[r].re + xj.im * t[r].im);
      }
    }
  }
  return tot;
}

// ---------------------------------------------------------------- momenta
// SoA block [npar][4][n]: component (ipar*4+mu) of event e at (ipar*4+mu)*n + e  (coalesced across a warp)
template <class R> TREX_HD void load_leg(const double* __restrict__ mom, long n, long e, int leg, R p[4]) {
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) p[mu] = R(mom[(long)(leg * 4 + mu) * n + e]);
}

#if defined(__CUDACC__)
__host__ __device__
#endif
constexpr int factorial(int n) { return n <= 1 ? 1 : n * factorial(n - 1); }

// ---------------------------------------------------------------- g g -> t t~ + (N-2) g
// legs: 0,1 incoming gluons; 2 top; 3 antitop; 4.. outgoing gluons. unit = gluon helicity bits (bit g of `gh` for
// gluon g in the order g1 g2 g3.. ) and the top helicity. x[leaf][v][theta] is stored in precision RC.
template <class R, class RC, int N, int NPASS> struct TtngLeafStore {
  static constexpr int NC = factorial(N);
  cx<RC> x[NC][2][2];
  spinor<R> v[2];          // v(p_tbar, -), v(p_tbar, +)
  R kq[2];
  template <int LEAF> TREX_HD void put(const spinor<R>* b0, const spinor<R>* b1) { (*this)(LEAF, b0, b1); }
  TREX_HD void operator()(int leaf, const spinor<R>* b0, const spinor<R>* b1) {
#pragma unroll
    for (int th = 0; th < 2; ++th) {
      const int p = NPASS == 2 ? th : 0;
#pragma unroll
      for (int iv = 0; iv < 2; ++iv) {
        cx<R> a0 = row_col(b0[p], v[iv]), a1 = row_col(b1[p], v[iv]);
        cfma(a0, a1, kq[th]);
        x[leaf][iv][th] = cx<RC>(RC(a0.re), RC(a0.im));
      }
    }
  }
};

template <class R, class RC, int N, int NPASS>
TREX_HD void ttng_unit(const double* __restrict__ mom, long n, long e, int gh, int lam_t, const ThetaPair& T,
                       const double* __restrict__ Cg, RC out[2]) {
  constexpr int NC = factorial(N);
  using Store = TtngLeafStore<R, RC, N, NPASS>;
  Store st;
  typename std::conditional<(N <= 2), TTNGS<R, N, NPASS, Store>, TTNG<R, N, NPASS, Store>>::type t;
#pragma unroll
  for (int g = 0; g < N; ++g) {
    const int leg = g < 2 ? g : g + 2;
    double p[4]; load_leg<double>(mom, n, e, leg, p);
    const int lam = ((gh >> g) & 1) ? +1 : -1;
    const bool incoming = g < 2;
    t.eps[g] = cast<R>(polvec<double>(p, lam, !incoming));
    const double sg = incoming ? 1.0 : -1.0;
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) t.K[g].c[mu] = sg * p[mu];
  }
  {
    double p[4]; load_leg<double>(mom, n, e, 2, p);
#pragma unroll
    for (int mu = 0; mu < 4; ++mu) t.pt.c[mu] = p[mu];
    t.ubar_t = cast<R>(bar(spinor_u<double>(p, lam_t, false)));
    double q[4]; load_leg<double>(mom, n, e, 3, q);
    st.v[0] = cast<R>(spinor_v<double>(q, -1, false));
    st.v[1] = cast<R>(spinor_v<double>(q, +1, false));
  }
#pragma unroll
  for (int p = 0; p < NPASS; ++p) { t.line[p].mt = T.mt[p]; t.line[p].mGt = T.mGt[p]; }
  st.kq[0] = R(T.kq[0]); st.kq[1] = R(T.kq[1]);
  t.run(&st);
#pragma unroll
  for (int th = 0; th < 2; ++th) {
    RC s = RC(0);
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) s += colour_quadform<RC, NC, 4>(&st.x[0][iv][th], Cg);
    out[th] = s;
  }
}

// ---------------------------------------------------------------- one light-quark line + t t~ + one gluon
// (q q~ -> t t~ g, q g -> t t~ q, g q~ -> t t~ q~; R-8). The light line (row spinor w at leg lrow, column
// spinor x at leg lcol) acts on the top line as a second gluon source; with the Fierz identity the five SM diagrams
// (+ dipole / contact insertions) reduce to four colour flows
//   c1 = T^a_{i1 j3} d_{i4 j2}, c2 = d_{i1 j3} T^a_{i4 j2}, c3 = T^a_{i1 j2} d_{i4 j3}, c4 = d_{i1 j2} T^a_{i4 j3}
//   J1 = (A(g,Q) + K4)/2, J2 = (A(Q,g) + K3)/2, J3 = -(A(g,Q) + A(Q,g))/6, J4 = -(K3 + K4)/6
// where A(.,.) are the two orderings of (gluon, quark-pair current) on the top line and K3 / K4 attach the current
// of the light line that has radiated the gluon at its row / column end. C = [[12,0,4,4],[0,12,4,4],[4,4,12,0],[4,4,0,12]].
struct QLineLegs { int lrow, lcol, lg, lg2; };   // leg numbers (lg2: second gluon of the two-gluon channels, trex_qq2.cuh); legs 0,1 are incoming


// Top line with TWO ordered sources (currents e1, e2 with momenta K1, K2 flowing into the line): the two orderings
// A(1,2), A(2,1), each as (order 0, order 1 in kappa) for both antitop helicities: A12[order][v], A21[order][v].
// Same recursion as TTNGS<R, 2, 1, .>, written out with the merged current formed once (J_21 = -J_12)
// and the orderings in a rolled loop, so that the live state is one line spinor pair (cf. k_gg_tt).
template <class R>
TREX_HD void two_source_line(const spinor<R>& ubar, const rvec4<double>& pt, const vec4<R>& e1, const rvec4<double>& K1,
                             const vec4<R>& e2, const rvec4<double>& K2, double mt_d, double mGt, const spinor<R> v[2],
                             cx<R> A12[2][2], cx<R> A21[2][2]) {
  spinor<R> d0, d1 = szero<R>();
  {
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
  const R mt = R(mt_d);
#pragma unroll 1
  for (int ord = 0; ord < 2; ++ord) {
    const vec4<R>& ea = ord ? e2 : e1; const vec4<R>& eb = ord ? e1 : e2;
    const rvec4<double>& Ka = ord ? K2 : K1; const rvec4<double>& Kb = ord ? K1 : K2;
    dspinor<R> U1;
    {
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
      const cx<double> den(q2 - mt_d * mt_d, mGt);
      const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
      const spinor<R> s0 = row_slash(c0, q), s1 = row_slash(c1, q);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        cx<R> n0 = s0.c[i]; cfma(n0, c0.c[i], mt);
        cx<R> n1 = s1.c[i]; cfma(n1, c1.c[i], mt);
        U1.o0.c[i] = n0 * pr; U1.o1.c[i] = n1 * pr;
      }
    }
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
    cx<R> (*A)[2] = ord ? A21 : A12;
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) { A[0][iv] = row_col(b0, v[iv]); A[1][iv] = row_col(b1, v[iv]); }
  }
}

// top line of the quark channels, given the gluon polarisation, the quark-pair current Jq and the two currents Jq3 / Jq4
// of the light line that has radiated the gluon: two-source ordered amplitudes + single-source amplitudes -> four colour
// flows -> J^dagger C J for theta_old and theta_new, both antitop helicities (see the comment block above)
template <class R, class RC>
TREX_HD void qq_close(const vec4<R>& eg, const rvec4<double>& Kg, const vec4<R>& Jq, const rvec4<double>& Kq, const vec4<R>& Jq3,
                      const vec4<R>& Jq4, const rvec4<double>& Ptot, const spinor<R>& ubar_t, const spinor<R> vtb[2],
                      const rvec4<double>& pt, const ThetaPair& T, RC out[2], double* dbg = nullptr) {
  const spinor<R>* stv = vtb;
  // single-source brackets of K3, K4: ubar_t [ i Jslash + (kappa/g_s) 2 sigma(P ^ J) ]; they depend neither on theta nor on
  // the antitop helicity, so they are formed once
  spinor<R> c30 = row_slash(ubar_t, Jq3), c31 = szero<R>(), c40 = row_slash(ubar_t, Jq4), c41 = szero<R>();
  { ften<R> F = fzero<R>(); wedge_acc(F, cast<R>(Ptot), Jq3); row_sigma_acc(c31, ubar_t, F); }
  { ften<R> F = fzero<R>(); wedge_acc(F, cast<R>(Ptot), Jq4); row_sigma_acc(c41, ubar_t, F); }
  cx<R> k30[2], k31[2], k40[2], k41[2];
#pragma unroll
  for (int iv = 0; iv < 2; ++iv) {
    k30[iv] = mul_i(row_col(c30, stv[iv])); k31[iv] = row_col(c31, stv[iv]);
    k40[iv] = mul_i(row_col(c40, stv[iv])); k41[iv] = row_col(c41, stv[iv]);
  }
  // top mass/width may differ between theta_old and theta_new: the two-source walk is repeated per theta when they do
  RC res[2];
  const bool same_line = (T.mt[0] == T.mt[1]) && (T.mGt[0] == T.mGt[1]);
  cx<R> A12[2][2], A21[2][2];   // [order][v]
  for (int th = 0; th < 2; ++th) {
    if (th == 0 || !same_line)
      two_source_line<R>(ubar_t, pt, eg, Kg, Jq, Kq, T.mt[th], T.mGt[th], vtb, A12, A21);
    const R kq = R(T.kq[th]);
    RC s = RC(0);
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) {
      cx<R> k3 = k30[iv]; cfma(k3, k31[iv], kq);
      cx<R> k4 = k40[iv]; cfma(k4, k41[iv], kq);
      cx<R> a12 = A12[0][iv]; cfma(a12, A12[1][iv], kq);
      cx<R> a21 = A21[0][iv]; cfma(a21, A21[1][iv], kq);
      cx<R> j1 = R(0.5) * (a12 + k4), j2 = R(0.5) * (a21 + k3);
      cx<R> j3 = R(-1.0 / 6.0) * (a12 + a21), j4 = R(-1.0 / 6.0) * (k3 + k4);
      cx<RC> J[4] = {cx<RC>(RC(j1.re), RC(j1.im)), cx<RC>(RC(j2.re), RC(j2.im)), cx<RC>(RC(j3.re), RC(j3.im)), cx<RC>(RC(j4.re), RC(j4.im))};
      // J^dagger C J with C = 12 on the diagonal, 4 between {1,2} and {3,4}, 0 inside the pairs
      RC d = RC(12) * (norm2(J[0]) + norm2(J[1]) + norm2(J[2]) + norm2(J[3]));
      cx<RC> a = J[0] + J[1], b = J[2] + J[3];
      d += RC(8) * (a.re * b.re + a.im * b.im);
      if (dbg) dbg[iv * 2 + th] = (double)d;                // diagnostics only (trex_debug_helicity_me2)
      s += d;
    }
    res[th] = s;
  }
  out[0] = res[0]; out[1] = res[1];
}

// ---------------------------------------------------------------- e- e+ -> mu- mu+ (photon + Z), all 16 helicities
// M = i [ e^2 (Je.Jm)/s + (gL JeL + gR JeR).(gL JmL + gR JmR)/(s - mZ^2 + i mZ GZ) ], J^mu_{L,R} = wbar gamma^mu P_{L,R} x.
// The four chiral current products d_ab = Je_a . Jm_b do not depend on theta: evaluated once, closed with both
// coupling sets.
template <class R>
TREX_HD void eemumu_event(const double* __restrict__ mom, long n, long e, const ThetaPair& T, R out[2]) {
  double p0[4], p1[4], p2[4], p3[4];
  load_leg<double>(mom, n, e, 0, p0); load_leg<double>(mom, n, e, 1, p1); load_leg<double>(mom, n, e, 2, p2); load_leg<double>(mom, n, e, 3, p3);
  double q[4]; for (int mu = 0; mu < 4; ++mu) q[mu] = p0[mu] + p1[mu];
  const double s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3];
  cx<R> propZ[2]; R propA[2];
  for (int th = 0; th < 2; ++th) {
    propA[th] = R(T.e2[th] / s);
    propZ[th] = cast<R>(cdiv(cx<double>(1, 0), cx<double>(s - T.mZ2[th], T.mZGZ[th])));
  }
  // the eight external wavefunctions once (not once per helicity combination)
  spinor<R> u1[2], vb2[2], ub3[2], v4[2];
#pragma unroll
  for (int l = 0; l < 2; ++l) {
    const int lam = l ? 1 : -1;
    u1[l] = cast<R>(spinor_u<double>(p0, lam, true));
    vb2[l] = cast<R>(bar(spinor_v<double>(p1, lam, true)));
    ub3[l] = cast<R>(bar(spinor_u<double>(p2, lam, true)));
    v4[l] = cast<R>(spinor_v<double>(p3, lam, true));
  }
  R sum[2] = {R(0), R(0)};
  // Massless lines: a spinor has one non-zero chiral 2-block (u(+), v(-): lower; u(-), v(+): upper; the bar swaps them)
  // and gamma^mu couples upper to lower, so vbar(l2) gamma^mu u(l1) vanishes EXACTLY unless l1 = -l2 (and likewise the
  // muon current): 4 of the 16 helicity combinations contribute, each with ONE chirality (a = L or R) per current.
#pragma unroll
  for (int he = 0; he < 2; ++he) {
#pragma unroll
    for (int hm = 0; hm < 2; ++hm) {
      // electron line: u(l1) with vbar(-l1); muon line: ubar(l3) with v(-l3); chirality index 0 = L (upper block of the
      // column spinor), 1 = R
      const spinor<R>& ue = u1[he]; const spinor<R>& ve = vb2[1 - he];
      const spinor<R>& um = ub3[hm]; const spinor<R>& vm = v4[1 - hm];
      const int a = he, b = hm;                            // u(-): upper block = L; the partner of ubar(-) is v(+): upper block = L
      const cx<R> d = dot(bilinear(ve, ue), bilinear(um, vm));
#pragma unroll
      for (int th = 0; th < 2; ++th) {
        const R g[2] = {R(T.gL[th]), R(T.gR[th])};
        const cx<R> M = d * propA[th] + (d * (g[a] * g[b])) * propZ[th];
        sum[th] += norm2(M);
      }
    }
  }
  out[0] = sum[0]; out[1] = sum[1];
}

}  // namespace trex
