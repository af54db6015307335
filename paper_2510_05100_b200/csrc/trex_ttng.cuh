// trex_ttng.cuh -- colour-flow amplitudes of a heavy quark line with N ordered gluon "sources".
//
// One thread evaluates ONE gluon-helicity / top-helicity configuration of ONE event. For every ordering sigma of the
// N sources it forms
//   A_sigma = sum over all colour-ordered Feynman diagrams of that ordering,
// by walking the tree of ordering prefixes depth first. At prefix (s_1..s_M) the thread holds
//   J[a][M]  = off-shell gluon current of the contiguous tuple (s_{a+1}..s_M)     (VVV + VVVV vertices, propagator)
//   U[p][M]  = top-line spinor after absorbing (s_1..s_M), with propagator, as a dual number in kappa (FFV vertices,
//              chromomagnetic FFV dipole and FFVV contact at order 1; at most one insertion, R-4)
// Only the current prefix path is alive (N(N+1)/2 currents, N line states): a few hundred doubles per thread instead
// of the O(N!) table a memoised recursion needs. p = 0..NPASS-1 indexes parameter points whose top mass / width
// differ (theta_old, theta_new): the gluon currents are shared between them.
// g_s is factored out: A = g_s^N (A0 + (kappa/g_s) A1); this file computes the open brackets b0, b1 (row spinors, to
// be contracted with v(p_tbar, lambda)) at g_s = 1 and hands them to a sink, leaves in lexicographic order of sigma.
#pragma once
#include "trex_math.cuh"

namespace trex {

struct TopLine {                         // per parameter point
  double mt, mGt;                        // m_t and m_t * Gamma_t
};

template <class R, int N, int NPASS, class Sink> struct TTNG {
  // inputs (thread-private copies; dynamically indexed by the source number, so they live in local memory)
  rvec4<double> K[N];       // incoming-convention momentum of each source (always double)
  vec4<R> eps[N];           // its polarisation / effective current
  rvec4<double> pt;         // top momentum (outgoing)
  spinor<R> ubar_t;         // ubar(p_t, lambda_t)
  TopLine line[NPASS];
  // path state
  vec4<R> J[N][N + 1];      // J[a][m], a < m
  rvec4<double> P[N][N + 1];// momentum of tuple (a+1..m)
  dspinor<R> U[NPASS][N];   // U[p][m], m = 0..N-1 (U[.][0] = ubar_t, order 1 = 0)
  int leaf;
  Sink* sink;

  template <int M> TREX_HD void level(unsigned used) {
    for (int g = 0; g < N; ++g) {
      if ((used >> g) & 1u) continue;
      // --- gluon currents of all tuples ending at position M
      J[M - 1][M] = eps[g];
      P[M - 1][M] = K[g];
#pragma unroll
      for (int a = M - 2; a >= 0; --a) {
        P[a][M] = radd(P[a][M - 1], K[g]);
        vec4<R> acc = vzero<R>();
#pragma unroll
        for (int c = a + 1; c < M; ++c) v3_acc(acc, P[a][c], J[a][c], P[c][M], J[c][M]);
#pragma unroll
        for (int c1 = a + 1; c1 < M; ++c1)
#pragma unroll
          for (int c2 = c1 + 1; c2 < M; ++c2) v4_acc(acc, J[a][c1], J[c1][c2], J[c2][M]);
        // (-i/P^2) * [(-i)V3 + (-i)V4] = -(V3 + V4)/P^2 at g_s = 1
        R s = R(-1.0 / rdot(P[a][M], P[a][M]));
#pragma unroll
        for (int i = 0; i < 4; ++i) J[a][M].c[i] = acc.c[i] * s;
      }
      // --- top line: bracket(M) = sum_a U(a) Gamma(J[a][M]) + order-1 field-strength insertions
      spinor<R> b0[NPASS], b1[NPASS];
#pragma unroll
      for (int p = 0; p < NPASS; ++p) { b0[p] = szero<R>(); b1[p] = szero<R>(); }
#pragma unroll
      for (int a = 0; a < M; ++a) {
        // F = P ^ J (dipole, gluon momentum into the vertex) + sum_c J[a][c] ^ J[c][M] (contact)
        ften<R> F = fzero<R>();
        wedge_acc(F, cast<R>(P[a][M]), J[a][M]);
#pragma unroll
        for (int c = a + 1; c < M; ++c) wedge_acc(F, J[a][c], J[c][M]);
#pragma unroll
        for (int p = 0; p < NPASS; ++p) {
          spinor<R> t0 = row_slash(U[p][a].o0, J[a][M]);
#pragma unroll
          for (int i = 0; i < 4; ++i) b0[p].c[i] += mul_i(t0.c[i]);
          if (a > 0) {                                   // U[.][0] has no order-1 part
            spinor<R> t1 = row_slash(U[p][a].o1, J[a][M]);
#pragma unroll
            for (int i = 0; i < 4; ++i) b1[p].c[i] += mul_i(t1.c[i]);
          }
          row_sigma_acc(b1[p], U[p][a].o0, F);
        }
      }
      if constexpr (M < N) {
        rvec4<double> qd = rsub(pt, P[0][M]);
        const double q2 = rdot(qd, qd);
        rvec4<R> q = cast<R>(qd);
#pragma unroll
        for (int p = 0; p < NPASS; ++p) {
          // S(q) = i (qslash + m) / (q^2 - m^2 + i m Gamma)
          cx<double> den(q2 - line[p].mt * line[p].mt, line[p].mGt);
          cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
          spinor<R> s0 = row_slash(b0[p], q), s1 = row_slash(b1[p], q);
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            cx<R> n0 = s0.c[i]; cfma(n0, b0[p].c[i], R(line[p].mt));
            cx<R> n1 = s1.c[i]; cfma(n1, b1[p].c[i], R(line[p].mt));
            U[p][M].o0.c[i] = n0 * pr; U[p][M].o1.c[i] = n1 * pr;
          }
        }
        level<(M < N ? M + 1 : N)>(used | (1u << g));
      } else {
        (*sink)(leaf, b0, b1);
        ++leaf;
      }
    }
  }

  TREX_HD void run(Sink* s) {
    sink = s; leaf = 0;
#pragma unroll
    for (int p = 0; p < NPASS; ++p) { U[p][0].o0 = ubar_t; U[p][0].o1 = szero<R>(); }
    level<1>(0u);
  }
};

// ---------------------------------------------------------------- fully static variant (N <= 3)
// The same walk with every gluon index, ordering prefix and leaf rank a template parameter: K[], eps[], J[][], U[][]
// and the sink's amplitude array are only ever indexed by compile-time constants, so the whole state lives in registers
// (the dynamic version above keeps it in local memory). One instantiation per tree node: 4 (N = 2), 15 (N = 3).
// Sink interface: template <int LEAF> void put(const spinor<R>* b0, const spinor<R>* b1).
template <class R, int N, int NPASS, class Sink> struct TTNGS {
  rvec4<double> K[N];
  vec4<R> eps[N];
  rvec4<double> pt;
  spinor<R> ubar_t;
  TopLine line[NPASS];
  vec4<R> J[N][N + 1];
  rvec4<double> P[N][N + 1];
  dspinor<R> U[NPASS][N];
  Sink* sink;

  TREX_HD static constexpr int fact(int n) { return n <= 1 ? 1 : n * fact(n - 1); }
  TREX_HD static constexpr int rank_unused(unsigned used, int g) { int r = 0; for (int m = 0; m < g; ++m) r += !((used >> m) & 1u); return r; }

  template <int M, unsigned USED, int LB, int G> TREX_HD void visit() {
    if constexpr (G < N) {
      if constexpr (!((USED >> G) & 1u)) body<M, USED, LB + rank_unused(USED, G) * fact(N - M), G>();
      visit<M, USED, LB, G + 1>();
    }
  }

  template <int M, unsigned USED, int LB, int G> TREX_HD void body() {
    J[M - 1][M] = eps[G];
    P[M - 1][M] = K[G];
#pragma unroll
    for (int a = M - 2; a >= 0; --a) {
      P[a][M] = radd(P[a][M - 1], K[G]);
      vec4<R> acc = vzero<R>();
#pragma unroll
      for (int c = a + 1; c < M; ++c) v3_acc(acc, P[a][c], J[a][c], P[c][M], J[c][M]);
#pragma unroll
      for (int c1 = a + 1; c1 < M; ++c1)
#pragma unroll
        for (int c2 = c1 + 1; c2 < M; ++c2) v4_acc(acc, J[a][c1], J[c1][c2], J[c2][M]);
      const R sc = R(-1.0 / rdot(P[a][M], P[a][M]));
#pragma unroll
      for (int i = 0; i < 4; ++i) J[a][M].c[i] = acc.c[i] * sc;
    }
    spinor<R> b0[NPASS], b1[NPASS];
#pragma unroll
    for (int p = 0; p < NPASS; ++p) { b0[p] = szero<R>(); b1[p] = szero<R>(); }
#pragma unroll
    for (int a = 0; a < M; ++a) {
      ften<R> F = fzero<R>();
      wedge_acc(F, cast<R>(P[a][M]), J[a][M]);
#pragma unroll
      for (int c = a + 1; c < M; ++c) wedge_acc(F, J[a][c], J[c][M]);
#pragma unroll
      for (int p = 0; p < NPASS; ++p) {
        const spinor<R> t0 = row_slash(U[p][a].o0, J[a][M]);
#pragma unroll
        for (int i = 0; i < 4; ++i) b0[p].c[i] += mul_i(t0.c[i]);
        if (a > 0) {
          const spinor<R> t1 = row_slash(U[p][a].o1, J[a][M]);
#pragma unroll
          for (int i = 0; i < 4; ++i) b1[p].c[i] += mul_i(t1.c[i]);
        }
        row_sigma_acc(b1[p], U[p][a].o0, F);
      }
    }
    if constexpr (M < N) {
      const rvec4<double> qd = rsub(pt, P[0][M]);
      const double q2 = rdot(qd, qd);
      const rvec4<R> q = cast<R>(qd);
#pragma unroll
      for (int p = 0; p < NPASS; ++p) {
        const cx<double> den(q2 - line[p].mt * line[p].mt, line[p].mGt);
        const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
        const spinor<R> s0 = row_slash(b0[p], q), s1 = row_slash(b1[p], q);
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          cx<R> n0 = s0.c[i]; cfma(n0, b0[p].c[i], R(line[p].mt));
          cx<R> n1 = s1.c[i]; cfma(n1, b1[p].c[i], R(line[p].mt));
          U[p][M].o0.c[i] = n0 * pr; U[p][M].o1.c[i] = n1 * pr;
        }
      }
      visit<(M < N ? M + 1 : N), (USED | (1u << G)), LB, 0>();
    } else {
      sink->template put<LB>(b0, b1);
    }
  }

  TREX_HD void run(Sink* s) {
    sink = s;
#pragma unroll
    for (int p = 0; p < NPASS; ++p) { U[p][0].o0 = ubar_t; U[p][0].o1 = szero<R>(); }
    visit<1, 0u, 0, 0>();
  }
};

}  // namespace trex
