// trex_memo.cuh -- g g -> t t~ + (N-2) g with a per-event table of off-shell gluon currents.
//
// The prefix walk of trex_ttng.cuh re-derives the current J(s_a+1 .. s_M) of a contiguous gluon tuple under every
// prefix and for every helicity of the gluons OUTSIDE the tuple, and keeps N(N+1)/2 currents per thread alive. Here a
// thread block owns one event and builds, level by level in shared memory, the table of ALL ordered-tuple currents
//     J(t_1 .. t_k ; helicities of t_1 .. t_k),   k = 1 .. N,
// once ("helicity recycling": a current depends only on the helicities of its own gluons), using the reflection
// identity J(t_k .. t_1) = (-1)^(k+1) J(t_1 .. t_k) to evaluate and store only tuples with t_1 < t_k:
//     N = 5: 10 + 40 + 240 + 960 + 1920 entries of 4 complex numbers  (instead of 980 currents per helicity unit).
// The top-quark line is then walked depth first by one thread per (gluon helicities, top helicity, first gluon,
// parameter point): its private state is the line spinors U[1..N-1] only; every current is a table lookup. The warps
// of the walk are uniform in the ordering prefix (lanes differ in helicities only), so there is no divergence, and the
// table is component-major ([re/im x mu][entry]) so that lanes reading entries that differ in helicity bits hit
// distinct banks and lanes reading the same entry broadcast.
// Colour-flow amplitudes x_sigma (theta_old, theta_new; both antitop helicities) go to a scratch matrix
// X[event][column = (h, lambda_t, lambda_tbar, theta)][sigma]; the colour sum J^dagger C J, the helicity sum and the
// epilogue run in a second kernel (trex_memo_tu.cu) that stages X tiles and C in shared memory.
#pragma once
#include "trex_math.cuh"
#include "trex_ttng.cuh"

namespace trex {

template <int N> struct MemoIdx {
  // f(n, k) = n! / (n-k)!
  TREX_HD static constexpr int falling(int n, int k) { int r = 1; for (int i = 0; i < k; ++i) r *= (n - i); return r; }
  TREX_HD static constexpr int ncanon(int k) { return k == 1 ? N : falling(N, k) / 2; }
  TREX_HD static constexpr int base(int k) { int b = 0; for (int j = 1; j < k; ++j) b += ncanon(j) << j; return b; }
  static constexpr int NE = base(N + 1);          // entries of all levels 1..N
  static constexpr int NSET = 1 << N;

  // canonical id of an ordered k-tuple with t[0] < t[k-1] (k >= 2): (pair {first,last}) x (rank of the middle)
  template <int K> TREX_HD static int canon_id(const int* t) {
    const int a = t[0], b = t[K - 1];
    int id = a * (2 * N - a - 1) / 2 + (b - a - 1);
    unsigned used = (1u << a) | (1u << b);
    int mid = 0;
#pragma unroll
    for (int i = 1; i < K - 1; ++i) {
      const int m = t[i];
      const int c = m - __builtin_popcount(used & ((1u << m) - 1u));
      mid = mid * (N - 1 - i) + c;              // mixed radix: N-2, N-3, ...
      used |= 1u << m;
    }
    return id * falling(N - 2, K - 2) + mid;
  }
  // inverse of canon_id
  template <int K> TREX_HD static void canon_tuple(int id, int* t) {
    constexpr int nmid = falling(N - 2, K - 2);
    int pair = id / nmid, mid = id - pair * nmid;
    int a = 0;
    while (pair >= N - 1 - a) { pair -= N - 1 - a; ++a; }
    const int b = a + 1 + pair;
    t[0] = a; t[K - 1] = b;
    unsigned used = (1u << a) | (1u << b);
    int digit[K > 2 ? K - 2 : 1];
#pragma unroll
    for (int i = K - 2; i >= 1; --i) { const int radix = N - 1 - i; digit[i - 1] = mid % radix; mid /= radix; }
#pragma unroll
    for (int i = 1; i < K - 1; ++i) {
      int c = digit[i - 1], m = 0;
      for (;; ++m) { if (!((used >> m) & 1u)) { if (c == 0) break; --c; } }
      t[i] = m; used |= 1u << m;
    }
  }
  TREX_HD static unsigned bitrev(unsigned bits, int k) {
    unsigned r = 0;
    for (int i = 0; i < k; ++i) r |= ((bits >> i) & 1u) << (k - 1 - i);
    return r;
  }
};

// table access: entry index and sign of J(t_0 .. t_{K-1}) with position-ordered helicity bits
template <int N, int K> TREX_HD int memo_entry(const int* t, unsigned bits, int& sign) {
  using I = MemoIdx<N>;
  if constexpr (K == 1) { sign = 1; return t[0] * 2 + (int)bits; }
  else {
    const bool fwd = t[0] < t[K - 1];
    int tt[K];
#pragma unroll
    for (int i = 0; i < K; ++i) tt[i] = fwd ? t[i] : t[K - 1 - i];
    const unsigned bb = fwd ? bits : I::bitrev(bits, K);
    sign = (fwd || (K & 1)) ? 1 : -1;            // reversed: (-1)^(K+1)
    return I::base(K) + (I::template canon_id<K>(tt) << K) + (int)bb;
  }
}
template <class R, int N, int K> TREX_HD vec4<R> memo_fetch(const R* __restrict__ tab, const int* t, unsigned bits) {
  int sign;
  const int e = memo_entry<N, K>(t, bits, sign);
  const R s = R(sign);
  vec4<R> J;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) J.c[mu] = cx<R>(s * tab[(2 * mu) * MemoIdx<N>::NE + e], s * tab[(2 * mu + 1) * MemoIdx<N>::NE + e]);
  return J;
}
template <class R, int N> TREX_HD void memo_store(R* __restrict__ tab, int e, const vec4<R>& J) {
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) { tab[(2 * mu) * MemoIdx<N>::NE + e] = J.c[mu].re; tab[(2 * mu + 1) * MemoIdx<N>::NE + e] = J.c[mu].im; }
}
template <int K> TREX_HD unsigned tuple_mask(const int* t) {
  unsigned m = 0;
#pragma unroll
  for (int i = 0; i < K; ++i) m |= 1u << t[i];
  return m;
}

// static dispatch helpers: J of the sub-tuple t[A .. A+L) of a K-tuple with bits `bits`
template <class R, int N, int L> TREX_HD vec4<R> memo_sub(const R* __restrict__ tab, const int* t, int a, unsigned bits) {
  return memo_fetch<R, N, L>(tab, t + a, (bits >> a) & ((1u << L) - 1u));
}

// ---- phase 1: one table entry of level K >= 2 (item = canonical id x helicity bits)
template <class R, int N, int K, int J1 = 1>
TREX_HD void memo_v3_splits(vec4<R>& acc, const R* __restrict__ tab, const rvec4<double>* __restrict__ pset, const int* t, unsigned bits) {
  if constexpr (J1 < K) {
    vec4<R> JL = memo_sub<R, N, J1>(tab, t, 0, bits), JR = memo_sub<R, N, K - J1>(tab, t, J1, bits);
    v3_acc(acc, pset[tuple_mask<J1>(t)], JL, pset[tuple_mask<K - J1>(t + J1)], JR);
    memo_v3_splits<R, N, K, J1 + 1>(acc, tab, pset, t, bits);
  }
}
template <class R, int N, int K, int J1 = 1, int J2 = 2>
TREX_HD void memo_v4_splits(vec4<R>& acc, const R* __restrict__ tab, const int* t, unsigned bits) {
  if constexpr (J2 < K) {
    vec4<R> A = memo_sub<R, N, J1>(tab, t, 0, bits), B = memo_sub<R, N, J2 - J1>(tab, t, J1, bits), C = memo_sub<R, N, K - J2>(tab, t, J2, bits);
    v4_acc(acc, A, B, C);
    if constexpr (J2 + 1 < K) memo_v4_splits<R, N, K, J1, J2 + 1>(acc, tab, t, bits);
    else if constexpr (J1 + 2 < K) memo_v4_splits<R, N, K, J1 + 1, J1 + 2>(acc, tab, t, bits);
  }
}
template <class R, int N, int K>
TREX_HD void memo_build_item(R* __restrict__ tab, const rvec4<double>* __restrict__ pset, int item) {
  using I = MemoIdx<N>;
  const int cid = item >> K;
  const unsigned bits = (unsigned)item & ((1u << K) - 1u);
  int t[K];
  I::template canon_tuple<K>(cid, t);
  vec4<R> acc = vzero<R>();
  memo_v3_splits<R, N, K>(acc, tab, pset, t, bits);
  memo_v4_splits<R, N, K>(acc, tab, t, bits);
  const rvec4<double>& P = pset[tuple_mask<K>(t)];
  // (-i/P^2) [(-i) V3 + (-i) V4] at g_s = 1; for K == N the propagator is that of the gluon feeding the t t~ line
  const R s = R(-1.0 / rdot(P, P));
  vec4<R> J;
#pragma unroll
  for (int i = 0; i < 4; ++i) J.c[i] = acc.c[i] * s;
  memo_store<R, N>(tab, I::base(K) + item, J);
}

// ---- phase 2: depth-first walk of the top line below a fixed first gluon, currents from the table
template <class R, int N, class Sink> struct TopWalk {
  const R* tab;                       // current table of this event
  const rvec4<double>* pset;          // momentum of every gluon subset (incoming convention)
  rvec4<double> pt;
  spinor<R> ubar_t;
  TopLine line;
  unsigned h;                         // physical gluon helicity bits (bit g = helicity of gluon g)
  int s[N];                           // ordering prefix
  unsigned pathbits;                  // helicity of s[i] at bit i
  unsigned prefmask[N + 1];           // gluons in s[0..m)
  dspinor<R> U[N];                    // U[m], m = 1..N-1 (U[0] = ubar_t, order 1 = 0)
  int leaf;
  Sink* sink;

  template <int M, int A> TREX_HD void bracket_terms(spinor<R>& b0, spinor<R>& b1, vec4<R>* Jend) {
    if constexpr (A < M) {
      // F = P ^ J (dipole) + sum_c J(s[A..c)) ^ J(s[c..M)) (contact)
      ften<R> F = fzero<R>();
      wedge_acc(F, cast<R>(pset[prefmask[M] ^ prefmask[A]]), Jend[A]);
      contact_terms<M, A, A + 1>(F, Jend);
      const spinor<R>& u0 = A == 0 ? ubar_t : U[A].o0;
      spinor<R> t0 = row_slash(u0, Jend[A]);
#pragma unroll
      for (int i = 0; i < 4; ++i) b0.c[i] += mul_i(t0.c[i]);
      if constexpr (A > 0) {
        spinor<R> t1 = row_slash(U[A].o1, Jend[A]);
#pragma unroll
        for (int i = 0; i < 4; ++i) b1.c[i] += mul_i(t1.c[i]);
      }
      row_sigma_acc(b1, u0, F);
      bracket_terms<M, A + 1>(b0, b1, Jend);
    }
  }
  template <int M, int A, int C> TREX_HD void contact_terms(ften<R>& F, const vec4<R>* Jend) {
    if constexpr (C < M) {
      vec4<R> JL = memo_fetch<R, N, C - A>(tab, s + A, (pathbits >> A) & ((1u << (C - A)) - 1u));
      wedge_acc(F, JL, Jend[C]);
      contact_terms<M, A, C + 1>(F, Jend);
    }
  }
  template <int M, int A> TREX_HD void fetch_ends(vec4<R>* Jend) {
    if constexpr (A < M) {
      Jend[A] = memo_fetch<R, N, M - A>(tab, s + A, pathbits >> A);
      fetch_ends<M, A + 1>(Jend);
    }
  }

  template <int M> TREX_HD void node(int g) {
    s[M - 1] = g;
    pathbits = (pathbits & ((1u << (M - 1)) - 1u)) | (((h >> g) & 1u) << (M - 1));
    prefmask[M] = prefmask[M - 1] | (1u << g);
    vec4<R> Jend[M];                                   // J(s[a..M)), a = 0..M-1
    fetch_ends<M, 0>(Jend);
    spinor<R> b0 = szero<R>(), b1 = szero<R>();
    bracket_terms<M, 0>(b0, b1, Jend);
    if constexpr (M < N) {
      rvec4<double> qd = rsub(pt, pset[prefmask[M]]);
      const double q2 = rdot(qd, qd);
      rvec4<R> q = cast<R>(qd);
      cx<double> den(q2 - line.mt * line.mt, line.mGt);
      cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
      spinor<R> s0 = row_slash(b0, q), s1 = row_slash(b1, q);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        cx<R> n0 = s0.c[i]; cfma(n0, b0.c[i], R(line.mt));
        cx<R> n1 = s1.c[i]; cfma(n1, b1.c[i], R(line.mt));
        U[M].o0.c[i] = n0 * pr; U[M].o1.c[i] = n1 * pr;
      }
      for (int g2 = 0; g2 < N; ++g2) {
        if ((prefmask[M] >> g2) & 1u) continue;
        node<(M < N ? M + 1 : N)>(g2);
      }
    } else {
      (*sink)(leaf, b0, b1);
      ++leaf;
    }
  }

  TREX_HD void run(int g1, Sink* sk) {
    sink = sk; leaf = 0; pathbits = 0; prefmask[0] = 0;
    node<1>(g1);
  }
};

// ---- per-event set-up: momentum of every gluon subset and the level-1 entries (polarisation vectors)
template <int N> TREX_HD void memo_pset_item(const double* __restrict__ mom, long ld, long e, unsigned set, rvec4<double>* __restrict__ pset) {
  rvec4<double> P;
  for (int mu = 0; mu < 4; ++mu) P.c[mu] = 0.0;
  for (int g = 0; g < N; ++g) {
    if (!((set >> g) & 1u)) continue;
    const int leg = g < 2 ? g : g + 2;
    const double sg = g < 2 ? 1.0 : -1.0;
    for (int mu = 0; mu < 4; ++mu) P.c[mu] += sg * mom[(long)(leg * 4 + mu) * ld + e];
  }
  pset[set] = P;
}
template <class R, int N> TREX_HD void memo_level1_item(const double* __restrict__ mom, long ld, long e, int item, R* __restrict__ tab) {
  const int g = item >> 1, lam = (item & 1) ? 1 : -1;
  const int leg = g < 2 ? g : g + 2;
  double p[4];
  for (int mu = 0; mu < 4; ++mu) p[mu] = mom[(long)(leg * 4 + mu) * ld + e];
  memo_store<R, N>(tab, item, cast<R>(polvec<double>(p, lam, g >= 2)));
}

// ---- leaf sink of the walk: x_sigma = A0 + (kappa/g_s) A1 for both antitop helicities -> X[col][sigma] (re, im)
template <class R, int N> struct MemoLeafStore {
  double* X;                 // this event's [ncols][NC][2]
  int colbase;               // ((h * 2 + lt) * 2 + iv) * 2 + theta  with iv = theta = 0
  int leaf0;                 // rank of the first ordering of this task's subtree
  int th_lo, th_hi;          // parameter points this task writes
  spinor<R> v[2];
  R kq[2];
  TREX_HD void operator()(int leaf, const spinor<R>& b0, const spinor<R>& b1) {
    constexpr int NC = MemoIdx<N>::falling(N, N);
#pragma unroll
    for (int iv = 0; iv < 2; ++iv) {
      const cx<R> a0 = row_col(b0, v[iv]), a1 = row_col(b1, v[iv]);
      for (int th = th_lo; th < th_hi; ++th) {
        cx<R> x = a0; cfma(x, a1, kq[th]);
        double* dst = X + ((long)(colbase + iv * 2 + th) * NC + leaf0 + leaf) * 2;
        dst[0] = (double)x.re; dst[1] = (double)x.im;
      }
    }
  }
};

// one walk task: (gluon helicities h, top helicity, first gluon g1, parameter point `pass` of `npass`)
template <class R, int N>
TREX_HD void memo_walk_task(const R* __restrict__ tab, const rvec4<double>* __restrict__ pset, const double* __restrict__ mom, long ld, long e,
                            const double mt[2], const double mGt[2], const double kq[2], unsigned h, int lt, int g1, int pass, int npass,
                            double* __restrict__ Xev) {
  using Store = MemoLeafStore<R, N>;
  Store st;
  TopWalk<R, N, Store> w;
  double p[4], q[4];
  for (int mu = 0; mu < 4; ++mu) { p[mu] = mom[(long)(2 * 4 + mu) * ld + e]; q[mu] = mom[(long)(3 * 4 + mu) * ld + e]; w.pt.c[mu] = p[mu]; }
  w.ubar_t = cast<R>(bar(spinor_u<double>(p, lt ? 1 : -1, false)));
  st.v[0] = cast<R>(spinor_v<double>(q, -1, false));
  st.v[1] = cast<R>(spinor_v<double>(q, +1, false));
  st.kq[0] = R(kq[0]); st.kq[1] = R(kq[1]);
  st.X = Xev;
  st.colbase = (int)((h * 2 + (unsigned)lt) * 4);
  st.leaf0 = g1 * MemoIdx<N>::falling(N - 1, N - 1);
  st.th_lo = npass == 1 ? 0 : pass; st.th_hi = npass == 1 ? 2 : pass + 1;
  w.tab = tab; w.pset = pset; w.h = h;
  w.line.mt = mt[pass]; w.line.mGt = mGt[pass];
  w.run(g1, &st);
}

}  // namespace trex
