// trex_table.cuh -- g g -> t t~ + (N-2) g from a per-event table of off-shell gluon currents.
//
// A thread block owns one event. The colour-ordered recursion of SURVEY.md C-4 needs, for every ordering sigma and every
// helicity configuration, the current J(t_1 .. t_k) of every contiguous gluon tuple and, at order kappa, the
// field-strength bracket   F(t_1 .. t_k) = P ^ J(t_1 .. t_k) + sum_c J(t_1 .. t_c) ^ J(t_c+1 .. t_k)
// (dipole + contact insertions on the top line, R-4). Both depend only on the tuple and on the helicities of
// ITS OWN gluons ("helicity recycling"), and J(t_k .. t_1) = (-1)^(k+1) J(t_1 .. t_k), same for F. So the block builds,
// level by level in shared memory, one table entry (J: 4 complex, 2 sigma.F as two 2x2 blocks: 6 complex) per
// canonical tuple (t_1 < t_k) and helicity assignment, and the top-quark line is then walked depth first by one thread
// per (ordering prefix, free helicities, top helicity [, parameter point]): every vertex on the line is two row-spinor x
// slash products and one row-spinor x sigma.F product with operands fetched from the table.
//
// To make the table, the colour-flow amplitudes X and the colour matrix fit the 227 KB of one SM for N = 5, the
// helicities of the first NFIX gluons are fixed by an outer loop of 2^NFIX iterations: the table of one iteration only
// holds the helicity assignments of the remaining ("free") gluons; X holds the columns (free helicities, lambda_t,
// lambda_tbar, theta) of that iteration and is closed with J^dagger C J before the next iteration starts.
#pragma once
#include "trex_math.cuh"
#include "trex_ttng.cuh"

namespace trex {

// ---------------------------------------------------------------- indexing of canonical tuples and table entries
template <int N, int NFIX> struct TabIdx {
  TREX_HD static constexpr int falling(int n, int k) { int r = 1; for (int i = 0; i < k; ++i) r *= (n - i); return r; }
  TREX_HD static constexpr int binom(int n, int k) { if (k < 0 || k > n) return 0; int r = 1; for (int i = 0; i < k; ++i) r = r * (n - i) / (i + 1); return r; }
  TREX_HD static constexpr int ncanon(int k) { return k == 1 ? N : falling(N, k) / 2; }       // canonical k-tuples
  TREX_HD static constexpr int cid_base(int k) { int b = 0; for (int j = 1; j < k; ++j) b += ncanon(j); return b; }
  static constexpr int NCID = cid_base(N + 1);
  static constexpr int NFREE = N - NFIX;
  // entries of level k: sum over canonical k-tuples of 2^(free gluons in the tuple)
  TREX_HD static constexpr int level_entries(int k) {
    int s = 0;
    for (int f = 0; f <= k; ++f) s += binom(NFIX, f) * binom(NFREE, k - f) * falling(k, k) * (1 << (k - f));
    return k == 1 ? s : s / 2;
  }
  TREX_HD static constexpr int entries_below(int k) { int s = 0; for (int j = 1; j < k; ++j) s += level_entries(j); return s; }
  static constexpr int NE = entries_below(N + 1);

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
  // inverse of canon_id (host side: the tuples are shipped to the kernel in the meta block)
  static void canon_tuple(int K, int id, int* t) {
    const int nmid = falling(N - 2, K - 2);
    int pair = id / nmid, mid = id - pair * nmid;
    int a = 0;
    while (pair >= N - 1 - a) { pair -= N - 1 - a; ++a; }
    const int b = a + 1 + pair;
    t[0] = a; t[K - 1] = b;
    unsigned used = (1u << a) | (1u << b);
    int digit[8];
    for (int i = K - 2; i >= 1; --i) { const int radix = N - 1 - i; digit[i - 1] = mid % radix; mid /= radix; }
    for (int i = 1; i < K - 1; ++i) {
      int c = digit[i - 1], m = 0;
      for (;; ++m) { if (!((used >> m) & 1u)) { if (c == 0) break; --c; } }
      t[i] = m; used |= 1u << m;
    }
  }
  TREX_HD static unsigned bitrev(unsigned bits, int k) {           // reverse the low k bits (bits above k are zero)
#if defined(__CUDA_ARCH__)
    return (__brev(bits) >> 1) >> (31 - k);
#else
    unsigned r = 0;
    for (int i = 0; i < k; ++i) r |= ((bits >> i) & 1u) << (k - 1 - i);
    return r;
#endif
  }
  // the r-th (r = 0, 1, ..) gluon not in `used`
  TREX_HD static int nth_unused(unsigned used, int r) {
    int g = 0, c = r;
#pragma unroll
    for (int m = 0; m < N; ++m) {
      const bool freeslot = !((used >> m) & 1u);
      if (freeslot && c == 0) g = m;
      if (freeslot) --c;
    }
    return g;
  }
  // meta block (ints), built once on the host: entry offset of every canonical tuple, first entry of every level,
  // the tuples themselves (4 bits per position) and the canonical tuple of every entry
  static constexpr int M_OFF = 0;                  // [NCID + 1]
  static constexpr int M_LVL = M_OFF + NCID + 1;   // [N + 2]: index K = first entry of level K, K = 1 .. N+1
  static constexpr int M_TUP = M_LVL + N + 2;      // [NCID]
  static constexpr int M_CID = M_TUP + NCID;       // [NE]
  // walk recipes (N <= 4, all helicities free): per ordering, in lexicographic order, four ints = the table references
  // of the seven tuples a walk task touches, 16 bits each: entry offset of the canonical tuple (bits 0-8), tuple is
  // reversed (bit 9: helicity bits are bit-reversed), sign -1 (bit 10); then the ordering itself and the rank of
  // (s1, s2) among ordered pairs:  w0 = (s1 s2 s3) | (s2 s3) << 16,  w1 = (s3) | (s1 s2 s3 s4) << 16,
  // w2 = (s2 s3 s4) | (s3 s4) << 16,  w3 = (s4) | (s1 | s2 << 2 | s3 << 4 | s4 << 6 | pair << 8) << 16
  static constexpr int M_REC = (M_CID + NE + 3) / 4 * 4;
  static constexpr int NREC = (N == 4 && NFIX == 0) ? 4 * 24 : 0;
  static constexpr int M_SIZE = M_REC + NREC;
  static int host_ref(const int* meta, const int* t, int L) {
    const bool fwd = L == 1 || t[0] < t[L - 1];
    int tt[8];
    for (int i = 0; i < L; ++i) tt[i] = fwd ? t[i] : t[L - 1 - i];
    int cid = tt[0];
    if (L == 2) cid = cid_base(2) + canon_id<2>(tt);
    if (L == 3) cid = cid_base(3) + canon_id<3>(tt);
    if (L == 4) cid = cid_base(4) + canon_id<4>(tt);
    return meta[M_OFF + cid] | (fwd ? 0 : 0x200) | ((fwd || (L & 1)) ? 0 : 0x400);
  }
  static void build_meta(int* meta) {
    int e = 0, cid = 0;
    for (int K = 1; K <= N; ++K) {
      meta[M_LVL + K] = e;
      for (int id = 0; id < ncanon(K); ++id, ++cid) {
        int t[8];
        if (K == 1) t[0] = id; else canon_tuple(K, id, t);
        int nf = 0, packed = 0;
        for (int i = 0; i < K; ++i) { nf += t[i] >= NFIX; packed |= t[i] << (4 * i); }
        meta[M_OFF + cid] = e;
        meta[M_TUP + cid] = packed;
        for (int b = 0; b < (1 << nf); ++b) meta[M_CID + e++] = cid;
      }
    }
    meta[M_OFF + cid] = e;
    meta[M_LVL + N + 1] = e;
    meta[M_LVL] = 0;
    if constexpr (NREC > 0) {
      int rank = 0;
      for (int s1 = 0; s1 < 4; ++s1) for (int s2 = 0; s2 < 4; ++s2) for (int s3 = 0; s3 < 4; ++s3) for (int s4 = 0; s4 < 4; ++s4) {
        if (s1 == s2 || s1 == s3 || s1 == s4 || s2 == s3 || s2 == s4 || s3 == s4) continue;
        const int s[4] = {s1, s2, s3, s4};
        int* w = meta + M_REC + 4 * rank++;
        w[0] = host_ref(meta, s, 3) | host_ref(meta, s + 1, 2) << 16;
        w[1] = host_ref(meta, s + 2, 1) | host_ref(meta, s, 4) << 16;
        w[2] = host_ref(meta, s + 1, 3) | host_ref(meta, s + 2, 2) << 16;
        const int pair = s1 * 3 + s2 - (s2 > s1 ? 1 : 0);
        w[3] = host_ref(meta, s + 3, 1) | (s1 | s2 << 2 | s3 << 4 | s4 << 6 | pair << 8) << 16;
      }
    }
  }
};

// ---------------------------------------------------------------- table access
// 10 complex components per entry, component-major: tab[comp * NE + entry] (re, im adjacent); comp 0..3 = J^mu,
// 4..9 = -i * 2 sigma.F in the form the row-spinor product consumes: with X+- = 2 (B +- iE) (the two chiral 2x2 blocks
// are X+.s and X-.s) the entries are -i (X+_3, X+_1 + i X+_2, X+_1 - i X+_2, X-_3, X-_1 + i X-_2, X-_1 - i X-_2).
// The factor -i lets the walk accumulate  sum_a [U_a Jslash_a - i U_a sigma.F_a]  and multiply by i once per node.
constexpr int TAB_NCOMP = 20;

template <class R> struct sigF { cx<R> p3, pt, pb, m3, mt, mb; };

// entry index and sign of the ordered tuple t[0..L) whose free gluons carry the (position-ordered) bits `cbits`
template <int N, int NFIX, int L> TREX_HD int tab_entry(const int* __restrict__ off, const int* t, unsigned cbits, int nf, int& sign) {
  using I = TabIdx<N, NFIX>;
  if constexpr (L == 1) { sign = 1; return off[t[0]] + (int)cbits; }
  else {
    const bool fwd = t[0] < t[L - 1];
    int tt[L];
#pragma unroll
    for (int i = 0; i < L; ++i) tt[i] = fwd ? t[i] : t[L - 1 - i];
    const unsigned bb = fwd ? cbits : I::bitrev(cbits, nf);
    sign = (fwd || (L & 1)) ? 1 : -1;            // reversed: (-1)^(L+1)
    return off[I::cid_base(L) + I::template canon_id<L>(tt)] + (int)bb;
  }
}
// x or -x without touching the floating-point pipes (sign-bit flip on the integer pipe)
TREX_HD double with_sign(double x, int sign) {
#if defined(__CUDA_ARCH__)
  return __hiloint2double(__double2hiint(x) ^ (sign < 0 ? (int)0x80000000 : 0), __double2loint(x));
#else
  return sign < 0 ? -x : x;
#endif
}
TREX_HD float with_sign(float x, int sign) {
#if defined(__CUDA_ARCH__)
  return __int_as_float(__float_as_int(x) ^ (sign < 0 ? (int)0x80000000 : 0));
#else
  return sign < 0 ? -x : x;
#endif
}
// (re, im) of one table component travel together: one 16-byte (fp64) / 8-byte (fp32) shared-memory access
template <class R> struct pair_of;
template <> struct pair_of<double> { using type = double2; };
template <> struct pair_of<float> { using type = float2; };
template <class R> TREX_HD cx<R> tab_get(const R* __restrict__ tab, int idx, int sign) {
  using P = typename pair_of<R>::type;
  const P v = reinterpret_cast<const P*>(tab)[idx];
  return cx<R>(with_sign(v.x, sign), with_sign(v.y, sign));
}
template <class R> TREX_HD void tab_put(R* __restrict__ tab, int idx, cx<R> c) {
  using P = typename pair_of<R>::type;
  P v; v.x = c.re; v.y = c.im;
  reinterpret_cast<P*>(tab)[idx] = v;
}
template <class R, int NE> TREX_HD vec4<R> tab_J(const R* __restrict__ tab, int e, int sign) {
  vec4<R> J;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) J.c[mu] = tab_get<R>(tab, mu * NE + e, sign);
  return J;
}
template <class R, int NE> TREX_HD sigF<R> tab_F(const R* __restrict__ tab, int e, int sign) {
  sigF<R> F;
  cx<R>* f = &F.p3;
#pragma unroll
  for (int i = 0; i < 6; ++i) f[i] = tab_get<R>(tab, (4 + i) * NE + e, sign);
  return F;
}
// -i * 2 sigma.F as the two 2x2 blocks the row-spinor product consumes
template <class R> TREX_HD sigF<R> make_sigF(const ften<R>& f) {
  cx<R> xp[3], xm[3];
#pragma unroll
  for (int i = 0; i < 3; ++i) { const cx<R> ie = mul_i(f.e[i]); xp[i] = R(2) * (f.b[i] + ie); xm[i] = R(2) * (f.b[i] - ie); }
  sigF<R> F;
  F.p3 = mul_mi(xp[2]); F.pt = mul_mi(xp[0] + mul_i(xp[1])); F.pb = mul_mi(xp[0] - mul_i(xp[1]));
  F.m3 = mul_mi(xm[2]); F.mt = mul_mi(xm[0] + mul_i(xm[1])); F.mb = mul_mi(xm[0] - mul_i(xm[1]));
  return F;
}
template <class R, int NE> TREX_HD void tab_store(R* __restrict__ tab, int e, const vec4<R>& J, const sigF<R>& F) {
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) tab_put<R>(tab, mu * NE + e, J.c[mu]);
  const cx<R>* f = &F.p3;
#pragma unroll
  for (int i = 0; i < 6; ++i) tab_put<R>(tab, (4 + i) * NE + e, f[i]);
}
template <class R, int NE> TREX_HD void tab_store(R* __restrict__ tab, int e, const vec4<R>& J, const ften<R>& f) {
  tab_store<R, NE>(tab, e, J, make_sigF<R>(f));
}
// a -= b * c
template <class R> TREX_HD void cfnma(cx<R>& a, cx<R> b, cx<R> c) {
  a.re -= b.re * c.re; a.re += b.im * c.im; a.im -= b.re * c.im; a.im -= b.im * c.re; }
// acc += r * aslash   (pure FMA form of row_slash; the caller multiplies the sum by i once)
template <class R> TREX_HD void row_slash_acc(spinor<R>& acc, const spinor<R>& r, const vec4<R>& a) {
  const cx<R> ap = a.c[0] + a.c[3], am = a.c[0] - a.c[3];
  const cx<R> at = a.c[1] + mul_i(a.c[2]), ab = a.c[1] - mul_i(a.c[2]);
  cfma(acc.c[0], r.c[2], ap); cfma(acc.c[0], r.c[3], at);
  cfma(acc.c[1], r.c[2], ab); cfma(acc.c[1], r.c[3], am);
  cfma(acc.c[2], r.c[0], am); cfnma(acc.c[2], r.c[1], at);
  cfma(acc.c[3], r.c[1], ap); cfnma(acc.c[3], r.c[0], ab);
}
// acc += r * (-i 2 sigma.F) with the pre-combined blocks of the table
template <class R> TREX_HD void row_sigma_acc_x(spinor<R>& acc, const spinor<R>& r, const sigF<R>& F) {
  cfma(acc.c[0], r.c[0], F.p3); cfma(acc.c[0], r.c[1], F.pt);
  cfma(acc.c[1], r.c[0], F.pb); cfnma(acc.c[1], r.c[1], F.p3);
  cfma(acc.c[2], r.c[2], F.m3); cfma(acc.c[2], r.c[3], F.mt);
  cfma(acc.c[3], r.c[2], F.mb); cfnma(acc.c[3], r.c[3], F.m3);
}

// ---------------------------------------------------------------- phase 1: one table entry of level K >= 2
// t[0..K) canonical tuple, fpos[i] = free gluons among t[0..i), fb = helicity bits of the free gluons in position order
// TS: entries per table component; PL, poff: references to entries of level <= PL are shifted by poff (the pipelined
// N = 4 kernel keeps two copies of its lowest levels, one per event parity)
template <class R, int N, int NFIX, int K, int TS = TabIdx<N, NFIX>::NE, int PL = 0> struct TabBuild {
  using I = TabIdx<N, NFIX>;
  static constexpr int NE = TS, KK = K;
  const R* tab; const int* off; const rvec4<double>* pset;
  int t[K], fpos[K + 1]; unsigned fb;
  int poff = 0;

  template <int L> TREX_HD vec4<R> sub(int a) const {
    int sign;
    const int nf = fpos[a + L] - fpos[a];
    int e = tab_entry<N, NFIX, L>(off, t + a, (fb >> fpos[a]) & ((1u << nf) - 1u), nf, sign);
    if constexpr (L <= PL) e += poff;
    return tab_J<R, NE>(tab, e, sign);
  }
  template <int L> TREX_HD unsigned mask(int a) const {
    unsigned m = 0;
#pragma unroll
    for (int i = 0; i < L; ++i) m |= 1u << t[a + i];
    return m;
  }
  // splits (left | right) of the tuple: three-gluon vertex and the contact part of F
  template <int J1> TREX_HD void v3_splits(vec4<R>& acc, ften<R>& F) const {
    if constexpr (J1 < K) {
      const vec4<R> JL = sub<J1>(0), JR = sub<K - J1>(J1);
      v3_acc(acc, pset[mask<J1>(0)], JL, pset[mask<K - J1>(J1)], JR);
      wedge_acc(F, JL, JR);
      v3_splits<J1 + 1>(acc, F);
    }
  }
  template <int J1, int J2> TREX_HD void v4_splits(vec4<R>& acc) const {
    if constexpr (J2 < K) {
      const vec4<R> A = sub<J1>(0), B = sub<J2 - J1>(J1), C = sub<K - J2>(J2);
      v4_acc(acc, A, B, C);
      if constexpr (J2 + 1 < K) v4_splits<J1, J2 + 1>(acc);
      else if constexpr (J1 + 2 < K) v4_splits<J1 + 1, J1 + 2>(acc);
    }
  }
  TREX_HD void compute(vec4<R>& J, ften<R>& F) const {
    vec4<R> acc = vzero<R>();
    F = fzero<R>();
    v3_splits<1>(acc, F);
    v4_splits<1, 2>(acc);
    const rvec4<double>& P = pset[mask<K>(0)];
    // (-i/P^2) [(-i) V3 + (-i) V4] at g_s = 1; for K == N the propagator is that of the gluon feeding the t t~ line
    const R s = R(-1.0 / rdot(P, P));
#pragma unroll
    for (int i = 0; i < 4; ++i) J.c[i] = acc.c[i] * s;
    wedge_acc(F, cast<R>(P), J);
  }
  TREX_HD void run(R* tabw, int e) const {
    vec4<R> J; ften<R> F;
    compute(J, F);
    tab_store<R, NE>(tabw, e, J, F);
  }
};

template <class R, int N, int NFIX, int K, class B>
TREX_HD void tab_build_setup(B& b, const R* __restrict__ tab, const int* __restrict__ meta, const rvec4<double>* __restrict__ pset, int e) {
  using I = TabIdx<N, NFIX>;
  b.tab = tab; b.off = meta + I::M_OFF; b.pset = pset;
  const int cid = meta[I::M_CID + e];
  const int packed = meta[I::M_TUP + cid];
  b.fb = (unsigned)(e - meta[I::M_OFF + cid]);
  b.fpos[0] = 0;
#pragma unroll
  for (int i = 0; i < K; ++i) { b.t[i] = (packed >> (4 * i)) & 15; b.fpos[i + 1] = b.fpos[i] + (b.t[i] >= NFIX ? 1 : 0); }
}
template <class R, int N, int NFIX, int K>
TREX_HD void tab_build_entry(R* __restrict__ tab, const int* __restrict__ meta, const rvec4<double>* __restrict__ pset, int e) {
  TabBuild<R, N, NFIX, K> b;
  tab_build_setup<R, N, NFIX, K>(b, tab, meta, pset, e);
  b.run(tab, e);
}
// level 1: J = polarisation vector, F = K ^ eps.  eps_all[(g * 2 + lambda) * 8 + (re, im per mu)]
template <class R, int N, int NFIX>
TREX_HD void tab_build_level1(R* __restrict__ tab, const int* __restrict__ meta, const rvec4<double>* __restrict__ pset,
                              const double* __restrict__ eps_all, unsigned itbits, int e) {
  using I = TabIdx<N, NFIX>;
  const int g = meta[I::M_CID + e];
  const int lam = g < NFIX ? (int)((itbits >> g) & 1u) : e - meta[I::M_OFF + g];
  vec4<R> J;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) J.c[mu] = cx<R>(R(eps_all[(g * 2 + lam) * 8 + 2 * mu]), R(eps_all[(g * 2 + lam) * 8 + 2 * mu + 1]));
  ften<R> F = fzero<R>();
  wedge_acc(F, cast<R>(pset[1u << g]), J);
  tab_store<R, I::NE>(tab, e, J, F);
}
// the same, handing J and F back (W-form kernels contract them further)
template <class R, int N, int NFIX>
TREX_HD void tab_level1_JF(const int* __restrict__ meta, const rvec4<double>* __restrict__ pset, const double* __restrict__ eps_all,
                           unsigned itbits, int e, vec4<R>& J, ften<R>& F) {
  using I = TabIdx<N, NFIX>;
  const int g = meta[I::M_CID + e];
  const int lam = g < NFIX ? (int)((itbits >> g) & 1u) : e - meta[I::M_OFF + g];
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) J.c[mu] = cx<R>(R(eps_all[(g * 2 + lam) * 8 + 2 * mu]), R(eps_all[(g * 2 + lam) * 8 + 2 * mu + 1]));
  F = fzero<R>();
  wedge_acc(F, cast<R>(pset[1u << g]), J);
}

// ---------------------------------------------------------------- suffix contractions ("W form", N = 4)
// The last vertex of an ordering closes the line with v(p_tbar): for a table entry e (the gluon tuple that ends the
// ordering) the column spinors   Wj_e = i Jslash_e v,   Wf_e = i (-i 2 sigma.F_e) v   do not depend on the rest of the
// ordering, so the leaf amplitude is a sum of row x column products  U_A . W_e  (12 complex multiply-adds per term and
// antitop helicity) instead of a row x matrix product per term followed by the closing. With U_0 = ubar(p_t) the A = 0
// term is the entry's own scalar  S_e = ubar W_e; likewise the A = 0 row of an inner node, ubar Gamma(J_e), is tabulated.
// (M v) for M = -i 2 sigma.F in the block form of row_sigma_acc_x: (r M)_0 = r0 p3 + r1 pt, (r M)_1 = r0 pb - r1 p3, ...
template <class R> TREX_HD spinor<R> sig_col(const sigF<R>& F, const spinor<R>& v) {
  spinor<R> o;
  o.c[0] = F.p3 * v.c[0]; cfma(o.c[0], F.pb, v.c[1]);
  o.c[1] = F.pt * v.c[0]; cfnma(o.c[1], F.p3, v.c[1]);
  o.c[2] = F.m3 * v.c[2]; cfma(o.c[2], F.mb, v.c[3]);
  o.c[3] = F.mt * v.c[2]; cfnma(o.c[3], F.m3, v.c[3]);
  return o;
}
template <class R> TREX_HD spinor<R> spinor_from(const double* __restrict__ p) {
  spinor<R> s;
#pragma unroll
  for (int i = 0; i < 4; ++i) s.c[i] = cx<R>(R(p[2 * i]), R(p[2 * i + 1]));
  return s;
}
// 8 complex components of one record, component-major with `stride` records per component
template <class R> TREX_HD void rec_put(R* __restrict__ t, int stride, int idx, const spinor<R>& a, const spinor<R>& b) {
#pragma unroll
  for (int i = 0; i < 4; ++i) { tab_put<R>(t, i * stride + idx, a.c[i]); tab_put<R>(t, (4 + i) * stride + idx, b.c[i]); }
}
template <class R> TREX_HD void rec_get(const R* __restrict__ t, int stride, int idx, int sign, spinor<R>& a, spinor<R>& b) {
#pragma unroll
  for (int i = 0; i < 4; ++i) { a.c[i] = tab_get<R>(t, i * stride + idx, sign); b.c[i] = tab_get<R>(t, (4 + i) * stride + idx, sign); }
}

// ---------------------------------------------------------------- phase 2: depth-first walk of the top line
// The first D gluons of the ordering are given (the task); below them every remaining ordering is visited. Private
// state: the line spinors U[UT+1..N-1] (dual numbers in kappa). Every vertex operand comes from the table.
// UT > 0 (all helicities free, NFIX = 0): the line states of the prefixes of length <= UT do not depend on the rest of
// the ordering nor on the other helicities; they are tabulated once per event and parameter point (utab, built by
// walks with STOP = 1 .. UT that store U[STOP] instead of descending) and the walk starts at level UT + 1.
//   utab[comp * nut + ubase + index], comp = (order 0 / 1, spinor component, re / im) = 0..15
//   index level 1: (state of (g1, hel)) * 2 + lt;   level 2: N1 + ((rank of (g1,g2) among ordered pairs) * 4 + hels) * 2 + lt
template <int N, int NFIX> struct UTabIdx {
  // level 1: one state per (gluon, helicity, lt); a gluon whose helicity the outer loop fixes has one helicity per iteration
  static constexpr int N1 = 2 * (NFIX + 2 * (N - NFIX)), N2 = 8 * N * (N - 1), NU = N1 + N2;
  TREX_HD static int level1(int g1, unsigned bits, int lt) {
    return (g1 < NFIX ? g1 : NFIX + 2 * (g1 - NFIX) + (int)(bits & 1u)) * 2 + lt;
  }
  // inverse of level1 >> 1
  TREX_HD static void level1_decode(int idx, int& g1, unsigned& bit) {
    if (idx < NFIX) { g1 = idx; bit = 0u; } else { g1 = NFIX + ((idx - NFIX) >> 1); bit = (unsigned)((idx - NFIX) & 1); }
  }
  TREX_HD static int level2(int g1, int g2, unsigned bits, int lt) {     // NFIX = 0 only
    return N1 + ((g1 * (N - 1) + g2 - (g2 > g1 ? 1 : 0)) * 4 + (int)(bits & 3u)) * 2 + lt;
  }
};

template <class R, int N, int NFIX, int D, class Sink, int UT = 0, int STOP = 0> struct TabWalk {
  using I = TabIdx<N, NFIX>;
  static constexpr int NE = I::NE;
  static_assert(UT <= 1 || (NFIX == 0 && UT == 2), "line-state tables: prefixes of length 1, or 2 with all helicities free");
  const R* tab; const int* off; const rvec4<double>* pset;
  R* utab; int nut, ubase, lt;        // line-state table (UT > 0 or STOP > 0)
  rvec4<double> pt;
  spinor<R> ubar_t;
  TopLine line;
  unsigned hfree;                     // helicity bit of free gluon g at bit (g - NFIX)
  int pref[D];
  int s[N];                           // ordering prefix
  unsigned cb;                        // helicity bits of the free gluons of the prefix, in path order
  int fpos[N + 1];                    // free gluons among s[0..m)
  unsigned prefmask[N + 1];
  dspinor<R> U[N];                    // U[m], m = 1..N-1 (U[0] = ubar_t, order 1 = 0)
  int leaf;
  Sink* sink;

  template <int A> TREX_HD int uindex() const {
    if constexpr (A == 1) return ubase + UTabIdx<N, NFIX>::level1(s[0], fpos[1] ? cb : 0u, lt);   // a fixed helicity has no bit in cb
    else return ubase + UTabIdx<N, NFIX>::level2(s[0], s[1], cb, lt);
  }
  // line state after the first A gluons: private, or from the per-event table
  template <int A> TREX_HD dspinor<R> state() const {
    if constexpr (A <= UT) {
      dspinor<R> u;
      const int e = uindex<A>();
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        u.o0.c[i] = tab_get<R>(utab, i * nut + e, 1);
        u.o1.c[i] = tab_get<R>(utab, (4 + i) * nut + e, 1);
      }
      return u;
    } else return U[A];
  }

  // s0 += U_a^(0) Jslash_a;  s1 += U_a^(1) Jslash_a - i U_a^(0) 2 sigma.F_a;  the bracket is (i s0, i s1)
  template <int M, int A> TREX_HD void bracket_terms(spinor<R>& s0, spinor<R>& s1) {
    if constexpr (A < M) {
      int sign;
      const int e = tab_entry<N, NFIX, M - A>(off, s + A, cb >> fpos[A], fpos[M] - fpos[A], sign);
      const vec4<R> J = tab_J<R, NE>(tab, e, sign);
      if constexpr (A == 0) {
        row_slash_acc(s0, ubar_t, J);
        row_sigma_acc_x(s1, ubar_t, tab_F<R, NE>(tab, e, sign));
      } else {
        const dspinor<R> u = state<A>();
        row_slash_acc(s0, u.o0, J);
        row_slash_acc(s1, u.o1, J);
        row_sigma_acc_x(s1, u.o0, tab_F<R, NE>(tab, e, sign));
      }
      bracket_terms<M, A + 1>(s0, s1);
    }
  }

  // bookkeeping of position M (no arithmetic)
  template <int M> TREX_HD void place(int g) {
    s[M - 1] = g;
    const bool isfree = g >= NFIX;
    const unsigned bit = isfree ? (hfree >> (g - NFIX)) & 1u : 0u;
    cb = (cb & ((1u << fpos[M - 1]) - 1u)) | (bit << fpos[M - 1]);
    fpos[M] = fpos[M - 1] + (isfree ? 1 : 0);
    prefmask[M] = prefmask[M - 1] | (1u << g);
  }

  template <int M> TREX_HD void node(int g) {
    place<M>(g);
    if constexpr (M <= UT) {
      // tabulated level: nothing to compute
      if constexpr (M < D) node<M + 1>(pref[M]);
      else descend<M>();
    } else {
      spinor<R> b0 = szero<R>(), b1 = szero<R>();
      bracket_terms<M, 0>(b0, b1);
#pragma unroll
      for (int i = 0; i < 4; ++i) { b0.c[i] = mul_i(b0.c[i]); b1.c[i] = mul_i(b1.c[i]); }
      if constexpr (M < N) {
        const rvec4<double> qd = rsub(pt, pset[prefmask[M]]);
        const double q2 = rdot(qd, qd);
        const rvec4<R> q = cast<R>(qd);
        const cx<double> den(q2 - line.mt * line.mt, line.mGt);
        const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), den));
        const spinor<R> s0 = row_slash(b0, q), s1 = row_slash(b1, q);
        dspinor<R> u;
#pragma unroll
        for (int i = 0; i < 4; ++i) {
          cx<R> n0 = s0.c[i]; cfma(n0, b0.c[i], R(line.mt));
          cx<R> n1 = s1.c[i]; cfma(n1, b1.c[i], R(line.mt));
          u.o0.c[i] = n0 * pr; u.o1.c[i] = n1 * pr;
        }
        if constexpr (M == STOP) {
          const int e = uindex<M>();
#pragma unroll
          for (int i = 0; i < 4; ++i) {
            tab_put<R>(utab, i * nut + e, u.o0.c[i]);
            tab_put<R>(utab, (4 + i) * nut + e, u.o1.c[i]);
          }
        } else {
          U[M] = u;
          if constexpr (M < D) node<M + 1>(pref[M]);
          else descend<M>();
        }
      } else {
        (*sink)(leaf, b0, b1);
        ++leaf;
      }
    }
  }
  template <int M> TREX_HD void descend() {
    if constexpr (M < N) {
      // every thread visits the r-th unused gluon at the same trip: uniform control flow across ordering prefixes
      for (int r = 0; r < N - M; ++r) node<(M < N ? M + 1 : N)>(I::nth_unused(prefmask[M], r));
    }
  }

  TREX_HD void run(Sink* sk) {
    sink = sk; leaf = 0; cb = 0; prefmask[0] = 0; fpos[0] = 0;
    node<1>(pref[0]);
  }
};

// the d-th ordered D-tuple of distinct gluons in lexicographic order
template <int N, int D> TREX_HD void prefix_of_rank(int rank, int* pref) {
  unsigned used = 0;
  int radix = TabIdx<N, 0>::falling(N, D);
#pragma unroll
  for (int i = 0; i < D; ++i) {
    radix /= (N - i);
    int c = rank / radix; rank -= c * radix;
    int m = 0;
    for (;; ++m) { if (!((used >> m) & 1u)) { if (c == 0) break; --c; } }
    pref[i] = m; used |= 1u << m;
  }
}

}  // namespace trex
