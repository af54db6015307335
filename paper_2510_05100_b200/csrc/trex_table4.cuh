// trex_table4.cuh -- g g -> t t~ g g (N = 4): the W-form current-table kernel as a software pipeline over events.
// Included by trex_table_tu.cu (inside its anonymous namespace) for TREX_TU_N == 4; see trex_table.cuh for the method.
//
// A block owns one event at a time, but the narrow steps of the NEXT event run beside the wide steps of the current one,
// so that no phase leaves most of the block waiting at a barrier:
//   phase B(i): level-4 entries of event i (warps 0-5)  |  "prep" of event i+1 (warps 6, 7): momenta, subset momenta,
//               polarisations, spinors, bilinears, table levels 1 and 2 with their W records, line states U1
//   phase C(i): top-line walk of event i (all warps)
//   phase D(i): colour sum of event i (fp64: six warps on the tensor cores)  |  level-3 entries + line states U2 of
//               event i+1 (the other six warps; all warps do both when the colour sum is in FFMA form)
//   epilogue(i) by warp 8, which is idle in phase B, while the others start phase B(i+1)
// Three block barriers per event. What prep writes is double-buffered by event parity: the per-event constants are two
// small blocks; the table entries of levels 1 and 2 (indices < PE), their W records and the U1 states have a second copy
// at the end of their arrays (index + poff). Which references are of level <= 2 is known at compile time.
#pragma once

template <class R, class RC> struct W4 {
  using I = TabIdx<4, 0>;
  using UI = UTabIdx<4, 0>;
  using G = TabGeom<R, RC, 4>;
  static constexpr int NE = I::NE, PE = I::entries_below(3), E4 = I::entries_below(4);
  // table stride (entries per component); odd, so that the closed scalars of lambda_t = -/+ (4 components apart, read by
  // the lanes of one warp in one instruction) fall into different halves of a 128-byte bank line
  static constexpr int TS = NE + PE + 1;
  static constexpr int NWR = 2 * (E4 + PE);             // W records: (entry below level 4, lambda_tbar)
  static constexpr int NUB = 2 * (E4 - PE);             // A = 0 rows of the level-3 entries: (entry, lambda_t)
  static constexpr int N1 = UI::N1, N2 = UI::N2, NU = N1 + N2, NUT = 2 * NU, US = NUT + 2 * N1;   // line-state records
  static constexpr int TB = 384, XS = G::XS, NC = 24;
#ifndef TREX_T4_NCW
#define TREX_T4_NCW 6
#endif
  static constexpr int NCW = TREX_T4_NCW;               // warps that take the tensor-core colour sum in phase D
  struct Small {                                        // per-event constants, one block per parity
    rvec4<double> pset[16];
    double eps[64], spin[32], pm[24];
    R bil[80];
  };
  static constexpr size_t al(size_t x) { return (x + 15) / 16 * 16; }
  static constexpr size_t o_tab = 0;
  static constexpr size_t o_x = o_tab + al(sizeof(R) * TAB_NCOMP * TS);
  static constexpr size_t o_w = o_x + al(sizeof(cx<RC>) * NC * XS);
  static constexpr size_t o_ub = o_w + al(sizeof(R) * 16 * NWR);
  static constexpr size_t o_utab = o_ub + al(sizeof(R) * 16 * NUB);
  static constexpr size_t o_part = o_utab + al(sizeof(R) * 16 * US);
  static constexpr size_t o_small = o_part + al(sizeof(double) * G::NCI);
  static constexpr size_t o_c = o_small + 2 * al(sizeof(Small));
  static constexpr size_t o_meta = o_c + al(sizeof(RC) * G::CN);
  static constexpr size_t bytes = o_meta + al(sizeof(int) * I::M_SIZE);
  static_assert(bytes <= 232448, "one SM has 227 KB of shared memory");
  __device__ static int uidx1(int pass, int idx, int par) { return par ? NUT + pass * N1 + idx : pass * NU + idx; }
};

template <class R> struct W4Ptr {        // shared-memory views of one block
  R* tab; R* wtab; R* ubt; R* utab;
  const int* meta;
};

// table entry of level K <= 3 finished: J and -i 2 sigma.F, W records, and (K = 3) the A = 0 rows
template <class R, class RC, int K>
__device__ __forceinline__ void w4_finish(const W4Ptr<R>& p, const typename W4<R, RC>::Small& sm, int e, int poff, const vec4<R>& J, const sigF<R>& F) {
  using W = W4<R, RC>;
  const int es = K <= 2 ? e + poff : e;                    // table slot; the W array ends at E4: odd copies at E4 + e
  const int ew = (K <= 2 && poff) ? e + W::E4 : e;
  tab_store<R, W::TS>(p.tab, es, J, F);
#pragma unroll
  for (int ltb = 0; ltb < 2; ++ltb) {
    const spinor<R> v = spinor_from<R>(sm.spin + (2 + ltb) * 8);
    spinor<R> wj = slash_col(J, v), wf = sig_col(F, v);
#pragma unroll
    for (int i = 0; i < 4; ++i) { wj.c[i] = mul_i(wj.c[i]); wf.c[i] = mul_i(wf.c[i]); }
    rec_put<R>(p.wtab, W::NWR, ew * 2 + ltb, wj, wf);
  }
  if constexpr (K == 3) {
#pragma unroll
    for (int lt = 0; lt < 2; ++lt) {
      const spinor<R> ub = spinor_from<R>(sm.spin + lt * 8);
      spinor<R> s0 = szero<R>(), s1 = szero<R>();
      row_slash_acc(s0, ub, J);
      row_sigma_acc_x(s1, ub, F);
      rec_put<R>(p.ubt, W::NUB, (e - W::PE) * 2 + lt, s0, s1);
    }
  }
}

// line state from its open bracket (s0, s1) [without the factor i]: U = i s (qslash + m) i / (q^2 - m^2 + i m Gamma)
template <class R> __device__ __forceinline__ dspinor<R> w4_propagate(spinor<R> s0, spinor<R> s1, const rvec4<double>& qd, double mt, double mGt) {
#pragma unroll
  for (int i = 0; i < 4; ++i) { s0.c[i] = mul_i(s0.c[i]); s1.c[i] = mul_i(s1.c[i]); }
  const double q2 = rdot(qd, qd);
  const rvec4<R> q = cast<R>(qd);
  const cx<R> pr = cast<R>(cdiv(cx<double>(0, 1), cx<double>(q2 - mt * mt, mGt)));
  const spinor<R> n0 = row_slash(s0, q), n1 = row_slash(s1, q);
  dspinor<R> U;
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    cx<R> x0 = n0.c[i]; cfma(x0, s0.c[i], R(mt));
    cx<R> x1 = n1.c[i]; cfma(x1, s1.c[i], R(mt));
    U.o0.c[i] = x0 * pr; U.o1.c[i] = x1 * pr;
  }
  return U;
}

// ---- prep of one event by warps 6 (role 0) and 7 (role 1); they meet once at named barrier 1
template <class R, class RC, int NPASS>
__device__ __forceinline__ void w4_prep(const W4Ptr<R>& p, typename W4<R, RC>::Small& sm, const EvIO& io, const ReweightArgs& a, long e, int par, int role, int lane) {
  using W = W4<R, RC>;
  using I = typename W::I;
  constexpr int N = 4;
  const int poff = par ? W::NE : 0;
  if (role == 0) {
    if (lane < 24) sm.pm[lane] = io.mom[(long)lane * io.ld + e];
    __syncwarp();
    if (lane < 16) {
      rvec4<double> P;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) P.c[mu] = 0.0;
#pragma unroll
      for (int g = 0; g < N; ++g) {
        if (!((lane >> g) & 1)) continue;
        const int leg = g < 2 ? g : g + 2;
        const double sg = g < 2 ? 1.0 : -1.0;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) P.c[mu] += sg * sm.pm[leg * 4 + mu];
      }
      sm.pset[lane] = P;
    } else if (lane < 28) {
      const int it = lane - 16;
      double q[4];
      if (it < 2 * N) {
        const int g = it >> 1, leg = g < 2 ? g : g + 2;
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) q[mu] = sm.pm[leg * 4 + mu];
        const vec4<double> ev = polvec<double>(q, (it & 1) ? 1 : -1, g >= 2);
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) { sm.eps[it * 8 + 2 * mu] = ev.c[mu].re; sm.eps[it * 8 + 2 * mu + 1] = ev.c[mu].im; }
      } else {
        const int k = it - 2 * N;                          // 0, 1: ubar(p_t, -/+); 2, 3: v(p_tbar, -/+)
#pragma unroll
        for (int mu = 0; mu < 4; ++mu) q[mu] = sm.pm[(k < 2 ? 2 : 3) * 4 + mu];
        const spinor<double> sp = k < 2 ? bar(spinor_u<double>(q, (k & 1) ? 1 : -1, false)) : spinor_v<double>(q, (k & 1) ? 1 : -1, false);
#pragma unroll
        for (int i = 0; i < 4; ++i) { sm.spin[k * 8 + 2 * i] = sp.c[i].re; sm.spin[k * 8 + 2 * i + 1] = sp.c[i].im; }
      }
    }
    __syncwarp();
    if (lane < 8) {                                        // level 1
      vec4<R> J; ften<R> Fw;
      tab_level1_JF<R, N, 0>(p.meta, sm.pset, sm.eps, 0u, lane, J, Fw);
      w4_finish<R, RC, 1>(p, sm, lane, poff, J, make_sigF<R>(Fw));
    } else if (lane < 12) {
      // bilinears of the closed line, per (lambda_t, lambda_tbar): i ubar Aslash v = sum_k c_k (a+, a-, at, ab)_k with
      // a+- = a0 +- a3, at/ab = a1 +- i a2, and i ubar (-i 2 sigma.F) v = sum_k c_k (p3, pt, pb, m3, mt, mb)_k (w4_top)
      const int combo = lane - 8, lt = combo >> 1, ltb = combo & 1;
      const spinor<R> r = spinor_from<R>(sm.spin + lt * 8), v = spinor_from<R>(sm.spin + (2 + ltb) * 8);
      cx<R> c[10];
      c[0] = r.c[2] * v.c[0]; cfma(c[0], r.c[1], v.c[3]);
      c[1] = r.c[3] * v.c[1]; cfma(c[1], r.c[0], v.c[2]);
      c[2] = r.c[3] * v.c[0]; cfnma(c[2], r.c[1], v.c[2]);
      c[3] = r.c[2] * v.c[1]; cfnma(c[3], r.c[0], v.c[3]);
      c[4] = r.c[0] * v.c[0]; cfnma(c[4], r.c[1], v.c[1]);
      c[5] = r.c[1] * v.c[0];
      c[6] = r.c[0] * v.c[1];
      c[7] = r.c[2] * v.c[2]; cfnma(c[7], r.c[3], v.c[3]);
      c[8] = r.c[3] * v.c[2];
      c[9] = r.c[2] * v.c[3];
#pragma unroll
      for (int k = 0; k < 10; ++k) tab_put<R>(sm.bil, combo * 10 + k, mul_i(c[k]));
    }
    __syncwarp();
    asm volatile("bar.sync 1, 64;" ::: "memory");
    if (lane < 24) {                                       // level 2
      const int e2 = W::I::entries_below(2) + lane;
      TabBuild<R, N, 0, 2, W::TS, 2> b;
      tab_build_setup<R, N, 0, 2>(b, p.tab, p.meta, sm.pset, e2);
      b.poff = poff;
      vec4<R> J; ften<R> Fw;
      b.compute(J, Fw);
      w4_finish<R, RC, 2>(p, sm, e2, poff, J, make_sigF<R>(Fw));
    }
  } else {
    asm volatile("bar.sync 1, 64;" ::: "memory");
    if (lane < W::N1 * NPASS) {                            // line states after one gluon: (gluon, helicity, lambda_t) x pass
      const int pass = lane / W::N1, idx = lane - pass * W::N1, lt = idx & 1, h = (idx >> 1) & 1, g = idx >> 2;
      const int e1 = g * 2 + h + poff;
      const spinor<R> ub = spinor_from<R>(sm.spin + lt * 8);
      spinor<R> s0 = szero<R>(), s1 = szero<R>();
      row_slash_acc(s0, ub, tab_J<R, W::TS>(p.tab, e1, 1));
      row_sigma_acc_x(s1, ub, tab_F<R, W::TS>(p.tab, e1, 1));
      rvec4<double> pt;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) pt.c[mu] = sm.pm[8 + mu];
      const dspinor<R> U = w4_propagate<R>(s0, s1, rsub(pt, sm.pset[1u << g]), a.T.mt[pass], a.T.mGt[pass]);
      rec_put<R>(p.utab, W::US, W::uidx1(pass, idx, par), U.o0, U.o1);
    }
  }
}

// ---- level-3 entries and the line states after two gluons of one event (needs its prep)
template <class R, class RC, int NPASS>
__device__ __forceinline__ void w4_build3(const W4Ptr<R>& p, const typename W4<R, RC>::Small& sm, const ReweightArgs& a, int par, int tid, int nthreads) {
  using W = W4<R, RC>;
  using I = typename W::I;
  constexpr int N = 4, NL3 = W::E4 - W::PE;
  const int poff = par ? W::NE : 0;
  for (int it = tid; it < NL3 + W::N2 * NPASS; it += nthreads) {
    if (it < NL3) {
      const int e = W::PE + it;
      TabBuild<R, N, 0, 3, W::TS, 2> b;
      tab_build_setup<R, N, 0, 3>(b, p.tab, p.meta, sm.pset, e);
      b.poff = poff;
      vec4<R> J; ften<R> Fw;
      b.compute(J, Fw);
      w4_finish<R, RC, 3>(p, sm, e, poff, J, make_sigF<R>(Fw));
    } else {
      const int u = it - NL3, pass = u / W::N2, r = u - pass * W::N2;
      const int lt = r & 1, pr = r >> 3;
      const unsigned bits = (unsigned)(r >> 1) & 3u;
      const int g1 = pr / 3, rr = pr - g1 * 3, g2 = rr + (rr >= g1 ? 1 : 0);
      const int t2[2] = {g1, g2};
      int sign;
      const int e12 = tab_entry<N, 0, 2>(p.meta + I::M_OFF, t2, bits, 2, sign) + poff;
      const spinor<R> ub = spinor_from<R>(sm.spin + lt * 8);
      spinor<R> s0 = szero<R>(), s1 = szero<R>();
      row_slash_acc(s0, ub, tab_J<R, W::TS>(p.tab, e12, sign));
      row_sigma_acc_x(s1, ub, tab_F<R, W::TS>(p.tab, e12, sign));
      dspinor<R> U1;
      rec_get<R>(p.utab, W::US, W::uidx1(pass, W::UI::level1(g1, bits & 1u, lt), par), 1, U1.o0, U1.o1);
      const int e2 = g2 * 2 + (int)(bits >> 1) + poff;
      const vec4<R> J = tab_J<R, W::TS>(p.tab, e2, 1);
      row_slash_acc(s0, U1.o0, J); row_slash_acc(s1, U1.o1, J);
      row_sigma_acc_x(s1, U1.o0, tab_F<R, W::TS>(p.tab, e2, 1));
      rvec4<double> pt;
#pragma unroll
      for (int mu = 0; mu < 4; ++mu) pt.c[mu] = sm.pm[8 + mu];
      const dspinor<R> U = w4_propagate<R>(s0, s1, rsub(pt, sm.pset[(1u << g1) | (1u << g2)]), a.T.mt[pass], a.T.mGt[pass]);
      rec_put<R>(p.utab, W::US, pass * W::NU + W::N1 + r, U.o0, U.o1);
    }
  }
}

// ---- a level-4 entry: J and F stay in registers and are closed with the bilinears into S0 = i ubar Jslash v,
// S1 = i ubar (-i 2 sigma.F) v for the four (lambda_t, lambda_tbar); stored in the entry's own table slots
template <class R, class RC>
__device__ __forceinline__ void w4_top(const W4Ptr<R>& p, const typename W4<R, RC>::Small& sm, int e, int par) {
  using W = W4<R, RC>;
  constexpr int N = 4;
  TabBuild<R, N, 0, N, W::TS, 2> b;
  tab_build_setup<R, N, 0, N>(b, p.tab, p.meta, sm.pset, e);
  b.poff = par ? W::NE : 0;
  vec4<R> acc = vzero<R>();
  ften<R> Fc = fzero<R>();
  b.template v3_splits<1>(acc, Fc);
  b.template v4_splits<1, 2>(acc);
  const rvec4<double>& P = sm.pset[15];
  const R sc = R(-1.0 / rdot(P, P));
  vec4<R> J;
#pragma unroll
  for (int i = 0; i < 4; ++i) J.c[i] = acc.c[i] * sc;
  wedge_acc(Fc, cast<R>(P), J);
  const sigF<R> F = make_sigF<R>(Fc);
  const cx<R> a4[4] = {J.c[0] + J.c[3], J.c[0] - J.c[3], J.c[1] + mul_i(J.c[2]), J.c[1] - mul_i(J.c[2])};
  const cx<R>* f6 = &F.p3;
#pragma unroll
  for (int combo = 0; combo < 4; ++combo) {
    cx<R> s0 = tab_get<R>(sm.bil, combo * 10, 1) * a4[0];
#pragma unroll
    for (int k = 1; k < 4; ++k) cfma(s0, tab_get<R>(sm.bil, combo * 10 + k, 1), a4[k]);
    cx<R> s1 = tab_get<R>(sm.bil, combo * 10 + 4, 1) * f6[0];
#pragma unroll
    for (int k = 1; k < 6; ++k) cfma(s1, tab_get<R>(sm.bil, combo * 10 + 4 + k, 1), f6[k]);
    tab_put<R>(p.tab, (combo * 2 + 0) * W::TS + e, s0);
    tab_put<R>(p.tab, (combo * 2 + 1) * W::TS + e, s1);
  }
}

// U . W terms of one leaf: a0 += sign U.o0 . Wj,  a1 += sign (U.o1 . Wj + U.o0 . Wf)
template <class R> __device__ __forceinline__ void w4_leaf_term(cx<R>& a0, cx<R>& a1, const dspinor<R>& U, const R* __restrict__ wtab, int nwr, int rec, int sign) {
  spinor<R> wj, wf;
  rec_get<R>(wtab, nwr, rec, 1, wj, wf);
  cx<R> t0 = U.o0.c[0] * wj.c[0], t1 = U.o1.c[0] * wj.c[0];
#pragma unroll
  for (int i = 1; i < 4; ++i) { cfma(t0, U.o0.c[i], wj.c[i]); cfma(t1, U.o1.c[i], wj.c[i]); }
#pragma unroll
  for (int i = 0; i < 4; ++i) cfma(t1, U.o0.c[i], wf.c[i]);
  a0 += cx<R>(with_sign(t0.re, sign), with_sign(t0.im, sign));
  a1 += cx<R>(with_sign(t1.re, sign), with_sign(t1.im, sign));
}

// ---- top-line walk: task = (ordering, helicities of s1 s2 s3, lambda_t, pass); closes both helicities of s4 and both
// antitop helicities from one line state U3 (see the "W form" section of trex_table.cuh)
// HS (helicity symmetry, R-21; one parameter-point pass, Gamma_t = 0): only the 192 tasks with lambda_t = - exist,
// one per thread of warps 0-5, and they run BESIDE the level-4 entries (warps 6-11): the closed scalars of level 4 enter a
// task only as the starting value of its sums, so the task keeps its sums (W4Held) and w4_walk_finish adds the scalars and
// writes the X tile after the block barrier.
template <class R> struct W4Held { cx<R> a0[4], a1[4]; int e4[4], colc[4], sg0, prank; };

template <class R, class RC, int NPASS, bool HS = false>
__device__ __forceinline__ void w4_walk(const W4Ptr<R>& p, const typename W4<R, RC>::Small& sm, cx<RC>* __restrict__ xs, const ReweightArgs& a, int par, int tid,
                                        W4Held<R>* held = nullptr) {
  static_assert(!HS || NPASS == 1, "the symmetric walk has one pass");
  using W = W4<R, RC>;
  using I = typename W::I;
  constexpr int TS = W::TS, XS = W::XS;
  const int poff = par ? W::NE : 0, poffw = par ? W::E4 : 0;
  rvec4<double> pt;
#pragma unroll
  for (int mu = 0; mu < 4; ++mu) pt.c[mu] = sm.pm[8 + mu];
  const R kq0 = R(a.T.kq[0]), kq1 = R(a.T.kq[1]);
  for (int task = tid; task < (HS ? 192 : 384 * NPASS); task += W::TB) {
    const int pass = HS ? 0 : task / 384, r = HS ? 2 * task : task - pass * 384;
    const int prank = r >> 4, lt = r & 1;
    const unsigned hp = (unsigned)(r >> 1) & 7u;             // helicities of s1, s2, s3 (bit i: s_{i+1})
    // table references of this ordering (TabIdx::M_REC): no index arithmetic on the critical path of the loads
    const int4 rc = reinterpret_cast<const int4*>(p.meta + I::M_REC)[prank];
    const auto ref = [](unsigned rf, unsigned bits, int nf, int& sign) {
      sign = (rf & 0x400u) ? -1 : 1;
      return (int)(rf & 0x1FFu) + (int)((rf & 0x200u) ? I::bitrev(bits, nf) : bits);
    };
    const unsigned sp = (unsigned)rc.w >> 16;
    const int s0i = (int)(sp & 3u), s3i = (int)((sp >> 6) & 3u);
    dspinor<R> U1, U2, U3;
    rec_get<R>(p.utab, W::US, W::uidx1(pass, W::UI::level1(s0i, hp & 1u, lt), par), 1, U1.o0, U1.o1);
    rec_get<R>(p.utab, W::US, pass * W::NU + W::N1 + (((int)(sp >> 8) * 4 + (int)(hp & 3u)) * 2 + lt), 1, U2.o0, U2.o1);
    // ---- node 3: U3 = [ ubar Gamma(J(s1 s2 s3)) + U1 Gamma(J(s2 s3)) + U2 Gamma(J(s3)) ] S(p_t - K(s1 s2 s3))
    {
      spinor<R> s0, s1;
      int sign;
      int e = ref((unsigned)rc.x & 0xFFFFu, hp, 3, sign);
      rec_get<R>(p.ubt, W::NUB, (e - W::PE) * 2 + lt, sign, s0, s1);
      e = ref((unsigned)rc.x >> 16, hp >> 1, 2, sign) + poff;
      {
        const vec4<R> J = tab_J<R, TS>(p.tab, e, sign);
        row_slash_acc(s0, U1.o0, J); row_slash_acc(s1, U1.o1, J);
        row_sigma_acc_x(s1, U1.o0, tab_F<R, TS>(p.tab, e, sign));
      }
      e = ref((unsigned)rc.y & 0xFFFFu, hp >> 2, 1, sign) + poff;
      {
        const vec4<R> J = tab_J<R, TS>(p.tab, e, sign);
        row_slash_acc(s0, U2.o0, J); row_slash_acc(s1, U2.o1, J);
        row_sigma_acc_x(s1, U2.o0, tab_F<R, TS>(p.tab, e, sign));
      }
      U3 = w4_propagate<R>(s0, s1, rsub(pt, sm.pset[15u ^ (1u << s3i)]), a.T.mt[pass], a.T.mGt[pass]);
    }
    // ---- leaves: the four (helicity of s4, lambda_tbar) combinations c = 2 h4 + ltb are closed together,
    //   a0[c] = S0 + sum_A U_A.o0 . Wj_A[c],   a1[c] = S1 + sum_A (U_A.o1 . Wj_A[c] + U_A.o0 . Wf_A[c]),
    // component by component, so that one line-state component multiplies eight table numbers in a row (the FP64 pipe
    // reads such a repeated operand from its reuse cache: two register reads per DFMA instead of three). The sign of a
    // reversed tuple depends on the ordering only and is folded into the line state once.
    int sg0, sg1, sg2, sg3;
    const int b4 = ref((unsigned)rc.y >> 16, 0u, 4, sg0), b1 = ref((unsigned)rc.z & 0xFFFFu, 0u, 3, sg1);
    const int b2 = ref((unsigned)rc.z >> 16, 0u, 2, sg2), b3 = ref((unsigned)rc.w & 0xFFFFu, 0u, 1, sg3);
    const bool r4 = ((unsigned)rc.y >> 16) & 0x200u, r1 = (unsigned)rc.z & 0x200u, r2 = ((unsigned)rc.z >> 16) & 0x200u;
    cx<R> a0[4], a1[4];
    int rec1[4], rec2[4], rec3[4], colc[4];
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      const unsigned h4 = (unsigned)c >> 1, hp4 = hp | (h4 << 3);
      const int ltb = c & 1;
      const int e4 = b4 + (int)(r4 ? I::bitrev(hp4, 4) : hp4);
      if constexpr (HS) { a0[c] = cx<R>(R(0), R(0)); a1[c] = cx<R>(R(0), R(0)); held->e4[c] = e4; }
      else {
        a0[c] = tab_get<R>(p.tab, ((lt * 2 + ltb) * 2 + 0) * TS + e4, sg0);
        a1[c] = tab_get<R>(p.tab, ((lt * 2 + ltb) * 2 + 1) * TS + e4, sg0);
      }
      rec1[c] = (b1 + (int)(r1 ? I::bitrev(hp4 >> 1, 3) : hp4 >> 1)) * 2 + ltb;
      rec2[c] = (b2 + (int)(r2 ? I::bitrev(hp4 >> 2, 2) : hp4 >> 2) + poffw) * 2 + ltb;
      rec3[c] = (b3 + (int)h4 + poffw) * 2 + ltb;
      unsigned hfree = 0;
#pragma unroll
      for (int i = 0; i < 4; ++i) hfree |= ((hp4 >> i) & 1u) << ((sp >> (2 * i)) & 3u);
      colc[c] = (((int)hfree * 2 + lt) * 2 + ltb) * 2;
    }
    const auto close_with = [&](const dspinor<R>& U, int sign, const int* rec) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const cx<R> u0(with_sign(U.o0.c[i].re, sign), with_sign(U.o0.c[i].im, sign));
        const cx<R> u1(with_sign(U.o1.c[i].re, sign), with_sign(U.o1.c[i].im, sign));
#pragma unroll
        for (int c = 0; c < 4; ++c) {
          const cx<R> wj = tab_get<R>(p.wtab, i * W::NWR + rec[c], 1), wf = tab_get<R>(p.wtab, (4 + i) * W::NWR + rec[c], 1);
          cfma(a0[c], u0, wj); cfma(a1[c], u0, wf); cfma(a1[c], u1, wj);
        }
      }
    };
    close_with(U1, sg1, rec1);
    close_with(U2, sg2, rec2);
    close_with(U3, sg3, rec3);
    if constexpr (HS) {
#pragma unroll
      for (int c = 0; c < 4; ++c) { held->a0[c] = a0[c]; held->a1[c] = a1[c]; held->colc[c] = colc[c]; }
      held->sg0 = sg0; held->prank = prank;
    } else
#pragma unroll
    for (int c = 0; c < 4; ++c) {
      if constexpr (NPASS == 1) {
        cx<R> x = a0[c]; cfma(x, a1[c], kq0);
        cx<R> y = a0[c]; cfma(y, a1[c], kq1);
        xs[prank * XS + colc[c]] = cx<RC>(RC(x.re), RC(x.im));
        xs[prank * XS + colc[c] + 1] = cx<RC>(RC(y.re), RC(y.im));
      } else {
        cx<R> x = a0[c]; cfma(x, a1[c], pass == 0 ? kq0 : kq1);
        xs[prank * XS + colc[c] + pass] = cx<RC>(RC(x.re), RC(x.im));
      }
    }
  }
}

// second half of a symmetric walk task (after the level-4 entries are complete): lambda_t = -, combos c = 2 h4 + ltb
template <class R, class RC>
__device__ __forceinline__ void w4_walk_finish(const W4Ptr<R>& p, cx<RC>* __restrict__ xs, const ReweightArgs& a, const W4Held<R>& h) {
  using W = W4<R, RC>;
  const R kq0 = R(a.T.kq[0]), kq1 = R(a.T.kq[1]);
#pragma unroll
  for (int c = 0; c < 4; ++c) {
    const int ltb = c & 1;
    const cx<R> a0 = h.a0[c] + tab_get<R>(p.tab, (ltb * 2 + 0) * W::TS + h.e4[c], h.sg0);
    const cx<R> a1 = h.a1[c] + tab_get<R>(p.tab, (ltb * 2 + 1) * W::TS + h.e4[c], h.sg0);
    cx<R> x = a0; cfma(x, a1, kq0);
    cx<R> y = a0; cfma(y, a1, kq1);
    xs[h.prank * W::XS + h.colc[c]] = cx<RC>(RC(x.re), RC(x.im));
    xs[h.prank * W::XS + h.colc[c] + 1] = cx<RC>(RC(y.re), RC(y.im));
  }
}

template <class R, class RC, int NPASS>
__global__ void __launch_bounds__(384, 1) k_table4w(const ReweightArgs a, const int* __restrict__ gmeta, const double* __restrict__ Cfold) {
  using W = W4<R, RC>;
  using G = typename W::G;
  using I = typename W::I;
  using F = FoldedC<W::NC>;
  using Small = typename W::Small;
  extern __shared__ __align__(16) unsigned char smem[];
  RC* Cs = reinterpret_cast<RC*>(smem + W::o_c);
  int* meta = reinterpret_cast<int*>(smem + W::o_meta);
  cx<RC>* xs = reinterpret_cast<cx<RC>*>(smem + W::o_x);
  double* part = reinterpret_cast<double*>(smem + W::o_part);
  Small* small = reinterpret_cast<Small*>(smem + W::o_small);
  W4Ptr<R> p;
  p.tab = reinterpret_cast<R*>(smem + W::o_tab); p.wtab = reinterpret_cast<R*>(smem + W::o_w);
  p.ubt = reinterpret_cast<R*>(smem + W::o_ub); p.utab = reinterpret_cast<R*>(smem + W::o_utab); p.meta = meta;
  const int tid = threadIdx.x, lane = tid & 31, wrp = tid >> 5;
  const EvIO io = resolve_io(a);
  const long e_first = blockIdx.x, e_step = gridDim.x;
  if (e_first >= io.n) return;
  for (int i = tid; i < I::M_SIZE; i += W::TB) meta[i] = gmeta[i];
  for (int i = tid; i < G::CN; i += W::TB) Cs[i] = RC(Cfold[i]);
  for (int i = tid; i < G::NCI; i += W::TB) part[i] = 0.0;
  __syncthreads();
  // pipeline prologue: prep and level 3 of the block's first event
  if (wrp == 6 || wrp == 7) w4_prep<R, RC, NPASS>(p, small[0], io, a, e_first, 0, wrp - 6, lane);
  __syncthreads();
  w4_build3<R, RC, NPASS>(p, small[0], a, 0, tid, W::TB);
  __syncthreads();
  int par = 0;
#ifdef TREX_PHASE_CLOCKS
  long long pc[4] = {0, 0, 0, 0}, t0 = clock64();
#define W4_TICK(k) do { if (tid == 0) { const long long t1 = clock64(); pc[k] += t1 - t0; t0 = t1; } } while (0)
#else
#define W4_TICK(k) do { } while (0)
#endif
  // helicity symmetry (one pass, Gamma_t = 0): 192 walk tasks beside the level-4 entries; colour sum over the columns of
  // lambda_t = - only; the sum is doubled in the epilogue
  const bool hs = NPASS == 1 && a.hsym && !a.dbg;
  const double hscale = hs ? 2.0 : 1.0;
  const auto epilogue = [&](long ev) {                    // by one warp: fixed-order reduction of the partial sums (slot parity = theta)
    double v = 0.0;
    for (int i = lane; i < G::NCI; i += 32) { v += part[i]; part[i] = 0.0; }
#pragma unroll
    for (int o = 16; o >= 2; o >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, o);
    const double s1 = __shfl_sync(0xFFFFFFFFu, v, 1);
    if (lane == 0) {
      const double mo = v * (a.T.pref[0] * hscale), mn = s1 * (a.T.pref[1] * hscale);
      const double norm = (mo == 0.0) ? 0.0 : 1.0 / mo;          // procReweightor::initialise
      io.w_out[ev] = io.w_in[ev] * norm * mn;                      // evaluate + append_wgts
      if (io.me2_old) io.me2_old[ev] = mo;
      if (io.me2_new) io.me2_new[ev] = mn;
    }
  };
  for (long e = e_first; e < io.n; e += e_step, par ^= 1) {
    const bool more = e + e_step < io.n;
    if constexpr (NPASS == 1) {
      if (hs) {
        // ---- phases B + C merged: walk tasks (warps 0-5) | level-4 entries (warps 6-11), then the epilogue of the previous
        // event (warp 8)
        W4Held<R> held;
        if (wrp < 6) w4_walk<R, RC, 1, true>(p, small[par], xs, a, par, tid, &held);
        else {
          w4_top<R, RC>(p, small[par], W::E4 + tid - 192, par);
          if (wrp == 8 && e != e_first) epilogue(e - e_step);
        }
        __syncthreads();
        W4_TICK(0);
        // the tasks add the level-4 scalars and write X (warps 0-5) | prep of the next event (warps 6, 7). (Measured: prep
        // behind the level-4 entries on the same warps, or two level-4 entries per thread on fewer warps, make the merged
        // phase longer than the walk tasks.)
        if (wrp < 6) w4_walk_finish<R, RC>(p, xs, a, held);
        else if (wrp < 8 && more) w4_prep<R, RC, NPASS>(p, small[par ^ 1], io, a, e + e_step, par ^ 1, wrp - 6, lane);
        __syncthreads();
        W4_TICK(1);
        if constexpr (G::DMMA || G::TF32) {
          if (wrp < W::NCW) colour_phase<R, RC, 4>(xs, Cs, part, tid, tid, W::NCW, true);
          else if (more) w4_build3<R, RC, NPASS>(p, small[par ^ 1], a, par ^ 1, tid - 32 * W::NCW, W::TB - 32 * W::NCW);
        } else {
          colour_phase<R, RC, 4>(xs, Cs, part, tid, tid, 0, true);
          if (more) w4_build3<R, RC, NPASS>(p, small[par ^ 1], a, par ^ 1, tid, W::TB);
        }
        __syncthreads();
        W4_TICK(2);
        if (!more && wrp == 8) epilogue(e);
        continue;
      }
    }
    // ---- phase B: level-4 entries of this event | prep of the next one
    if (wrp < 6) w4_top<R, RC>(p, small[par], W::E4 + tid, par);
    else if (wrp < 8 && more) w4_prep<R, RC, NPASS>(p, small[par ^ 1], io, a, e + e_step, par ^ 1, wrp - 6, lane);
    __syncthreads();
    W4_TICK(0);
    // ---- phase C: top-line walk
    w4_walk<R, RC, NPASS>(p, small[par], xs, a, par, tid);
    __syncthreads();
    W4_TICK(1);
    if (a.dbg && e == 0)                                    // diagnostics only (trex_debug_xtile)
      for (int i = tid; i < W::NC * G::NCOLT; i += W::TB) {
        const int row = i / G::NCOLT, col = i - row * G::NCOLT;
        const cx<RC> x = xs[row * W::XS + col];
        a.dbg[2 * i] = (double)x.re; a.dbg[2 * i + 1] = (double)x.im;
      }
    // ---- phase D: colour sum of this event | level 3 of the next one. With the colour sum on the tensor cores three
    // warps take it (384 mma for 32 column blocks) while the other nine build the 96 level-3 entries and the U2 states of
    // the next event on the FP64 pipe -- the two pipes work side by side; the FMA colour sum (mixed / fp32 modes) is done
    // by all warps before they turn to level 3.
    if constexpr (G::DMMA || G::TF32) {
      if (wrp < W::NCW) colour_phase<R, RC, 4>(xs, Cs, part, tid, tid, W::NCW);
      else if (more) w4_build3<R, RC, NPASS>(p, small[par ^ 1], a, par ^ 1, tid - 32 * W::NCW, W::TB - 32 * W::NCW);
    } else {
      colour_phase<R, RC, 4>(xs, Cs, part, tid, tid);
      if (more) w4_build3<R, RC, NPASS>(p, small[par ^ 1], a, par ^ 1, tid, W::TB);
    }
    __syncthreads();
    W4_TICK(2);
    // ---- fixed-order reduction of the partial sums (slot parity = theta) + epilogue by warp 8, which has nothing to do
    // in phase B and clears what it has read; the other warps already work on the next event
    if (wrp == 8) epilogue(e);
    W4_TICK(3);
  }
#ifdef TREX_PHASE_CLOCKS
  if (tid == 0 && blockIdx.x == 0) printf("k_table4w phases [cycles of block 0]: B (level 4 | prep) %lld  C (walk) %lld  D (colour | level 3) %lld  epilogue %lld\n", pc[0], pc[1], pc[2], pc[3]);
#endif
}
