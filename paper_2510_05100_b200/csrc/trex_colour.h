// trex_colour.h -- host-side construction of the colour matrices.
//
// C_{sigma sigma'} = sum over adjoint indices of tr(T^{a_s1} .. T^{a_sn} T^{a_s'n} .. T^{a_s'1}),  tr(T^a T^b) = delta^{ab}/2,
// evaluated by repeated use of the SU(3) Fierz identity
//     T^a_{ij} T^a_{kl} = 1/2 ( d_il d_kj - 1/3 d_ij d_kl )
//  => tr(T^a X T^a Y) = 1/2 [ tr X tr Y - 1/3 tr(XY) ],   tr(T^a X) tr(T^a Y) = 1/2 [ tr(XY) - 1/3 tr X tr Y ],
// in exact rational arithmetic (no generator matrices are ever written down). Orderings are enumerated in
// lexicographic order, which is the order in which the prefix walk of trex_ttng.cuh reaches its leaves.
#pragma once
#include <algorithm>
#include <cstdint>
#include <numeric>
#include <vector>

namespace trex_colour {

struct Frac {
  int64_t n, d;
  Frac(int64_t n_ = 0, int64_t d_ = 1) : n(n_), d(d_) { norm(); }
  void norm() { int64_t g = std::gcd(n < 0 ? -n : n, d); if (g > 1) { n /= g; d /= g; } if (d < 0) { n = -n; d = -d; } }
  Frac operator+(const Frac& o) const { return Frac(n * o.d + o.n * d, d * o.d); }
  Frac operator-(const Frac& o) const { return Frac(n * o.d - o.n * d, d * o.d); }
  Frac operator*(const Frac& o) const { return Frac(n * o.n, d * o.d); }
  double value() const { return (double)n / (double)d; }
};

using Word = std::vector<int>;            // cyclic string of adjoint labels inside one trace

// value of a product of traces in which every label occurs exactly twice
inline Frac reduce(std::vector<Word> traces) {
  Frac pref(1, 1);
  for (;;) {
    size_t t0 = traces.size();
    for (size_t t = 0; t < traces.size(); ++t) {
      if (traces[t].size() == 1) return Frac(0, 1);      // tr T^a = 0
      if (!traces[t].empty() && t0 == traces.size()) t0 = t;
    }
    if (t0 == traces.size()) {                            // only empty traces left: tr 1 = 3 each
      for (size_t t = 0; t < traces.size(); ++t) pref = pref * Frac(3, 1);
      return pref;
    }
    Word w = traces[t0];
    const int a = w[0];
    // second occurrence in the same trace?
    auto it = std::find(w.begin() + 1, w.end(), a);
    std::vector<Word> rest;
    for (size_t t = 0; t < traces.size(); ++t) if (t != t0) rest.push_back(traces[t]);
    if (it != w.end()) {
      Word X(w.begin() + 1, it), Y(it + 1, w.end());
      std::vector<Word> A = rest, B = rest;
      A.push_back(X); A.push_back(Y);
      Word XY = X; XY.insert(XY.end(), Y.begin(), Y.end()); B.push_back(XY);
      return pref * Frac(1, 2) * (reduce(A) - Frac(1, 3) * reduce(B));
    }
    // in another trace
    for (size_t t = 0; t < rest.size(); ++t) {
      auto jt = std::find(rest[t].begin(), rest[t].end(), a);
      if (jt == rest[t].end()) continue;
      Word X(w.begin() + 1, w.end());
      Word Y(jt + 1, rest[t].end()); Y.insert(Y.end(), rest[t].begin(), jt);   // rotate so that a leads, drop it
      std::vector<Word> base;
      for (size_t s = 0; s < rest.size(); ++s) if (s != t) base.push_back(rest[s]);
      std::vector<Word> A = base, B = base;
      Word XY = X; XY.insert(XY.end(), Y.begin(), Y.end()); A.push_back(XY);
      B.push_back(X); B.push_back(Y);
      return pref * Frac(1, 2) * (reduce(A) - Frac(1, 3) * reduce(B));
    }
    return Frac(0, 1);   // unreachable for well-formed input
  }
}

inline std::vector<std::vector<int>> orderings(int n) {
  std::vector<int> p(n); std::iota(p.begin(), p.end(), 0);
  std::vector<std::vector<int>> out;
  do out.push_back(p); while (std::next_permutation(p.begin(), p.end()));
  return out;
}

// full n! x n! matrix, row-major
inline std::vector<double> ttng_colour_matrix(int n) {
  auto ord = orderings(n);
  const int nc = (int)ord.size();
  std::vector<double> C((size_t)nc * nc);
  // the entry depends only on sigma^-1 o sigma': reduce one row, then relabel
  std::vector<double> row(nc);
  for (int j = 0; j < nc; ++j) {
    Word w(ord[0].begin(), ord[0].end());
    for (int k = n - 1; k >= 0; --k) w.push_back(ord[j][k]);
    row[j] = reduce({w}).value();
  }
  auto index_of = [&](const std::vector<int>& p) { return (int)(std::lower_bound(ord.begin(), ord.end(), p) - ord.begin()); };
  for (int i = 0; i < nc; ++i) {
    std::vector<int> inv(n);
    for (int k = 0; k < n; ++k) inv[ord[i][k]] = k;
    for (int j = 0; j < nc; ++j) {
      std::vector<int> rel(n);
      for (int k = 0; k < n; ++k) rel[k] = inv[ord[j][k]];
      C[(size_t)i * nc + j] = row[index_of(rel)];
    }
  }
  return C;
}

// One light line + t t~ + two gluons (trex_qq2.cuh): twelve flows. With (S1, S2) one of
//   0 (ab, -), 1 (ba, -), 2 (a, b), 3 (b, a), 4 (-, ab), 5 (-, ba)
// type I (flows 0..5) is (S1)_{t k} (S2)_{r tb}, type II (flows 6..11) is (S1)_{t tb} (S2)_{r k}. T^a is hermitian, so the
// conjugate of a string is the reversed string with its indices swapped, and the sums over all colours are
//   I  x I'  : tr(S1 rev S1') tr(S2 rev S2')        II x II' : the same
//   I  x II' : tr(S1 rev S2' S2 rev S1')
inline std::vector<double> qq2_colour_matrix() {
  const Word s1[6] = {{0, 1}, {1, 0}, {0}, {1}, {}, {}}, s2[6] = {{}, {}, {1}, {0}, {0, 1}, {1, 0}};
  auto rev = [](Word w) { std::reverse(w.begin(), w.end()); return w; };
  auto cat = [](std::initializer_list<Word> ws) { Word o; for (const Word& w : ws) o.insert(o.end(), w.begin(), w.end()); return o; };
  std::vector<double> C(144);
  for (int i = 0; i < 12; ++i)
    for (int j = 0; j < 12; ++j) {
      const int p = i % 6, q = j % 6;
      Frac v;
      if ((i < 6) == (j < 6)) v = reduce({cat({s1[p], rev(s1[q])}), cat({s2[p], rev(s2[q])})});
      else if (i < 6) v = reduce({cat({s1[p], rev(s2[q]), s2[p], rev(s1[q])})});
      else v = reduce({cat({s1[q], rev(s2[p]), s2[q], rev(s1[p])})});
      C[i * 12 + j] = v.value();
    }
  return C;
}

}  // namespace trex_colour
