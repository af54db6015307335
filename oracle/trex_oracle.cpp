// trex_oracle.cpp -- TEST INFRASTRUCTURE ONLY (CPU oracle). Never linked or imported by the product path.
//
// A plain, slow, from-scratch evaluator of what the hot path computes (eqs.(2)-(5)):
//     w' = w * |M(p; theta_new)|^2 / |M(p; theta_old)|^2 ,   with the zero guard of PAPER.md:789-799,
// where |M|^2 is the LO tree-level, helicity- and colour-summed, initial-state averaged squared matrix
// element ("helicity-summed"). The paper delegates the amplitude itself to external routines
// (PAPER.md:994, 1221, 1269), so the Feynman rules below are the textbook ones, fixed as readings R-1..R-9 in
// DESIGN.md section 3 (= SURVEY.md 8(c) C-1..C-6). Everything is written with explicit 4x4 Dirac matrices and
// explicit SU(3) generators so that it can be checked against a textbook by eye; nothing here is tuned.
//
// Engines:
//   eemumu : e- e+ -> mu- mu+ via s-channel photon + Z, direct helicity sum            (R-5)
//   E1     : g g -> t t~ + (n-2) g by colour-ordered (Berends-Giele type) recursion,
//            A_sigma for all n! orderings, then  sum_hel A^dagger C A / N_avg              (R-6)
//   E2     : colour-dressed brute force with EXPLICIT colour indices on every line, summing
//            |M|^2 over all external colour assignments; also handles one light-quark line
//            (q q~ -> t t~ g and crossings).                                              (R-7, R-8)
// The top-quark line carries dual numbers (order 0 and order 1 in kappa = c_tG v/(sqrt2 Lambda^2)): at most one
// chromomagnetic insertion per amplitude (R-4), so |M|^2 = A + kappa B + kappa^2 D exactly.
//
// Pins (tests/test_oracle_*.py, run with -m "not gpu"): closed forms for e+e- -> mu+mu-, gg -> tt~ (SM and the
// linear c_tG term), q q~ -> t t~; completeness/Dirac equation of the spinors; transversality of the
// polarisations; Ward identity; Lorentz invariance; exact quadratic c_tG dependence; E1 == E2; colour-matrix
// entries vs. their known values; diagram-independent brute-force colour sums.
//
// Build: g++ -O2 -fopenmp -shared -fPIC (see oracle/build.py). Templated on the real type: `double`
// (timed as the CPU baseline) and `long double` (adjudicator when GPU and double oracle disagree).

#include <array>
#include <cmath>
#include <atomic>
#include <complex>
#include <cstdint>
#include <cstring>
#include <map>
#include <mutex>
#include <vector>
#include <algorithm>
#include <numeric>

namespace {

// ---------------------------------------------------------------- counting scalar (flop count (iii))
// Instantiating the evaluator on this type tallies every real addition / subtraction, multiplication, division and
// square root the plain algorithm performs: "FLOPs per event counted from the oracle" (BASELINE.json north star).
struct Count {
  double v;
  static std::atomic<long long> n_add, n_mul, n_div, n_sqrt;
  Count() : v(0) {}
  Count(double x) : v(x) {}
  Count(long double x) : v((double)x) {}
  Count(int x) : v(x) {}
  explicit operator double() const { return v; }
  Count operator-() const { return Count(-v); }
  Count& operator+=(Count o) { ++n_add; v += o.v; return *this; }
  Count& operator-=(Count o) { ++n_add; v -= o.v; return *this; }
  Count& operator*=(Count o) { ++n_mul; v *= o.v; return *this; }
  Count& operator/=(Count o) { ++n_div; v /= o.v; return *this; }
};
std::atomic<long long> Count::n_add{0}, Count::n_mul{0}, Count::n_div{0}, Count::n_sqrt{0};
inline Count operator+(Count a, Count b) { return a += b; }
inline Count operator-(Count a, Count b) { return a -= b; }
inline Count operator*(Count a, Count b) { return a *= b; }
inline Count operator/(Count a, Count b) { return a /= b; }
inline bool operator==(Count a, Count b) { return a.v == b.v; }
inline bool operator!=(Count a, Count b) { return a.v != b.v; }
inline bool operator<(Count a, Count b) { return a.v < b.v; }
inline bool operator>(Count a, Count b) { return a.v > b.v; }
inline bool operator<=(Count a, Count b) { return a.v <= b.v; }
inline bool operator>=(Count a, Count b) { return a.v >= b.v; }
inline Count osqrt(Count x) { ++Count::n_sqrt; return Count(std::sqrt(x.v)); }
inline Count oacos(Count x) { return Count(std::acos(x.v)); }
template <class T> T osqrt(T x) { return std::sqrt(x); }
template <class T> T oacos(T x) { return std::acos(x); }

constexpr int NTHETA = 16;
enum { TH_ALPHA_S = 0, TH_ALPHA_EM, TH_SIN2W, TH_MZ, TH_GAMMAZ, TH_MT, TH_GAMMAT, TH_CTG, TH_LAMBDA, TH_VEV };

template <class R> using Cx = std::complex<R>;
template <class R> using Spinor = std::array<Cx<R>, 4>;   // column or row, by context
template <class R> using Vec4 = std::array<Cx<R>, 4>;     // upper-index Lorentz vector (E,x,y,z)
template <class R> using Mat4 = std::array<std::array<Cx<R>, 4>, 4>;

template <class R> R pi_() { return oacos(R(-1)); }
const int METRIC[4] = {1, -1, -1, -1};

// ---------------------------------------------------------------- Dirac algebra (chiral basis, R-1)
template <class R> struct Dirac {
  Mat4<R> g[4];          // gamma^mu
  Mat4<R> g5, PL, PR, one;
  Mat4<R> sig[4][4];     // sigma^{mu nu} = (i/2)[gamma^mu, gamma^nu]
  Dirac() {
    const Cx<R> I(0, 1);
    for (auto& m : g) for (auto& r : m) r.fill(Cx<R>(0));
    for (auto& r : g5) r.fill(Cx<R>(0));
    for (auto& r : one) r.fill(Cx<R>(0));
    // gamma^0 = [[0,1],[1,0]]
    g[0][0][2] = g[0][1][3] = g[0][2][0] = g[0][3][1] = 1;
    // gamma^i = [[0,sigma^i],[-sigma^i,0]]
    const Cx<R> Z(R(0)), E(R(1));
    Cx<R> s[3][2][2] = {{{Z, E}, {E, Z}}, {{Z, -I}, {I, Z}}, {{E, Z}, {Z, -E}}};
    for (int i = 0; i < 3; ++i)
      for (int a = 0; a < 2; ++a)
        for (int b = 0; b < 2; ++b) {
          g[i + 1][a][2 + b] = s[i][a][b];
          g[i + 1][2 + a][b] = -s[i][a][b];
        }
    g5[0][0] = g5[1][1] = -1; g5[2][2] = g5[3][3] = 1;
    for (int a = 0; a < 4; ++a) one[a][a] = 1;
    for (int a = 0; a < 4; ++a)
      for (int b = 0; b < 4; ++b) {
        PL[a][b] = (one[a][b] - g5[a][b]) / R(2);
        PR[a][b] = (one[a][b] + g5[a][b]) / R(2);
      }
    for (int m = 0; m < 4; ++m)
      for (int n = 0; n < 4; ++n)
        for (int a = 0; a < 4; ++a)
          for (int b = 0; b < 4; ++b) {
            Cx<R> c(R(0));
            for (int k = 0; k < 4; ++k) c += g[m][a][k] * g[n][k][b] - g[n][a][k] * g[m][k][b];
            sig[m][n][a][b] = I * c / R(2);
          }
  }
};
template <class R> const Dirac<R>& dirac() { static const Dirac<R> d; return d; }

template <class R> Mat4<R> mzero() { Mat4<R> m; for (auto& r : m) r.fill(Cx<R>(0)); return m; }
template <class R> Mat4<R> madd(const Mat4<R>& a, const Mat4<R>& b) {
  Mat4<R> m; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) m[i][j] = a[i][j] + b[i][j]; return m; }
template <class R> Mat4<R> mscale(const Mat4<R>& a, Cx<R> s) {
  Mat4<R> m; for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) m[i][j] = a[i][j] * s; return m; }
template <class R> Mat4<R> mmul(const Mat4<R>& a, const Mat4<R>& b) {
  Mat4<R> m = mzero<R>();
  for (int i = 0; i < 4; ++i) for (int k = 0; k < 4; ++k) for (int j = 0; j < 4; ++j) m[i][j] += a[i][k] * b[k][j];
  return m; }
// row spinor times matrix, matrix times column spinor, row times column
template <class R> Spinor<R> rowmul(const Spinor<R>& r, const Mat4<R>& m) {
  Spinor<R> o; o.fill(Cx<R>(0)); for (int j = 0; j < 4; ++j) for (int i = 0; i < 4; ++i) o[j] += r[i] * m[i][j]; return o; }
template <class R> Spinor<R> colmul(const Mat4<R>& m, const Spinor<R>& c) {
  Spinor<R> o; o.fill(Cx<R>(0)); for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) o[i] += m[i][j] * c[j]; return o; }
template <class R> Cx<R> rowcol(const Spinor<R>& r, const Spinor<R>& c) {
  Cx<R> s(R(0)); for (int i = 0; i < 4; ++i) s += r[i] * c[i]; return s; }
template <class R> Spinor<R> sadd(const Spinor<R>& a, const Spinor<R>& b) {
  Spinor<R> o; for (int i = 0; i < 4; ++i) o[i] = a[i] + b[i]; return o; }
template <class R> Spinor<R> szero() { Spinor<R> o; o.fill(Cx<R>(0)); return o; }

// Minkowski product WITHOUT complex conjugation, both vectors with upper indices
template <class R> Cx<R> mdot(const Vec4<R>& a, const Vec4<R>& b) {
  return a[0] * b[0] - a[1] * b[1] - a[2] * b[2] - a[3] * b[3]; }
template <class R> Vec4<R> vadd(const Vec4<R>& a, const Vec4<R>& b) {
  Vec4<R> o; for (int i = 0; i < 4; ++i) o[i] = a[i] + b[i]; return o; }
template <class R> Vec4<R> vsub(const Vec4<R>& a, const Vec4<R>& b) {
  Vec4<R> o; for (int i = 0; i < 4; ++i) o[i] = a[i] - b[i]; return o; }
template <class R> Vec4<R> vscale(const Vec4<R>& a, Cx<R> s) {
  Vec4<R> o; for (int i = 0; i < 4; ++i) o[i] = a[i] * s; return o; }
template <class R> bool vis_zero(const Vec4<R>& a) { for (int i = 0; i < 4; ++i) if (a[i] != Cx<R>(0)) return false; return true; }
template <class R> Vec4<R> vzero() { Vec4<R> o; o.fill(Cx<R>(0)); return o; }

// slash(a) = gamma^mu a_mu
template <class R> Mat4<R> slash(const Vec4<R>& a) {
  const auto& d = dirac<R>();
  Mat4<R> m = mzero<R>();
  for (int mu = 0; mu < 4; ++mu) m = madd(m, mscale(d.g[mu], a[mu] * R(METRIC[mu])));
  return m; }
// sigma^{mu nu} a_mu b_nu
template <class R> Mat4<R> sigma_ab(const Vec4<R>& a, const Vec4<R>& b) {
  const auto& d = dirac<R>();
  Mat4<R> m = mzero<R>();
  for (int mu = 0; mu < 4; ++mu) for (int nu = 0; nu < 4; ++nu) {
    if (mu == nu) continue;
    m = madd(m, mscale(d.sig[mu][nu], a[mu] * R(METRIC[mu]) * b[nu] * R(METRIC[nu])));
  }
  return m; }

// ---------------------------------------------------------------- external wavefunctions (R-2)
template <class R> struct Chi { Cx<R> plus[2], minus[2]; };
template <class R> Chi<R> two_spinors(const R p[4]) {
  Chi<R> c;
  R pt2 = p[1] * p[1] + p[2] * p[2];
  R pabs = osqrt(pt2 + p[3] * p[3]);
  // |p| + pz, evaluated without cancellation when pz < 0
  R ppz = p[3] >= R(0) ? pabs + p[3] : pt2 / (pabs - p[3]);
  if (pabs == R(0)) {           // at rest: the pz -> +0 limit
    c.plus[0] = 1; c.plus[1] = 0; c.minus[0] = 0; c.minus[1] = 1; return c;
  }
  if (ppz == R(0)) {            // exactly along -z
    c.plus[0] = 0; c.plus[1] = 1; c.minus[0] = -1; c.minus[1] = 0; return c;
  }
  R N = R(1) / osqrt(R(2) * pabs * ppz);
  c.plus[0] = N * ppz; c.plus[1] = N * Cx<R>(p[1], p[2]);
  c.minus[0] = N * Cx<R>(-p[1], p[2]); c.minus[1] = N * ppz;
  return c; }

// u(p,lambda) = (w_{-l} chi_l ; w_l chi_l), v(p,lambda) = (-l w_l chi_{-l} ; l w_{-l} chi_{-l}), w_pm = sqrt(E pm |p|)
// `massless` legs are on shell by definition: E := |p|, so w_- = 0 exactly (R-2; sqrt(E-|p|) would
// otherwise amplify the rounding of the input momenta to a spurious 1e-8 wrong-chirality component)
template <class R> Spinor<R> spinor_u(const R p[4], int lam, bool massless = false) {
  Chi<R> c = two_spinors<R>(p);
  R pabs = osqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  R wp = osqrt(std::max(R(0), p[0] + pabs)), wm = osqrt(std::max(R(0), p[0] - pabs));
  if (massless) { wp = osqrt(R(2) * pabs); wm = 0; }
  const Cx<R>* chi = lam > 0 ? c.plus : c.minus;
  R up = lam > 0 ? wm : wp, lo = lam > 0 ? wp : wm;
  return Spinor<R>{up * chi[0], up * chi[1], lo * chi[0], lo * chi[1]}; }
template <class R> Spinor<R> spinor_v(const R p[4], int lam, bool massless = false) {
  Chi<R> c = two_spinors<R>(p);
  R pabs = osqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  R wp = osqrt(std::max(R(0), p[0] + pabs)), wm = osqrt(std::max(R(0), p[0] - pabs));
  if (massless) { wp = osqrt(R(2) * pabs); wm = 0; }
  const Cx<R>* chi = lam > 0 ? c.minus : c.plus;   // chi_{-lambda}
  R up = lam > 0 ? -wp : wm, lo = lam > 0 ? wm : -wp;
  return Spinor<R>{up * chi[0], up * chi[1], lo * chi[0], lo * chi[1]}; }
// bar(psi) = psi^dagger gamma^0 (as a row)
template <class R> Spinor<R> bar(const Spinor<R>& s) {
  const auto& d = dirac<R>();
  Spinor<R> cj; for (int i = 0; i < 4; ++i) cj[i] = std::conj(s[i]);
  return rowmul(cj, d.g[0]); }
// eps(p,lambda) = (-lambda e1 - i e2)/sqrt2 for a massless vector
template <class R> Vec4<R> polvec(const R p[4], int lam) {
  R pt = osqrt(p[1] * p[1] + p[2] * p[2]);
  R pabs = osqrt(pt * pt + p[3] * p[3]);
  R e1[4], e2[4];
  if (pt < R(1e-14) * pabs || pt == R(0)) {
    R sg = p[3] >= 0 ? R(1) : R(-1);
    e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
    e2[0] = 0; e2[1] = 0; e2[2] = sg; e2[3] = 0;
  } else {
    e1[0] = 0; e1[1] = p[1] * p[3] / (pabs * pt); e1[2] = p[2] * p[3] / (pabs * pt); e1[3] = -pt / pabs;
    e2[0] = 0; e2[1] = -p[2] / pt; e2[2] = p[1] / pt; e2[3] = 0;
  }
  const R rs2 = R(1) / osqrt(R(2));
  Vec4<R> e;
  for (int i = 0; i < 4; ++i) e[i] = Cx<R>(-R(lam) * e1[i], -e2[i]) * rs2;
  return e; }
template <class R> Vec4<R> vconj(const Vec4<R>& a) { Vec4<R> o; for (int i = 0; i < 4; ++i) o[i] = std::conj(a[i]); return o; }
template <class R> Vec4<R> realvec(const R p[4], R sign) { Vec4<R> o; for (int i = 0; i < 4; ++i) o[i] = Cx<R>(sign * p[i], 0); return o; }

// ---------------------------------------------------------------- SU(3) (R-3): T^a = lambda^a/2, f^{abc}
struct SU3 {
  std::complex<double> T[8][3][3];
  double f[8][8][8];
  SU3() {
    using C = std::complex<double>;
    std::memset(T, 0, sizeof T);
    const C I(0, 1);
    T[0][0][1] = T[0][1][0] = 0.5;
    T[1][0][1] = -0.5 * I; T[1][1][0] = 0.5 * I;
    T[2][0][0] = 0.5; T[2][1][1] = -0.5;
    T[3][0][2] = T[3][2][0] = 0.5;
    T[4][0][2] = -0.5 * I; T[4][2][0] = 0.5 * I;
    T[5][1][2] = T[5][2][1] = 0.5;
    T[6][1][2] = -0.5 * I; T[6][2][1] = 0.5 * I;
    double s3 = 1.0 / osqrt(3.0);
    T[7][0][0] = T[7][1][1] = 0.5 * s3; T[7][2][2] = -s3;
    // f^{abc} = -2i tr([T^a,T^b] T^c)
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
      C tr = 0;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k)
        tr += (T[a][i][j] * T[b][j][k] - T[b][i][j] * T[a][j][k]) * T[c][k][i];
      f[a][b][c] = (C(0, -2) * tr).real();
    }
  }
};
const SU3& su3() { static const SU3 s; return s; }

// C_{sigma sigma'} = sum_{a_1..a_n} tr(T^{a_s1}...T^{a_sn} T^{a_s'n}...T^{a_s'1})  by explicit Gell-Mann contraction.
// Only the row sigma = identity is computed by brute force; C_{sigma sigma'} = C_{id, sigma^-1 o sigma'} follows from
// relabelling the summed indices (R-6). Permutations in lexicographic order.
std::vector<std::vector<int>> all_perms(int n) {
  std::vector<int> p(n); std::iota(p.begin(), p.end(), 0);
  std::vector<std::vector<int>> out;
  do out.push_back(p); while (std::next_permutation(p.begin(), p.end()));
  return out; }

double colour_entry_bruteforce(int n, const std::vector<int>& s, const std::vector<int>& sp) {
  using C = std::complex<double>;
  const SU3& g = su3();
  long ncfg = 1; for (int i = 0; i < n; ++i) ncfg *= 8;
  C total = 0;
  std::vector<int> a(n);
  for (long cfg = 0; cfg < ncfg; ++cfg) {
    long c = cfg; for (int i = 0; i < n; ++i) { a[i] = c % 8; c /= 8; }
    C M[3][3] = {{1, 0, 0}, {0, 1, 0}, {0, 0, 1}}, N[3][3];
    auto mul = [&](int gen) {
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { N[i][j] = 0; for (int k = 0; k < 3; ++k) N[i][j] += M[i][k] * g.T[gen][k][j]; }
      std::memcpy(M, N, sizeof M); };
    for (int i = 0; i < n; ++i) mul(a[s[i]]);
    for (int i = n - 1; i >= 0; --i) mul(a[sp[i]]);
    total += M[0][0] + M[1][1] + M[2][2];
  }
  return total.real(); }

const std::vector<double>& colour_matrix(int n) {   // n! x n!, row-major, lexicographic permutation order
  static std::map<int, std::vector<double>> cache;
  static std::mutex mtx;
  std::lock_guard<std::mutex> lk(mtx);
  auto it = cache.find(n);
  if (it != cache.end()) return it->second;
  auto perms = all_perms(n);
  int np = (int)perms.size();
  std::map<std::vector<int>, int> index;
  for (int i = 0; i < np; ++i) index[perms[i]] = i;
  std::vector<double> row(np);
  #pragma omp parallel for schedule(dynamic)
  for (int j = 0; j < np; ++j) row[j] = colour_entry_bruteforce(n, perms[0], perms[j]);
  std::vector<double> C((size_t)np * np);
  for (int i = 0; i < np; ++i) {
    std::vector<int> inv(n); for (int k = 0; k < n; ++k) inv[perms[i][k]] = k;
    for (int j = 0; j < np; ++j) {
      std::vector<int> comp(n); for (int k = 0; k < n; ++k) comp[k] = inv[perms[j][k]];
      C[(size_t)i * np + j] = row[index[comp]];
    }
  }
  return cache[n] = C; }

// ---------------------------------------------------------------- parameters
template <class R> struct Params {
  R gs, ee, sw2, mZ, GZ, mt, Gt, kappa;
  explicit Params(const double* th) {
    gs = osqrt(R(4) * pi_<R>() * R(th[TH_ALPHA_S]));
    ee = osqrt(R(4) * pi_<R>() * R(th[TH_ALPHA_EM]));
    sw2 = th[TH_SIN2W]; mZ = th[TH_MZ]; GZ = th[TH_GAMMAZ]; mt = th[TH_MT]; Gt = th[TH_GAMMAT];
    kappa = R(th[TH_CTG]) * R(th[TH_VEV]) / (osqrt(R(2)) * R(th[TH_LAMBDA]) * R(th[TH_LAMBDA]));
  }
};

// dual number on the top line: value = o0 + kappa * o1, kappa^2 dropped (R-4)
template <class R> struct DualSpinor { Spinor<R> o0, o1; };
template <class R> struct DualC { Cx<R> o0, o1; };

// fermion propagator i(qslash + m)/(q^2 - m^2 + i m Gamma)   (R-3: width in the denominator only)
template <class R> Mat4<R> fermion_prop(const Vec4<R>& q, R m, R G) {
  const auto& d = dirac<R>();
  Cx<R> den = mdot(q, q) - m * m + Cx<R>(0, m * G);
  return mscale(madd(slash(q), mscale(d.one, Cx<R>(m))), Cx<R>(0, 1) / den); }

// top-gluon vertex Gamma(J,q) = i g_s Jslash  +  kappa * 2 sigma^{mu nu} q_mu J_nu  (q = gluon momentum INTO the vertex)
template <class R> void vertex_ttg(const Params<R>& P, const Vec4<R>& J, const Vec4<R>& q, Mat4<R>& g0, Mat4<R>& g1) {
  g0 = mscale(slash(J), Cx<R>(0, P.gs));
  g1 = mscale(sigma_ab(q, J), Cx<R>(2)); }
// ttgg contact, ordered (T^b T^c coefficient): kappa * 2 g_s sigma^{mu nu} J1_mu J2_nu
template <class R> Mat4<R> vertex_ttgg(const Params<R>& P, const Vec4<R>& J1, const Vec4<R>& J2) {
  return mscale(sigma_ab(J1, J2), Cx<R>(R(2) * P.gs)); }

// ordered 3- and 4-gluon Lorentz structures (R-6)
template <class R> Vec4<R> V3(const Vec4<R>& k1, const Vec4<R>& J1, const Vec4<R>& k2, const Vec4<R>& J2) {
  Vec4<R> P = vadd(k1, k2), o;
  Vec4<R> a = vscale(vadd(P, k1), Cx<R>(-1));   // -P - k1
  Vec4<R> b = vadd(k2, P);                      //  k2 + P
  Vec4<R> d = vsub(k1, k2);
  Cx<R> aJ2 = mdot(a, J2), J1J2 = mdot(J1, J2), bJ1 = mdot(b, J1);
  for (int m = 0; m < 4; ++m) o[m] = J1[m] * aJ2 + d[m] * J1J2 + J2[m] * bJ1;
  return o; }
template <class R> Vec4<R> V4(const Vec4<R>& J1, const Vec4<R>& J2, const Vec4<R>& J3) {
  Cx<R> d23 = mdot(J2, J3), d12 = mdot(J1, J2), d13 = mdot(J1, J3);
  Vec4<R> o;
  for (int m = 0; m < 4; ++m) o[m] = J1[m] * d23 + J3[m] * d12 - R(2) * J2[m] * d13;
  return o; }

// ---------------------------------------------------------------- event view
template <class R> struct Event {
  int npar; R p[8][4];
  Event(const double* mom, long n, long i, int npar_) : npar(npar_) {
    for (int a = 0; a < npar; ++a) for (int mu = 0; mu < 4; ++mu) p[a][mu] = R(mom[((long)a * 4 + mu) * n + i]);
  }
};
inline int hel_of(int h, int leg) { return ((h >> leg) & 1) ? +1 : -1; }

// ================================================================= engine: e- e+ -> mu- mu+  (R-5)
template <class R> R eemumu_me2(const Event<R>& ev, const Params<R>& P) {
  const auto& d = dirac<R>();
  R s = 0;
  { R q[4]; for (int m = 0; m < 4; ++m) q[m] = ev.p[0][m] + ev.p[1][m]; s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3]; }
  R cw2 = R(1) - P.sw2, sc = osqrt(P.sw2 * cw2);
  R gL = P.ee / sc * (R(-0.5) + P.sw2), gR = P.ee / sc * P.sw2;
  Mat4<R> GZ = madd(mscale(d.PL, Cx<R>(gL)), mscale(d.PR, Cx<R>(gR)));
  const Cx<R> I(0, 1);
  Cx<R> prop_a = -I / s, prop_z = -I / (Cx<R>(s - P.mZ * P.mZ, P.mZ * P.GZ));
  R sum = 0;
  for (int h = 0; h < 16; ++h) {
    Spinor<R> u1 = spinor_u<R>(ev.p[0], hel_of(h, 0), true);      // incoming e-
    Spinor<R> vb2 = bar(spinor_v<R>(ev.p[1], hel_of(h, 1), true)); // incoming e+
    Spinor<R> ub3 = bar(spinor_u<R>(ev.p[2], hel_of(h, 2), true)); // outgoing mu-
    Spinor<R> v4 = spinor_v<R>(ev.p[3], hel_of(h, 3), true);       // outgoing mu+
    Cx<R> M(R(0));
    for (int mu = 0; mu < 4; ++mu) {
      Mat4<R> va = mscale(d.g[mu], I * P.ee);                     // i e gamma^mu
      Mat4<R> vz = mscale(mmul(d.g[mu], GZ), I);                  // i gamma^mu (gL PL + gR PR)
      Cx<R> ea = rowcol(vb2, colmul(va, u1)), ma = rowcol(ub3, colmul(va, v4));
      Cx<R> ez = rowcol(vb2, colmul(vz, u1)), mz = rowcol(ub3, colmul(vz, v4));
      M += R(METRIC[mu]) * (ea * prop_a * ma + ez * prop_z * mz);
    }
    sum += std::norm(M);
  }
  return sum / R(4); }

// ================================================================= engine E1: colour-ordered recursion (R-6)
template <class R> struct TTNG {
  int n;                                  // number of gluons
  std::vector<int> gl_leg;                // gluon index -> leg index in process order g g t t~ g...
  Vec4<R> K[8], eps[8];                   // incoming-convention momenta, polarisations (eps* for outgoing)
  Vec4<R> pt; Spinor<R> ubar_t, v_tb;
  const Params<R>& P;
  std::map<uint32_t, Vec4<R>> memoJ;
  std::map<uint32_t, DualSpinor<R>> memoU;

  TTNG(const Event<R>& ev, const Params<R>& P_, int h, int gauge_gluon) : P(P_) {
    n = ev.npar - 2;
    gl_leg = {0, 1}; for (int l = 4; l < ev.npar; ++l) gl_leg.push_back(l);
    for (int g = 0; g < n; ++g) {
      int leg = gl_leg[g]; bool incoming = leg < 2;
      K[g] = realvec<R>(ev.p[leg], incoming ? R(1) : R(-1));
      Vec4<R> e = polvec<R>(ev.p[leg], hel_of(h, leg));
      eps[g] = incoming ? e : vconj(e);
      if (g == gauge_gluon) eps[g] = K[g];             // Ward-identity probe
    }
    pt = realvec<R>(ev.p[2], R(1));
    ubar_t = bar(spinor_u<R>(ev.p[2], hel_of(h, 2)));  // outgoing top
    v_tb = spinor_v<R>(ev.p[3], hel_of(h, 3));         // outgoing antitop
  }
  static uint32_t code(const int* t, int len) { uint32_t c = len; for (int i = 0; i < len; ++i) c = c * 8 + t[i]; return c; }
  Vec4<R> Psum(const int* t, int len) const { Vec4<R> s = vzero<R>(); for (int i = 0; i < len; ++i) s = vadd(s, K[t[i]]); return s; }

  // J(t_0..t_{len-1})
  Vec4<R> J(const int* t, int len) {
    if (len == 1) return eps[t[0]];
    uint32_t c = code(t, len);
    auto it = memoJ.find(c); if (it != memoJ.end()) return it->second;
    const Cx<R> I(0, 1);
    Vec4<R> acc = vzero<R>();
    for (int m = 1; m < len; ++m)
      acc = vadd(acc, vscale(V3(Psum(t, m), J(t, m), Psum(t + m, len - m), J(t + m, len - m)), -I * P.gs));
    for (int m1 = 1; m1 < len; ++m1) for (int m2 = m1 + 1; m2 < len; ++m2)
      acc = vadd(acc, vscale(V4(J(t, m1), J(t + m1, m2 - m1), J(t + m2, len - m2)), -I * P.gs * P.gs));
    Vec4<R> Pt = Psum(t, len);
    Vec4<R> out = vscale(acc, -I / mdot(Pt, Pt));
    memoJ[c] = out; return out; }

  // bracket of (R-6): sum_a Ubar(a) Gamma(J(a+1..m)) + sum_{a<b} Ubar0(a) Gamma_c(J(a+1..b), J(b+1..m)), no propagator
  DualSpinor<R> bracket(const int* t, int m) {
    DualSpinor<R> acc{szero<R>(), szero<R>()};
    for (int a = 0; a < m; ++a) {
      DualSpinor<R> Ua = Ubar(t, a);
      Mat4<R> g0, g1; vertex_ttg(P, J(t + a, m - a), Psum(t + a, m - a), g0, g1);
      acc.o0 = sadd(acc.o0, rowmul(Ua.o0, g0));
      acc.o1 = sadd(acc.o1, sadd(rowmul(Ua.o1, g0), rowmul(Ua.o0, g1)));
    }
    for (int a = 0; a < m; ++a) for (int b = a + 1; b < m; ++b) {
      DualSpinor<R> Ua = Ubar(t, a);
      acc.o1 = sadd(acc.o1, rowmul(Ua.o0, vertex_ttgg(P, J(t + a, b - a), J(t + b, m - b))));
    }
    return acc; }
  // Ubar(t_0..t_{m-1}) including its propagator S(p_t - P_{1m})
  DualSpinor<R> Ubar(const int* t, int m) {
    if (m == 0) return DualSpinor<R>{ubar_t, szero<R>()};
    uint32_t c = code(t, m);
    auto it = memoU.find(c); if (it != memoU.end()) return it->second;
    DualSpinor<R> b = bracket(t, m);
    Mat4<R> S = fermion_prop<R>(vsub(pt, Psum(t, m)), P.mt, P.Gt);
    DualSpinor<R> out{rowmul(b.o0, S), rowmul(b.o1, S)};
    memoU[c] = out; return out; }
  DualC<R> amplitude(const std::vector<int>& sigma) {
    DualSpinor<R> b = bracket(sigma.data(), n);
    return DualC<R>{rowcol(b.o0, v_tb), rowcol(b.o1, v_tb)}; }
};

// me2 coefficients: me2(kappa) = A + kappa B + kappa^2 D
template <class R> struct ABD { R A, B, D; R at(R k) const { return A + k * B + k * k * D; } };

template <class R> ABD<R> ttng_abd(const Event<R>& ev, const Params<R>& P, int gauge_gluon = -1, int hel_only = -1) {
  int n = ev.npar - 2;
  auto perms = all_perms(n);
  int np = (int)perms.size();
  const std::vector<double>& C = colour_matrix(n);
  R A = 0, B = 0, D = 0;
  std::vector<DualC<R>> amp(np);
  for (int h = 0; h < (1 << ev.npar); ++h) {
    if (hel_only >= 0 && h != hel_only) continue;
    TTNG<R> t(ev, P, h, gauge_gluon);
    for (int i = 0; i < np; ++i) amp[i] = t.amplitude(perms[i]);
    for (int i = 0; i < np; ++i) for (int j = 0; j < np; ++j) {
      R c = R(C[(size_t)i * np + j]);
      A += c * (std::conj(amp[i].o0) * amp[j].o0).real();
      B += c * (std::conj(amp[i].o0) * amp[j].o1 + std::conj(amp[i].o1) * amp[j].o0).real();
      D += c * (std::conj(amp[i].o1) * amp[j].o1).real();
    }
  }
  R fact = 1; for (int k = 2; k <= n - 2; ++k) fact *= k;
  R navg = R(4) * R(64) * fact;
  return ABD<R>{A / navg, B / navg, D / navg}; }

// ================================================================= engine E2: explicit colour brute force (R-7, R-8)
// Sources: gluon legs (each with a fixed external adjoint colour) and optionally one light-quark pair "Q"
// (row end with fundamental colour k, column end with fundamental colour l).
template <class R> struct ColJ { Vec4<R> c[8]; };                       // J^{a mu}
template <class R> struct ColDS { DualSpinor<R> c[3]; };                // heavy-line state with colour index
template <class R> struct ColS { Spinor<R> c[3]; };                     // light-line state with colour index

template <class R> struct E2 {
  const Params<R>& P;
  int ns = 0;                       // number of sources
  int qsrc = -1;                    // index of the light-pair source or -1
  Vec4<R> K[8];                     // incoming-convention momentum of each source (Q: sum of both ends)
  Vec4<R> eps[8]; int gcol[8];      // gluon sources
  Vec4<R> Krow, Kcol; Spinor<R> wrow, xcol; int crow = 0, ccol = 0;   // light line
  Vec4<R> pt; Spinor<R> ubar_t, v_tb; int ctop = 0;
  std::vector<ColJ<R>> Jc; std::vector<char> haveJ;
  std::vector<ColDS<R>> Hc; std::vector<char> haveH;      // memo only (same values as recomputing)

  explicit E2(const Params<R>& P_) : P(P_) {}
  Vec4<R> Pof(int S) const { Vec4<R> s = vzero<R>(); for (int i = 0; i < ns; ++i) if (S >> i & 1) s = vadd(s, K[i]); return s; }

  // light-line states over gluon-only subsets
  ColS<R> Wrow(int S) {
    ColS<R> out; for (auto& s : out.c) s = szero<R>();
    if (S == 0) { out.c[crow] = wrow; return out; }
    const SU3& g = su3();
    for (int Sp = S; Sp; Sp = (Sp - 1) & S) {
      ColS<R> prev = Wrow(S & ~Sp); const ColJ<R>& Jp = J(Sp);
      for (int a = 0; a < 8; ++a) {
        Mat4<R> v = mscale(slash(Jp.c[a]), Cx<R>(0, P.gs));
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
          Cx<R> t((R)g.T[a][i][j].real(), (R)g.T[a][i][j].imag()); if (t == Cx<R>(0)) continue;
          Spinor<R> r = rowmul(prev.c[i], v); for (int k = 0; k < 4; ++k) out.c[j][k] += t * r[k];
        }
      }
    }
    Vec4<R> q = vsub(vscale(Krow, Cx<R>(-1)), Pof(S));
    Mat4<R> Sp_ = fermion_prop<R>(q, R(0), R(0));
    for (auto& s : out.c) s = rowmul(s, Sp_);
    return out; }
  ColS<R> Xcol(int S) {
    ColS<R> out; for (auto& s : out.c) s = szero<R>();
    if (S == 0) { out.c[ccol] = xcol; return out; }
    const SU3& g = su3();
    for (int Sp = S; Sp; Sp = (Sp - 1) & S) {
      ColS<R> prev = Xcol(S & ~Sp); const ColJ<R>& Jp = J(Sp);
      for (int a = 0; a < 8; ++a) {
        Mat4<R> v = mscale(slash(Jp.c[a]), Cx<R>(0, P.gs));
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
          Cx<R> t((R)g.T[a][i][j].real(), (R)g.T[a][i][j].imag()); if (t == Cx<R>(0)) continue;
          Spinor<R> r = colmul(v, prev.c[j]); for (int k = 0; k < 4; ++k) out.c[i][k] += t * r[k];
        }
      }
    }
    Vec4<R> q = vadd(Kcol, Pof(S));
    Mat4<R> Sp_ = fermion_prop<R>(q, R(0), R(0));
    for (auto& s : out.c) s = colmul(Sp_, s);
    return out; }

  // colour-dressed off-shell current of source subset S
  const ColJ<R>& J(int S) {
    if (haveJ[S]) return Jc[S];
    const SU3& g = su3(); const auto& d = dirac<R>();
    const Cx<R> I(0, 1);
    ColJ<R> out; for (auto& v : out.c) v = vzero<R>();
    bool single = (S & (S - 1)) == 0;
    int idx = 0; while (!(S >> idx & 1)) ++idx;
    if (single && idx != qsrc) {
      out.c[gcol[idx]] = eps[idx];
      Jc[S] = out; haveJ[S] = 1; return Jc[S];
    }
    // three-gluon vertices: unordered partitions {S1,S2}; keep the one where S1 holds the lowest set bit
    int low = S & -S;
    for (int S1 = S; S1; S1 = (S1 - 1) & S) {
      int S2 = S & ~S1; if (!S2 || !(S1 & low)) continue;
      const ColJ<R>& J1 = J(S1); const ColJ<R>& J2 = J(S2);
      Vec4<R> k1 = Pof(S1), k2 = Pof(S2);
      for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
        if (vis_zero(J1.c[b]) || vis_zero(J2.c[c])) continue;
        Vec4<R> v = V3(k1, J1.c[b], k2, J2.c[c]);
        for (int a = 0; a < 8; ++a) { R f = (R)g.f[a][b][c]; if (f == 0) continue;
          for (int m = 0; m < 4; ++m) out.c[a][m] += P.gs * f * v[m]; }
      }
    }
    // four-gluon vertices: unordered partitions {S1,S2,S3}
    for (int S1 = S; S1; S1 = (S1 - 1) & S) {
      if (!(S1 & low)) continue;
      int rest = S & ~S1; if (!rest) continue;
      int low2 = rest & -rest;
      for (int S2 = rest; S2; S2 = (S2 - 1) & rest) {
        int S3 = rest & ~S2; if (!S3 || !(S2 & low2)) continue;
        const ColJ<R>& J1 = J(S1); const ColJ<R>& J2 = J(S2); const ColJ<R>& J3 = J(S3);
        for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int dd = 0; dd < 8; ++dd) {
          Cx<R> d12 = mdot(J1.c[b], J2.c[c]), d13 = mdot(J1.c[b], J3.c[dd]), d23 = mdot(J2.c[c], J3.c[dd]);
          if (d12 == Cx<R>(0) && d13 == Cx<R>(0) && d23 == Cx<R>(0)) continue;
          for (int a = 0; a < 8; ++a) {
            R c1 = 0, c2 = 0, c3 = 0;   // f^{abe}f^{cde}, f^{ace}f^{bde}, f^{ade}f^{bce}
            for (int e = 0; e < 8; ++e) {
              c1 += (R)(g.f[a][b][e] * g.f[c][dd][e]); c2 += (R)(g.f[a][c][e] * g.f[b][dd][e]); c3 += (R)(g.f[a][dd][e] * g.f[b][c][e]);
            }
            if (c1 == 0 && c2 == 0 && c3 == 0) continue;
            for (int m = 0; m < 4; ++m) {
              Cx<R> t1 = J2.c[c][m] * d13 - J3.c[dd][m] * d12;
              Cx<R> t2 = J1.c[b][m] * d23 - J3.c[dd][m] * d12;
              Cx<R> t3 = J1.c[b][m] * d23 - J2.c[c][m] * d13;
              out.c[a][m] += -I * P.gs * P.gs * (c1 * t1 + c2 * t2 + c3 * t3);
            }
          }
        }
      }
    }
    // direct light-line emission of the off-shell gluon
    if (qsrc >= 0 && (S >> qsrc & 1)) {
      int G = S & ~(1 << qsrc);
      for (int S1 = G;; S1 = (S1 - 1) & G) {
        int S2 = G & ~S1;
        ColS<R> W = Wrow(S1), X = Xcol(S2);
        for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
          Cx<R> t((R)g.T[a][i][j].real(), (R)g.T[a][i][j].imag()); if (t == Cx<R>(0)) continue;
          for (int m = 0; m < 4; ++m)
            out.c[a][m] += t * I * P.gs * rowcol(W.c[i], colmul(d.g[m], X.c[j]));
        }
        if (S1 == 0) break;
      }
    }
    Vec4<R> Pt = Pof(S); Cx<R> pr = -I / mdot(Pt, Pt);
    for (auto& v : out.c) v = vscale(v, pr);
    Jc[S] = out; haveJ[S] = 1; return Jc[S]; }

  // heavy line bracket for subset S (no propagator) and state (with propagator)
  ColDS<R> Hbracket(int S) {
    const SU3& g = su3();
    ColDS<R> acc; for (auto& s : acc.c) { s.o0 = szero<R>(); s.o1 = szero<R>(); }
    for (int Sp = S; Sp; Sp = (Sp - 1) & S) {
      ColDS<R> prev = Hstate(S & ~Sp); const ColJ<R>& Jp = J(Sp); Vec4<R> q = Pof(Sp);
      for (int a = 0; a < 8; ++a) {
        Mat4<R> g0, g1; vertex_ttg(P, Jp.c[a], q, g0, g1);
        for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
          Cx<R> t((R)g.T[a][i][j].real(), (R)g.T[a][i][j].imag()); if (t == Cx<R>(0)) continue;
          Spinor<R> r0 = rowmul(prev.c[i].o0, g0);
          Spinor<R> r1 = sadd(rowmul(prev.c[i].o1, g0), rowmul(prev.c[i].o0, g1));
          for (int k = 0; k < 4; ++k) { acc.c[j].o0[k] += t * r0[k]; acc.c[j].o1[k] += t * r1[k]; }
        }
      }
    }
    // contact t t~ g g: 2 i kappa g_s f^{abc} T^a sigma^{mu nu} J^b_mu(S1) J^c_nu(S2), unordered disjoint {S1,S2} in S
    for (int S1 = S; S1; S1 = (S1 - 1) & S) {
      int rest = S & ~S1;
      for (int S2 = rest; S2; S2 = (S2 - 1) & rest) {
        if (S1 > S2) continue;                       // unordered pair once
        ColDS<R> prev = Hstate(S & ~S1 & ~S2); const ColJ<R>& J1 = J(S1); const ColJ<R>& J2 = J(S2);
        for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
          if (vis_zero(J1.c[b]) || vis_zero(J2.c[c])) continue;
          Mat4<R> sg = sigma_ab(J1.c[b], J2.c[c]);
          for (int a = 0; a < 8; ++a) { R f = (R)g.f[a][b][c]; if (f == 0) continue;
            for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
              Cx<R> t((R)g.T[a][i][j].real(), (R)g.T[a][i][j].imag()); if (t == Cx<R>(0)) continue;
              Spinor<R> r = rowmul(prev.c[i].o0, sg);
              for (int k = 0; k < 4; ++k) acc.c[j].o1[k] += Cx<R>(0, 2) * P.gs * f * t * r[k];
            }
          }
        }
      }
    }
    return acc; }
  ColDS<R> Hstate(int S) {
    ColDS<R> out;
    if (S == 0) { for (auto& s : out.c) { s.o0 = szero<R>(); s.o1 = szero<R>(); } out.c[ctop].o0 = ubar_t; return out; }
    if (haveH[S]) return Hc[S];
    ColDS<R> b = Hbracket(S);
    Mat4<R> Sp_ = fermion_prop<R>(vsub(pt, Pof(S)), P.mt, P.Gt);
    for (int j = 0; j < 3; ++j) { out.c[j].o0 = rowmul(b.c[j].o0, Sp_); out.c[j].o1 = rowmul(b.c[j].o1, Sp_); }
    Hc[S] = out; haveH[S] = 1; return out; }
  // amplitudes M_{ctop, j} for j = antitop colour
  void amplitudes(DualC<R> M[3]) {
    Jc.assign(1 << ns, ColJ<R>()); haveJ.assign(1 << ns, 0);
    Hc.assign(1 << ns, ColDS<R>()); haveH.assign(1 << ns, 0);
    ColDS<R> b = Hbracket((1 << ns) - 1);
    for (int j = 0; j < 3; ++j) M[j] = DualC<R>{rowcol(b.c[j].o0, v_tb), rowcol(b.c[j].o1, v_tb)};
  }
};

// subprocess kinds handled by E2
enum Kind { K_TTNG = 0, K_QQB = 1, K_QG = 2, K_GQB = 3 };   // gg->tt~+ng ; q q~->tt~g ; q g->tt~q ; g q~->tt~q~

template <class R> ABD<R> e2_abd(const Event<R>& ev, const Params<R>& P, int kind, int gauge_gluon, int hel_only) {
  R A = 0, B = 0, D = 0;
  int nh = 1 << ev.npar;
  for (int h = 0; h < nh; ++h) {
    if (hel_only >= 0 && h != hel_only) continue;
    E2<R> e(P);
    e.pt = realvec<R>(ev.p[2], R(1));
    e.ubar_t = bar(spinor_u<R>(ev.p[2], hel_of(h, 2)));
    e.v_tb = spinor_v<R>(ev.p[3], hel_of(h, 3));
    std::vector<int> gl;     // gluon legs
    if (kind == K_TTNG) { gl = {0, 1}; for (int l = 4; l < ev.npar; ++l) gl.push_back(l); }
    else if (kind == K_QQB) { for (int l = 4; l < ev.npar; ++l) gl.push_back(l); }
    else if (kind == K_QG) { gl = {1}; for (int l = 5; l < ev.npar; ++l) gl.push_back(l); }     // leg 4 is the outgoing quark
    else { gl = {0}; for (int l = 5; l < ev.npar; ++l) gl.push_back(l); }
    e.ns = 0;
    for (int leg : gl) {
      bool inc = leg < 2; int s = e.ns++;
      e.K[s] = realvec<R>(ev.p[leg], inc ? R(1) : R(-1));
      Vec4<R> pv = polvec<R>(ev.p[leg], hel_of(h, leg));
      e.eps[s] = inc ? pv : vconj(pv);
      if (s == gauge_gluon) e.eps[s] = e.K[s];
    }
    int ngl = e.ns;
    if (kind != K_TTNG) {
      e.qsrc = e.ns++;
      int lrow, lcol;   // legs at the row (bar) end and the column end of the light line
      if (kind == K_QQB) { lcol = 0; lrow = 1; }        // u(p0) incoming quark ; vbar(p1) incoming antiquark
      else if (kind == K_QG) { lcol = 0; lrow = 4; }    // u(p0) incoming quark ; ubar(p4) outgoing quark
      else { lrow = 1; lcol = 4; }                      // vbar(p1) incoming antiquark ; v(p4) outgoing antiquark
      bool row_in = lrow < 2, col_in = lcol < 2;
      e.Krow = realvec<R>(ev.p[lrow], row_in ? R(1) : R(-1));
      e.Kcol = realvec<R>(ev.p[lcol], col_in ? R(1) : R(-1));
      e.wrow = row_in ? bar(spinor_v<R>(ev.p[lrow], hel_of(h, lrow), true)) : bar(spinor_u<R>(ev.p[lrow], hel_of(h, lrow), true));
      e.xcol = col_in ? spinor_u<R>(ev.p[lcol], hel_of(h, lcol), true) : spinor_v<R>(ev.p[lcol], hel_of(h, lcol), true);
      e.K[e.qsrc] = vadd(e.Krow, e.Kcol);
    }
    long ncfg = 1; for (int i = 0; i < ngl; ++i) ncfg *= 8;
    int nlight = (kind == K_TTNG) ? 1 : 9;
    for (long cfg = 0; cfg < ncfg; ++cfg) {
      long c = cfg; for (int i = 0; i < ngl; ++i) { e.gcol[i] = c % 8; c /= 8; }
      for (int lc = 0; lc < nlight; ++lc) {
        e.crow = lc / 3; e.ccol = lc % 3;
        for (int ct = 0; ct < 3; ++ct) {
          e.ctop = ct;
          DualC<R> M[3]; e.amplitudes(M);
          for (int j = 0; j < 3; ++j) {
            A += std::norm(M[j].o0);
            B += R(2) * (std::conj(M[j].o0) * M[j].o1).real();
            D += std::norm(M[j].o1);
          }
        }
      }
    }
  }
  R navg;
  if (kind == K_TTNG) { int n = ev.npar - 2; R fact = 1; for (int k = 2; k <= n - 2; ++k) fact *= k; navg = R(4) * R(64) * fact; }
  else if (kind == K_QQB) { R fact = 1; for (int k = 2; k <= ev.npar - 4; ++k) fact *= k; navg = R(4) * R(9) * fact; }   // identical final gluons
  else { R fact = 1; for (int k = 2; k <= ev.npar - 5; ++k) fact *= k; navg = R(4) * R(24) * fact; }
  return ABD<R>{A / navg, B / navg, D / navg}; }

// ---------------------------------------------------------------- subprocess dispatch (ids of include/rex_trex.h)
// 0 e-e+->mu-mu+ ; 1..4 gg->tt~+{0,1,2,3}g (E1) ; 5,6 q q~->tt~g ; 7 u g->tt~u ; 8 g u~->tt~u~ (E2)
// 9 (oracle only, for the closed-form pin F-4): u u~ -> t t~ ; 10..20: further flavours, see npar_of
// 10..20: the same three one-light-line channels for the other massless flavours -- QCD does not see the flavour, it only
// labels the class: 10, 11, 12 = s s~, c c~, b b~ > t t~ g ; 13..16 = d g, s g, c g, b g > t t~ q ; 17..20 = g d~, g s~,
// g c~, g b~ > t t~ q~
inline int npar_of(int sid) {
  static const int t[10] = {4, 4, 5, 6, 7, 5, 5, 5, 5, 4};
  if (sid >= 0 && sid < 10) return t[sid];
  if (sid >= 21 && sid <= 35) return 6;             // 21 u u~ > t t~ g g ; 22 u g > t t~ u g ; 23 g u~ > t t~ u~ g ; 24..35: d, s, c, b
  return (sid >= 10 && sid <= 20) ? 5 : -1; }
inline int kind_of(int sid) {
  if (sid >= 21) return (sid - 21) % 3 == 0 ? K_QQB : ((sid - 21) % 3 == 1 ? K_QG : K_GQB);
  if (sid >= 10) return sid <= 12 ? K_QQB : (sid <= 16 ? K_QG : K_GQB);
  return sid <= 4 ? K_TTNG : ((sid <= 6 || sid == 9) ? K_QQB : (sid == 7 ? K_QG : K_GQB)); }

template <class R> R me2_one(int sid, const Event<R>& ev, const double* theta) {
  Params<R> P(theta);
  if (sid == 0) return eemumu_me2<R>(ev, P);
  if (sid <= 4) return ttng_abd<R>(ev, P).at(P.kappa);
  return e2_abd<R>(ev, P, kind_of(sid), -1, -1).at(P.kappa); }

template <class R> int me2_batch(int sid, const double* mom, long n, const double* theta, double* out) {
  int npar = npar_of(sid); if (npar < 0) return -2;
  if (sid >= 1 && sid <= 4) colour_matrix(npar - 2);   // build outside the parallel region
  #pragma omp parallel for schedule(dynamic, 1)
  for (long i = 0; i < n; ++i) { Event<R> ev(mom, n, i, npar); out[i] = (double)me2_one<R>(sid, ev, theta); }
  return 0; }

template <class R> int abd_batch(int sid, int engine, const double* mom, long n, const double* theta, int gauge_gluon, int hel_only, double* out) {
  int npar = npar_of(sid); if (npar < 0 || sid == 0) return -2;
  if (engine == 1) { if (sid > 4) return -2; colour_matrix(npar - 2); }
  #pragma omp parallel for schedule(dynamic, 1)
  for (long i = 0; i < n; ++i) {
    Event<R> ev(mom, n, i, npar); Params<R> P(theta);
    ABD<R> r = engine == 1 ? ttng_abd<R>(ev, P, gauge_gluon, hel_only) : e2_abd<R>(ev, P, kind_of(sid), gauge_gluon, hel_only);
    out[3 * i] = (double)r.A; out[3 * i + 1] = (double)r.B; out[3 * i + 2] = (double)r.D;
  }
  return 0; }

// the reweighting itself: eq.(5) PAPER.md:714 with the guard of PAPER.md:789-799; |M|^2 evaluated twice, plainly
template <class R> int reweight_batch(int sid, const double* mom, long n, const double* th_old, const double* th_new,
                                      const double* w_in, double* w_out, double* me2_old, double* me2_new) {
  int npar = npar_of(sid); if (npar < 0) return -2;
  if (sid >= 1 && sid <= 4) colour_matrix(npar - 2);
  #pragma omp parallel for schedule(dynamic, 1)
  for (long i = 0; i < n; ++i) {
    Event<R> ev(mom, n, i, npar);
    R mo = me2_one<R>(sid, ev, th_old), mn = me2_one<R>(sid, ev, th_new);
    R norm = (mo == R(0)) ? R(0) : R(1) / mo;                // procReweightor::initialise
    R w = R(w_in[i]) * norm * mn;                            // evaluate + append_wgts
    w_out[i] = (double)w;
    if (me2_old) me2_old[i] = (double)mo;
    if (me2_new) me2_new[i] = (double)mn;
  }
  return 0; }

}  // namespace

// ================================================================= C interface (ctypes, oracle/oracle.py)
extern "C" {

int oracle_npar(int sid) { return npar_of(sid); }

int oracle_me2(int sid, const double* mom, long n, const double* theta, double* out, int use_long_double) {
  return use_long_double ? me2_batch<long double>(sid, mom, n, theta, out) : me2_batch<double>(sid, mom, n, theta, out); }

// engine 1 = E1 (colour-ordered), 2 = E2 (explicit colour). out[3n] = (A,B,D). gauge_gluon: -1 or gluon index whose
// polarisation is replaced by its momentum. hel_only: -1 = sum all helicities, else restrict to that helicity index.
int oracle_abd(int sid, int engine, const double* mom, long n, const double* theta, int gauge_gluon, int hel_only,
               double* out, int use_long_double) {
  return use_long_double ? abd_batch<long double>(sid, engine, mom, n, theta, gauge_gluon, hel_only, out)
                         : abd_batch<double>(sid, engine, mom, n, theta, gauge_gluon, hel_only, out); }

int oracle_reweight(int sid, const double* mom, long n, const double* th_old, const double* th_new, const double* w_in,
                    double* w_out, double* me2_old, double* me2_new, int use_long_double) {
  return use_long_double ? reweight_batch<long double>(sid, mom, n, th_old, th_new, w_in, w_out, me2_old, me2_new)
                         : reweight_batch<double>(sid, mom, n, th_old, th_new, w_in, w_out, me2_old, me2_new); }

// E1 colour-flow amplitudes of ONE event and ONE helicity: out[np][2 orders][re,im], np = n! (lexicographic orderings)
int oracle_ttng_amps(int sid, const double* mom_one, const double* theta, int hel, int gauge_gluon, double* out) {
  int npar = npar_of(sid); if (sid < 1 || sid > 4) return -2;
  Event<long double> ev(mom_one, 1, 0, npar); Params<long double> P(theta);
  TTNG<long double> t(ev, P, hel, gauge_gluon);
  auto perms = all_perms(npar - 2);
  for (size_t i = 0; i < perms.size(); ++i) {
    auto a = t.amplitude(perms[i]);
    out[4 * i + 0] = (double)a.o0.real(); out[4 * i + 1] = (double)a.o0.imag();
    out[4 * i + 2] = (double)a.o1.real(); out[4 * i + 3] = (double)a.o1.imag();
  }
  return 0; }

// colour matrix of t t~ + n gluons: out[n! * n!]
int oracle_colour_matrix(int n, double* out) {
  if (n < 1 || n > 5) return -1;
  const auto& C = colour_matrix(n); std::memcpy(out, C.data(), C.size() * sizeof(double)); return 0; }
// one entry by direct brute force (independent of the relabelling shortcut)
double oracle_colour_entry(int n, const int* sigma, const int* sigma_p) {
  return colour_entry_bruteforce(n, std::vector<int>(sigma, sigma + n), std::vector<int>(sigma_p, sigma_p + n)); }

// external wavefunctions for the pins: kind 0 = u, 1 = v, 2 = ubar, 3 = vbar, 4 = eps ; out[4][re,im]
int oracle_wavefunction(int kind, const double* p, int lam, int massless, double* out) {
  long double q[4] = {p[0], p[1], p[2], p[3]};
  std::array<std::complex<long double>, 4> w;
  switch (kind) {
    case 0: w = spinor_u<long double>(q, lam, massless != 0); break;
    case 1: w = spinor_v<long double>(q, lam, massless != 0); break;
    case 2: w = bar(spinor_u<long double>(q, lam, massless != 0)); break;
    case 3: w = bar(spinor_v<long double>(q, lam, massless != 0)); break;
    case 4: w = polvec<long double>(q, lam); break;
    default: return -1;
  }
  for (int i = 0; i < 4; ++i) { out[2 * i] = (double)w[i].real(); out[2 * i + 1] = (double)w[i].imag(); }
  return 0; }
// gamma^mu (mu = 0..3), gamma5 (4): out[4][4][re,im]
int oracle_gamma(int mu, double* out) {
  const auto& d = dirac<double>(); if (mu < 0 || mu > 4) return -1;
  const Mat4<double>& m = mu == 4 ? d.g5 : d.g[mu];
  for (int i = 0; i < 4; ++i) for (int j = 0; j < 4; ++j) { out[(i * 4 + j) * 2] = m[i][j].real(); out[(i * 4 + j) * 2 + 1] = m[i][j].imag(); }
  return 0; }

// flop count of the plain algorithm for ONE event (old + new |M|^2 and the weight): out[4] = additions/subtractions,
// multiplications, divisions, square roots on real numbers
int oracle_count_flops(int sid, const double* mom_one, const double* th_old, const double* th_new, long long* out) {
  int npar = npar_of(sid); if (npar < 0) return -2;
  if (sid >= 1 && sid <= 4) colour_matrix(npar - 2);
  double w_in = 1.0, w_out, mo, mn;
  reweight_batch<Count>(sid, mom_one, 1, th_old, th_new, &w_in, &w_out, &mo, &mn);   // builds the static Dirac tables once
  Count::n_add = 0; Count::n_mul = 0; Count::n_div = 0; Count::n_sqrt = 0;
  int rc = reweight_batch<Count>(sid, mom_one, 1, th_old, th_new, &w_in, &w_out, &mo, &mn);
  out[0] = Count::n_add; out[1] = Count::n_mul; out[2] = Count::n_div; out[3] = Count::n_sqrt;
  return rc; }

}  // extern "C"
