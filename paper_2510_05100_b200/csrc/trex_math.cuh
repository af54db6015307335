// trex_math.cuh -- per-thread helicity-amplitude building blocks.
//
// Chiral (Weyl) representation, metric (+,-,-,-), p = (E,px,py,pz), all Lorentz vectors with UPPER indices:
//   gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s^i],[-s^i,0]]  =>  aslash = [[0, a0 - a.s],[a0 + a.s, 0]],
//   sigma^{mu nu} a_mu b_nu = diag((a x b + iE).s , (a x b - iE).s),  E = a0 b - b0 a   (2x2 blocks).
// The 2x2 block structure is used everywhere: a slash costs 8 complex multiplications, not 16.
// Strong coupling g_s is factored OUT of every routine here (amplitudes scale as g_s^n, R-4b).
#pragma once
#include <math.h>

#if defined(__CUDACC__)
#define TREX_HD __host__ __device__ __forceinline__
#else
#define TREX_HD inline
#endif

namespace trex {

template <class R> struct cx {
  R re, im;
  TREX_HD cx() {}
  TREX_HD cx(R r, R i) : re(r), im(i) {}
};
template <class R> TREX_HD cx<R> operator+(cx<R> a, cx<R> b) { return cx<R>(a.re + b.re, a.im + b.im); }
template <class R> TREX_HD cx<R> operator-(cx<R> a, cx<R> b) { return cx<R>(a.re - b.re, a.im - b.im); }
template <class R> TREX_HD cx<R> operator-(cx<R> a) { return cx<R>(-a.re, -a.im); }
template <class R> TREX_HD cx<R> operator*(cx<R> a, cx<R> b) {
  return cx<R>(a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re); }
template <class R> TREX_HD cx<R> operator*(cx<R> a, R s) { return cx<R>(a.re * s, a.im * s); }
template <class R> TREX_HD cx<R> operator*(R s, cx<R> a) { return cx<R>(a.re * s, a.im * s); }
template <class R> TREX_HD cx<R>& operator+=(cx<R>& a, cx<R> b) { a.re += b.re; a.im += b.im; return a; }
template <class R> TREX_HD cx<R>& operator-=(cx<R>& a, cx<R> b) { a.re -= b.re; a.im -= b.im; return a; }
template <class R> TREX_HD cx<R> conj(cx<R> a) { return cx<R>(a.re, -a.im); }
template <class R> TREX_HD cx<R> mul_i(cx<R> a) { return cx<R>(-a.im, a.re); }      // i * a
template <class R> TREX_HD cx<R> mul_mi(cx<R> a) { return cx<R>(a.im, -a.re); }     // -i * a
template <class R> TREX_HD R norm2(cx<R> a) { return a.re * a.re + a.im * a.im; }
// a += b * c
template <class R> TREX_HD void cfma(cx<R>& a, cx<R> b, cx<R> c) {
  a.re += b.re * c.re; a.re -= b.im * c.im; a.im += b.re * c.im; a.im += b.im * c.re; }
template <class R> TREX_HD void cfma(cx<R>& a, cx<R> b, R c) { a.re += b.re * c; a.im += b.im * c; }
template <class R> TREX_HD cx<R> cdiv(cx<R> a, cx<R> b) {
  R d = R(1) / (b.re * b.re + b.im * b.im);
  return cx<R>((a.re * b.re + a.im * b.im) * d, (a.im * b.re - a.re * b.im) * d); }

template <class R> struct vec4 { cx<R> c[4]; };      // complex Lorentz vector (current, polarisation)
template <class R> struct rvec4 { R c[4]; };         // real Lorentz vector (momentum)
template <class R> struct spinor { cx<R> c[4]; };    // row or column 4-spinor, by context
template <class R> struct dspinor { spinor<R> o0, o1; };  // dual number in kappa on the top line (R-4)
template <class R> struct ften { cx<R> b[3], e[3]; };     // antisymmetric tensor a^mu b^nu - a^nu b^mu: (a x b, a0 b - b0 a)

// precision casts: momenta and kinematic invariants are always carried in double (an fp32 amplitude must not lose
// s_ij = 2 k_i.k_j of nearly collinear legs, or q^2 - m^2 of a nearly on-shell propagator, to cancellation)
template <class R> TREX_HD rvec4<R> cast(const rvec4<double>& a) { rvec4<R> o; for (int i = 0; i < 4; ++i) o.c[i] = R(a.c[i]); return o; }
template <class R> TREX_HD cx<R> cast(const cx<double>& a) { return cx<R>(R(a.re), R(a.im)); }
template <class R> TREX_HD vec4<R> cast(const vec4<double>& a) { vec4<R> o; for (int i = 0; i < 4; ++i) o.c[i] = cast<R>(a.c[i]); return o; }
template <class R> TREX_HD spinor<R> cast(const spinor<double>& a) { spinor<R> o; for (int i = 0; i < 4; ++i) o.c[i] = cast<R>(a.c[i]); return o; }

template <class R> TREX_HD R rdot(const rvec4<R>& a, const rvec4<R>& b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3]; }
// Minkowski products without complex conjugation
template <class R> TREX_HD cx<R> dot(const rvec4<R>& a, const vec4<R>& b) {
  return cx<R>(a.c[0] * b.c[0].re - a.c[1] * b.c[1].re - a.c[2] * b.c[2].re - a.c[3] * b.c[3].re,
               a.c[0] * b.c[0].im - a.c[1] * b.c[1].im - a.c[2] * b.c[2].im - a.c[3] * b.c[3].im); }
template <class R> TREX_HD cx<R> dot(const vec4<R>& a, const vec4<R>& b) {
  cx<R> s = a.c[0] * b.c[0];
  cfma(s, -a.c[1], b.c[1]); cfma(s, -a.c[2], b.c[2]); cfma(s, -a.c[3], b.c[3]);
  return s; }
template <class R> TREX_HD rvec4<R> radd(const rvec4<R>& a, const rvec4<R>& b) {
  rvec4<R> o; for (int i = 0; i < 4; ++i) o.c[i] = a.c[i] + b.c[i]; return o; }
template <class R> TREX_HD rvec4<R> rsub(const rvec4<R>& a, const rvec4<R>& b) {
  rvec4<R> o; for (int i = 0; i < 4; ++i) o.c[i] = a.c[i] - b.c[i]; return o; }
template <class R> TREX_HD spinor<R> szero() { spinor<R> s; for (int i = 0; i < 4; ++i) s.c[i] = cx<R>(0, 0); return s; }
template <class R> TREX_HD vec4<R> vzero() { vec4<R> s; for (int i = 0; i < 4; ++i) s.c[i] = cx<R>(0, 0); return s; }
template <class R> TREX_HD ften<R> fzero() { ften<R> f; for (int i = 0; i < 3; ++i) { f.b[i] = cx<R>(0, 0); f.e[i] = cx<R>(0, 0); } return f; }

// ---------------------------------------------------------------- external wavefunctions (R-1, R-2)
// chi_+ = N (|p|+pz, px + i py), chi_- = N (-px + i py, |p|+pz), N = 1/sqrt(2|p|(|p|+pz)); pz -> -|p|: chi_+ = (0,1), chi_- = (-1,0)
// 1/sqrt(x): one special-function evaluation + Newton steps on the device, instead of a square root followed by a division
template <class R> TREX_HD R inv_sqrt(R x) {
#if defined(__CUDA_ARCH__)
  return rsqrt(x);
#else
  return R(1) / sqrt(x);
#endif
}
template <class R> TREX_HD void two_spinors(const R p[4], cx<R> plus[2], cx<R> minus[2], R& pabs) {
  const R pt2 = p[1] * p[1] + p[2] * p[2], p2 = pt2 + p[3] * p[3];
  if (p2 == R(0)) { pabs = R(0); plus[0] = cx<R>(1, 0); plus[1] = cx<R>(0, 0); minus[0] = cx<R>(0, 0); minus[1] = cx<R>(1, 0); return; }
  pabs = p2 * inv_sqrt(p2);
  R ppz = p[3] >= R(0) ? pabs + p[3] : pt2 / (pabs - p[3]);     // |p|+pz without cancellation
  if (ppz == R(0)) { plus[0] = cx<R>(0, 0); plus[1] = cx<R>(1, 0); minus[0] = cx<R>(-1, 0); minus[1] = cx<R>(0, 0); return; }
  R N = inv_sqrt(R(2) * pabs * ppz);
  plus[0] = cx<R>(N * ppz, 0); plus[1] = cx<R>(N * p[1], N * p[2]);
  minus[0] = cx<R>(-N * p[1], N * p[2]); minus[1] = cx<R>(N * ppz, 0);
}
// u(p,l) = (w_{-l} chi_l ; w_l chi_l), w_pm = sqrt(E pm |p|). massless: E := |p| (w_- = 0 exactly)
template <class R> TREX_HD spinor<R> spinor_u(const R p[4], int lam, bool massless) {
  cx<R> cp[2], cm[2]; R pabs; two_spinors<R>(p, cp, cm, pabs);
  R wp = sqrt(fmax(R(0), p[0] + pabs)), wm = sqrt(fmax(R(0), p[0] - pabs));
  if (massless) { wp = sqrt(R(2) * pabs); wm = R(0); }
  const cx<R>* chi = lam > 0 ? cp : cm;
  R up = lam > 0 ? wm : wp, lo = lam > 0 ? wp : wm;
  spinor<R> s; s.c[0] = up * chi[0]; s.c[1] = up * chi[1]; s.c[2] = lo * chi[0]; s.c[3] = lo * chi[1]; return s;
}
// v(p,l) = (-l w_l chi_{-l} ; l w_{-l} chi_{-l})
template <class R> TREX_HD spinor<R> spinor_v(const R p[4], int lam, bool massless) {
  cx<R> cp[2], cm[2]; R pabs; two_spinors<R>(p, cp, cm, pabs);
  R wp = sqrt(fmax(R(0), p[0] + pabs)), wm = sqrt(fmax(R(0), p[0] - pabs));
  if (massless) { wp = sqrt(R(2) * pabs); wm = R(0); }
  const cx<R>* chi = lam > 0 ? cm : cp;
  R up = lam > 0 ? -wp : wm, lo = lam > 0 ? wm : -wp;
  spinor<R> s; s.c[0] = up * chi[0]; s.c[1] = up * chi[1]; s.c[2] = lo * chi[0]; s.c[3] = lo * chi[1]; return s;
}
// psibar = psi^dagger gamma^0: swaps the two chiral blocks
template <class R> TREX_HD spinor<R> bar(const spinor<R>& s) {
  spinor<R> o; o.c[0] = conj(s.c[2]); o.c[1] = conj(s.c[3]); o.c[2] = conj(s.c[0]); o.c[3] = conj(s.c[1]); return o; }
// eps(p,l) = (-l e1 - i e2)/sqrt2, e1 = (0, px pz/(|p| pT), py pz/(|p| pT), -pT/|p|), e2 = (0, -py/pT, px/pT, 0)
template <class R> TREX_HD vec4<R> polvec(const R p[4], int lam, bool conjugate) {
  const R pt2 = p[1] * p[1] + p[2] * p[2], p2 = pt2 + p[3] * p[3];
  R e1[4], e2[4];
  if (pt2 < R(1e-28) * p2 || pt2 == R(0)) {
    R sg = p[3] >= 0 ? R(1) : R(-1);
    e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0;
    e2[0] = 0; e2[1] = 0; e2[2] = sg; e2[3] = 0;
  } else {
    // two independent reciprocal square roots instead of two square roots and three divisions
    const R ipt = inv_sqrt(pt2), ip = inv_sqrt(p2);
    const R ipp = ipt * ip, pt = pt2 * ipt;
    e1[0] = 0; e1[1] = p[1] * p[3] * ipp; e1[2] = p[2] * p[3] * ipp; e1[3] = -pt * ip;
    e2[0] = 0; e2[1] = -p[2] * ipt; e2[2] = p[1] * ipt; e2[3] = 0;
  }
  const R rs2 = R(0.70710678118654752440);
  R sgn = conjugate ? R(1) : R(-1);
  vec4<R> e;
  for (int i = 0; i < 4; ++i) e.c[i] = cx<R>(-R(lam) * e1[i] * rs2, sgn * e2[i] * rs2);
  return e;
}

// ---------------------------------------------------------------- Dirac algebra in 2x2 blocks
// row spinor times aslash, complex a
template <class R> TREX_HD spinor<R> row_slash(const spinor<R>& r, const vec4<R>& a) {
  cx<R> ap = a.c[0] + a.c[3], am = a.c[0] - a.c[3];
  cx<R> at = a.c[1] + mul_i(a.c[2]), ab = a.c[1] - mul_i(a.c[2]);
  spinor<R> o;
  o.c[0] = r.c[2] * ap; cfma(o.c[0], r.c[3], at);
  o.c[1] = r.c[2] * ab; cfma(o.c[1], r.c[3], am);
  o.c[2] = r.c[0] * am; cfma(o.c[2], -r.c[1], at);
  o.c[3] = r.c[1] * ap; cfma(o.c[3], -r.c[0], ab);
  return o; }
// row spinor times qslash, real q
template <class R> TREX_HD spinor<R> row_slash(const spinor<R>& r, const rvec4<R>& q) {
  R ap = q.c[0] + q.c[3], am = q.c[0] - q.c[3];
  cx<R> at(q.c[1], q.c[2]), ab(q.c[1], -q.c[2]);
  spinor<R> o;
  o.c[0] = r.c[2] * ap; cfma(o.c[0], r.c[3], at);
  o.c[1] = r.c[2] * ab; cfma(o.c[1], r.c[3], am);
  o.c[2] = r.c[0] * am; cfma(o.c[2], -r.c[1], at);
  o.c[3] = r.c[1] * ap; cfma(o.c[3], -r.c[0], ab);
  return o; }
// aslash times column spinor (real and complex a)
template <class R> TREX_HD spinor<R> slash_col(const vec4<R>& a, const spinor<R>& x) {
  cx<R> ap = a.c[0] + a.c[3], am = a.c[0] - a.c[3];
  cx<R> at = a.c[1] + mul_i(a.c[2]), ab = a.c[1] - mul_i(a.c[2]);
  spinor<R> o;
  o.c[0] = am * x.c[2]; cfma(o.c[0], -ab, x.c[3]);
  o.c[1] = ap * x.c[3]; cfma(o.c[1], -at, x.c[2]);
  o.c[2] = ap * x.c[0]; cfma(o.c[2], ab, x.c[1]);
  o.c[3] = at * x.c[0]; cfma(o.c[3], am, x.c[1]);
  return o; }
template <class R> TREX_HD spinor<R> slash_col(const rvec4<R>& q, const spinor<R>& x) {
  R ap = q.c[0] + q.c[3], am = q.c[0] - q.c[3];
  cx<R> at(q.c[1], q.c[2]), ab(q.c[1], -q.c[2]);
  spinor<R> o;
  o.c[0] = x.c[2] * am; cfma(o.c[0], -ab, x.c[3]);
  o.c[1] = x.c[3] * ap; cfma(o.c[1], -at, x.c[2]);
  o.c[2] = x.c[0] * ap; cfma(o.c[2], ab, x.c[1]);
  o.c[3] = at * x.c[0]; cfma(o.c[3], x.c[1], am);
  return o; }
template <class R> TREX_HD cx<R> row_col(const spinor<R>& r, const spinor<R>& x) {
  cx<R> s = r.c[0] * x.c[0]; cfma(s, r.c[1], x.c[1]); cfma(s, r.c[2], x.c[2]); cfma(s, r.c[3], x.c[3]); return s; }
// w gamma^mu x for mu = 0..3 (upper index)
template <class R> TREX_HD vec4<R> bilinear(const spinor<R>& w, const spinor<R>& x) {
  // gamma^0: w0 x2 + w1 x3 + w2 x0 + w3 x1 ; gamma^i = [[0,s^i],[-s^i,0]]
  cx<R> a02 = w.c[0] * x.c[2], a13 = w.c[1] * x.c[3], a20 = w.c[2] * x.c[0], a31 = w.c[3] * x.c[1];
  cx<R> a03 = w.c[0] * x.c[3], a12 = w.c[1] * x.c[2], a21 = w.c[2] * x.c[1], a30 = w.c[3] * x.c[0];
  vec4<R> o;
  o.c[0] = (a02 + a13) + (a20 + a31);
  o.c[1] = (a03 + a12) - (a21 + a30);                 // s^1 = [[0,1],[1,0]]
  o.c[2] = mul_mi(a03 - a12) + mul_i(a21 - a30);      // s^2 = [[0,-i],[i,0]]: upper w0(-i)x3 + w1(i)x2 ; lower -(w2(-i)x1 + w3(i)x0)
  o.c[3] = (a02 - a13) - (a20 - a31);                 // s^3 = diag(1,-1)
  return o; }

// wedge: f += a ^ b   (a x b, a0 b - b0 a), real a
template <class R> TREX_HD void wedge_acc(ften<R>& f, const rvec4<R>& a, const vec4<R>& b) {
  f.b[0] += a.c[2] * b.c[3] - a.c[3] * b.c[2];
  f.b[1] += a.c[3] * b.c[1] - a.c[1] * b.c[3];
  f.b[2] += a.c[1] * b.c[2] - a.c[2] * b.c[1];
  for (int i = 0; i < 3; ++i) f.e[i] += a.c[0] * b.c[i + 1] - a.c[i + 1] * b.c[0];
}
template <class R> TREX_HD void wedge_acc(ften<R>& f, const vec4<R>& a, const vec4<R>& b) {
  cfma(f.b[0], a.c[2], b.c[3]); cfma(f.b[0], -a.c[3], b.c[2]);
  cfma(f.b[1], a.c[3], b.c[1]); cfma(f.b[1], -a.c[1], b.c[3]);
  cfma(f.b[2], a.c[1], b.c[2]); cfma(f.b[2], -a.c[2], b.c[1]);
  for (int i = 0; i < 3; ++i) { cfma(f.e[i], a.c[0], b.c[i + 1]); cfma(f.e[i], -a.c[i + 1], b.c[0]); }
}
// o += r * (2 sigma^{mu nu} F_{mu nu}/2) = r * diag((2B + 2iE).s, (2B - 2iE).s)
template <class R> TREX_HD void row_sigma_acc(spinor<R>& o, const spinor<R>& r, const ften<R>& f) {
  cx<R> xp[3], xm[3];
  for (int i = 0; i < 3; ++i) { cx<R> ie = mul_i(f.e[i]); xp[i] = R(2) * (f.b[i] + ie); xm[i] = R(2) * (f.b[i] - ie); }
  cx<R> pt = xp[0] + mul_i(xp[1]), pb = xp[0] - mul_i(xp[1]);
  cx<R> mt = xm[0] + mul_i(xm[1]), mb = xm[0] - mul_i(xm[1]);
  // X.s = [[X3, X1 - iX2],[X1 + iX2, -X3]]
  cfma(o.c[0], r.c[0], xp[2]); cfma(o.c[0], r.c[1], pt);
  cfma(o.c[1], r.c[0], pb);    cfma(o.c[1], -r.c[1], xp[2]);
  cfma(o.c[2], r.c[2], xm[2]); cfma(o.c[2], r.c[3], mt);
  cfma(o.c[3], r.c[2], mb);    cfma(o.c[3], -r.c[3], xm[2]);
}

// ---------------------------------------------------------------- ordered gluon vertices (R-6), g_s = 1
// acc += J1 ((-P-k1).J2) + (k1-k2)(J1.J2) + J2 ((k2+P).J1), P = k1 + k2
template <class R> TREX_HD void v3_acc(vec4<R>& acc, const rvec4<double>& k1, const vec4<R>& J1, const rvec4<double>& k2, const vec4<R>& J2) {
  rvec4<R> a, b, d;
  for (int i = 0; i < 4; ++i) { a.c[i] = R(-(2.0 * k1.c[i] + k2.c[i])); b.c[i] = R(2.0 * k2.c[i] + k1.c[i]); d.c[i] = R(k1.c[i] - k2.c[i]); }
  cx<R> aJ2 = dot(a, J2), bJ1 = dot(b, J1), J1J2 = dot(J1, J2);
  for (int i = 0; i < 4; ++i) { cfma(acc.c[i], J1.c[i], aJ2); cfma(acc.c[i], J1J2, d.c[i]); cfma(acc.c[i], J2.c[i], bJ1); }
}
// acc += J1 (J2.J3) + J3 (J1.J2) - 2 J2 (J1.J3)
template <class R> TREX_HD void v4_acc(vec4<R>& acc, const vec4<R>& J1, const vec4<R>& J2, const vec4<R>& J3) {
  cx<R> d23 = dot(J2, J3), d12 = dot(J1, J2), d13 = R(-2) * dot(J1, J3);
  for (int i = 0; i < 4; ++i) { cfma(acc.c[i], J1.c[i], d23); cfma(acc.c[i], J3.c[i], d12); cfma(acc.c[i], J2.c[i], d13); }
}

}  // namespace trex
