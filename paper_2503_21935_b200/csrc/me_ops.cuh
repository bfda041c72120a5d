// me_ops.cuh -- register-resident building blocks of the tree-level amplitudes (sm_100a device code).
//
// These are the B200 counterparts of the HELAS/ALOHA routines BASELINE.json north_star (b) names
// (ixxxxx/oxxxxx/vxxxxx, FFV1_0/FFV1_1/FFV1_2, VVV1P0_1, VVVV*), restated from the textbook Feynman
// rules of SURVEY.md 8(c) / Appendix A ("Feynman diagrams") in a form chosen for the
// FMA pipes:
//   * CHIRAL (Weyl) representation: gamma^0 = [[0,1],[1,0]], gamma^i = [[0,s_i],[-s_i,0]]; a slashed
//     vector is two 2x2 blocks, so a vertex costs 8 complex multiplies instead of 16.
//   * "phase-stripped" rules: every factor i of the Feynman rules is pulled out of the
//     currents; what is left has REAL couplings and every colour-flow coefficient is +-1.
//        three-gluon current   J = (g/K^2)  [ (A.B)(kA-kB) + ((kA+2kB).A) B - ((2kA+kB).B) A ]
//        four-gluon current    J = (g^2/K^2) { (A.C)B-(B.C)A , (A.B)C-(B.C)A , (A.B)C-(A.C)B }
//        quark line            R' = R Jslash (qslash + m) * g/(q^2 - m^2 + i m Gamma)
//        closure               A  = g * (R Jslash) . v
//     all momenta incoming, metric (+,-,-,-), 4-vectors with upper indices.
// Everything is a template on the arithmetic type T (double or float): BASELINE.json north_star (f).
// No code here is shared with oracle/ (Dirac representation, literal rules, C++ on the host).
#pragma once

#ifndef ME_HD
#define ME_HD __host__ __device__ __forceinline__
#endif

namespace me {

template <typename T>
struct cx {
  T re, im;
};
template <typename T>
struct vec4 {  // complex Lorentz vector, upper index: c[0] = time component
  cx<T> c[4];
};
template <typename T>
struct mom4 {  // real momentum (E, px, py, pz)
  T c[4];
};
template <typename T>
struct spin4 {  // Dirac spinor in the chiral representation (row or column by context)
  cx<T> c[4];
};

template <typename T> ME_HD cx<T> mk(T re, T im) { cx<T> r; r.re = re; r.im = im; return r; }
template <typename T> ME_HD cx<T> operator+(cx<T> a, cx<T> b) { return mk<T>(a.re + b.re, a.im + b.im); }
template <typename T> ME_HD cx<T> operator-(cx<T> a, cx<T> b) { return mk<T>(a.re - b.re, a.im - b.im); }
template <typename T> ME_HD cx<T> operator-(cx<T> a) { return mk<T>(-a.re, -a.im); }
// a*b + c as one operation of the scalar type (overloaded for the packed float pair of me_group.cuh)
template <typename T> ME_HD T fmad(T a, T b, T c) { return a * b + c; }
template <typename T> ME_HD cx<T> operator*(cx<T> a, cx<T> b) {
  return mk<T>(fmad(a.re, b.re, (-a.im) * b.im), fmad(a.re, b.im, a.im * b.re));
}
template <typename T> ME_HD cx<T> operator*(T s, cx<T> a) { return mk<T>(s * a.re, s * a.im); }
// a + b*c
template <typename T> ME_HD cx<T> fma(cx<T> b, cx<T> c, cx<T> a) {
  return mk<T>(fmad(-b.im, c.im, fmad(b.re, c.re, a.re)), fmad(b.im, c.re, fmad(b.re, c.im, a.im)));
}
// a - b*c
template <typename T> ME_HD cx<T> fnma(cx<T> b, cx<T> c, cx<T> a) {
  return mk<T>(fmad(b.im, c.im, fmad(-b.re, c.re, a.re)), fmad(-b.im, c.re, fmad(-b.re, c.im, a.im)));
}
template <typename T> ME_HD cx<T> fma(T s, cx<T> c, cx<T> a) { return mk<T>(fmad(s, c.re, a.re), fmad(s, c.im, a.im)); }
template <typename T> ME_HD cx<T> conj(cx<T> a) { return mk<T>(a.re, -a.im); }
template <typename T> ME_HD T norm2(cx<T> a) { return a.re * a.re + a.im * a.im; }
// i * a
template <typename T> ME_HD cx<T> times_i(cx<T> a) { return mk<T>(-a.im, a.re); }

template <typename T> ME_HD mom4<T> operator+(mom4<T> a, mom4<T> b) {
  mom4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i];
  return r;
}
template <typename T> ME_HD mom4<T> operator-(mom4<T> a, mom4<T> b) {
  mom4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] - b.c[i];
  return r;
}
template <typename T> ME_HD mom4<T> neg(mom4<T> a) {
  mom4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = -a.c[i];
  return r;
}
template <typename T> ME_HD T mdot(mom4<T> a, mom4<T> b) {
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}
// Minkowski product, no complex conjugation
template <typename T> ME_HD cx<T> mdot(const vec4<T>& a, const vec4<T>& b) {
  cx<T> r = a.c[0] * b.c[0];
#if !defined(ME_MDOT_FMA) || ME_MDOT_FMA
  r = fnma(a.c[1], b.c[1], r);   // four FMAs per component (r - a*b as a product and a subtraction is six operations)
  r = fnma(a.c[2], b.c[2], r);
  r = fnma(a.c[3], b.c[3], r);
#else
  r = r - a.c[1] * b.c[1];
  r = r - a.c[2] * b.c[2];
  r = r - a.c[3] * b.c[3];
#endif
  return r;
}
template <typename T> ME_HD cx<T> mdot(mom4<T> k, const vec4<T>& a) {
  return mk<T>(k.c[0] * a.c[0].re - k.c[1] * a.c[1].re - k.c[2] * a.c[2].re - k.c[3] * a.c[3].re,
               k.c[0] * a.c[0].im - k.c[1] * a.c[1].im - k.c[2] * a.c[2].im - k.c[3] * a.c[3].im);
}
template <typename T> ME_HD vec4<T> operator+(const vec4<T>& a, const vec4<T>& b) {
  vec4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i];
  return r;
}
template <typename T> ME_HD vec4<T> operator-(const vec4<T>& a, const vec4<T>& b) {
  vec4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] - b.c[i];
  return r;
}
template <typename T> ME_HD vec4<T> zero_vec4() {
  vec4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = mk<T>(T(0), T(0));
  return r;
}
template <typename T> ME_HD spin4<T> operator+(const spin4<T>& a, const spin4<T>& b) {
  spin4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i];
  return r;
}

// ---------------------------------------------------------------------------------------------
// External wavefunctions, helicity = physical helicity in the given frame.
// ---------------------------------------------------------------------------------------------
// Helicity-independent part of a massless vector's polarisation: e1/sqrt2 and e2/sqrt2 (spatial
// parts only, time components vanish).  eps(lambda) = -lambda e1/sqrt2 - i e2/sqrt2.
template <typename T>
struct polbasis {
  T e1[3], e2[3];
};
template <typename T> ME_HD polbasis<T> make_polbasis(mom4<T> p) {
  polbasis<T> b;
  const T px = p.c[1], py = p.c[2], pz = p.c[3];
  const T pt2 = px * px + py * py;
  const T rs2 = T(0.70710678118654752440);
  if (pt2 == T(0)) {
    b.e1[0] = rs2; b.e1[1] = T(0); b.e1[2] = T(0);
    b.e2[0] = T(0); b.e2[1] = (pz >= T(0)) ? rs2 : -rs2; b.e2[2] = T(0);
  } else {
    const T pp = sqrt(pt2 + pz * pz), pt = sqrt(pt2);
    const T a = rs2 / (pp * pt), c = rs2 / pt;
    b.e1[0] = px * pz * a; b.e1[1] = py * pz * a; b.e1[2] = -pt2 * a;
    b.e2[0] = -py * c; b.e2[1] = px * c; b.e2[2] = T(0);
  }
  return b;
}
// lambda = +-1; outgoing = true gives the complex conjugate (final-state vector)
template <typename T> ME_HD vec4<T> polvec(const polbasis<T>& b, int lambda, bool outgoing) {
  vec4<T> e;
  const T s = (lambda > 0) ? T(-1) : T(1);
  const T t = outgoing ? T(1) : T(-1);
  e.c[0] = mk<T>(T(0), T(0));
#pragma unroll
  for (int i = 0; i < 3; i++) e.c[i + 1] = mk<T>(s * b.e1[i], t * b.e2[i]);
  return e;
}

// Two-component helicity spinors chi_+ and chi_- of direction p, and omega_+- = sqrt(E +- |p|).
template <typename T>
struct spinbasis {
  cx<T> xp[2], xm[2];  // chi_+, chi_-
  T wp, wm;            // omega_+, omega_-
};
template <typename T> ME_HD spinbasis<T> make_spinbasis(mom4<T> p, T m) {
  spinbasis<T> s;
  const T px = p.c[1], py = p.c[2], pz = p.c[3];
  const T pt2 = px * px + py * py;
  const T pp = sqrt(pt2 + pz * pz);
  s.wp = sqrt(p.c[0] + pp);
  // E - |p| = m^2 / (E + |p|): no cancellation
  s.wm = (m > T(0)) ? m / s.wp : T(0);
  if (pp == T(0)) {  // at rest: quantise along +z
    s.xp[0] = mk<T>(T(1), T(0)); s.xp[1] = mk<T>(T(0), T(0));
    s.xm[0] = mk<T>(T(0), T(0)); s.xm[1] = mk<T>(T(1), T(0));
  } else if ((pt2 == T(0) && pz < T(0)) || ((pz >= T(0)) ? pp + pz : pt2 / (pp - pz)) == T(0)) {
    // exactly backward, or so close to it that |p| + pz underflows (fp32): the -z limit of the formulas below
    s.xp[0] = mk<T>(T(0), T(0)); s.xp[1] = mk<T>(T(1), T(0));
    s.xm[0] = mk<T>(T(-1), T(0)); s.xm[1] = mk<T>(T(0), T(0));
  } else {
    // |p| + pz without cancellation for backward directions
    const T ppz = (pz >= T(0)) ? pp + pz : pt2 / (pp - pz);
    const T n = rsqrt(T(2) * pp * ppz);
    s.xp[0] = mk<T>(n * ppz, T(0)); s.xp[1] = mk<T>(n * px, n * py);
    s.xm[0] = mk<T>(-n * px, n * py); s.xm[1] = mk<T>(n * ppz, T(0));
  }
  return s;
}
// u(p,lambda) = ( w_{-lambda} chi_lambda ; w_lambda chi_lambda )            (column)
template <typename T> ME_HD spin4<T> spinor_u(const spinbasis<T>& s, int lambda) {
  spin4<T> u;
  const cx<T>* x = (lambda > 0) ? s.xp : s.xm;
  const T wu = (lambda > 0) ? s.wm : s.wp, wl = (lambda > 0) ? s.wp : s.wm;
  u.c[0] = wu * x[0]; u.c[1] = wu * x[1]; u.c[2] = wl * x[0]; u.c[3] = wl * x[1];
  return u;
}
// v(p,lambda) = ( -lambda w_lambda chi_{-lambda} ; lambda w_{-lambda} chi_{-lambda} )   (column)
template <typename T> ME_HD spin4<T> spinor_v(const spinbasis<T>& s, int lambda) {
  spin4<T> v;
  const cx<T>* x = (lambda > 0) ? s.xm : s.xp;
  const T wu = (lambda > 0) ? -s.wp : s.wm, wl = (lambda > 0) ? s.wm : -s.wp;
  v.c[0] = wu * x[0]; v.c[1] = wu * x[1]; v.c[2] = wl * x[0]; v.c[3] = wl * x[1];
  return v;
}
// psi-bar = psi^dagger gamma^0 (row): swaps the two 2-component halves and conjugates
template <typename T> ME_HD spin4<T> bar(const spin4<T>& u) {
  spin4<T> r;
  r.c[0] = conj(u.c[2]); r.c[1] = conj(u.c[3]); r.c[2] = conj(u.c[0]); r.c[3] = conj(u.c[1]);
  return r;
}

// branch-free choice between two register-resident spinors (no dynamic indexing -> no local memory)
template <typename T> ME_HD spin4<T> select(bool first, const spin4<T>& a, const spin4<T>& b) {
  spin4<T> r;
#pragma unroll
  for (int i = 0; i < 4; i++) r.c[i] = mk<T>(first ? a.c[i].re : b.c[i].re, first ? a.c[i].im : b.c[i].im);
  return r;
}

// ---------------------------------------------------------------------------------------------
// Gluon currents
// ---------------------------------------------------------------------------------------------
// three-gluon current (VVV1P0_1): gk = g / K^2, K = kA + kB
template <typename T>
ME_HD vec4<T> vvv_current(const vec4<T>& A, const vec4<T>& B, mom4<T> kA, mom4<T> kB, T gk) {
  const cx<T> ab = mdot(A, B);
  mom4<T> kab, k1, k2;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    kab.c[i] = gk * (kA.c[i] - kB.c[i]);
    k1.c[i] = gk * (kA.c[i] + T(2) * kB.c[i]);
    k2.c[i] = -gk * (T(2) * kA.c[i] + kB.c[i]);
  }
  const cx<T> ca = mdot(k1, A);  // multiplies B
  const cx<T> cb = mdot(k2, B);  // multiplies A
  vec4<T> J;
#pragma unroll
  for (int i = 0; i < 4; i++) {
    cx<T> t = kab.c[i] * ab;
    t = fma(ca, B.c[i], t);
    t = fma(cb, A.c[i], t);
    J.c[i] = t;
  }
  return J;
}
// four-gluon currents (VVVV1/3/4P0_1), the three colour structures at once: g2k = g^2 / K^2
//   J0 <-> [[A,B],C]: (A.C)B - (B.C)A ;  J1 <-> [[A,C],B]: (A.B)C - (B.C)A ;  J2 <-> [[B,C],A]: (A.B)C - (A.C)B
template <typename T>
ME_HD void vvvv_currents(const vec4<T>& A, const vec4<T>& B, const vec4<T>& C, T g2k, vec4<T>& J0, vec4<T>& J1,
                         vec4<T>& J2) {
  const cx<T> ab = g2k * mdot(A, B), ac = g2k * mdot(A, C), bc = g2k * mdot(B, C);
#pragma unroll
  for (int i = 0; i < 4; i++) {
    const cx<T> abC = ab * C.c[i], acB = ac * B.c[i], bcA = bc * A.c[i];
    J0.c[i] = acB - bcA;
    J1.c[i] = abC - bcA;
    J2.c[i] = abC - acB;
  }
}

// ---------------------------------------------------------------------------------------------
// Quark line (row spinor running from the outgoing t towards the outgoing tbar)
// ---------------------------------------------------------------------------------------------
// R * Jslash  (FFV1 vertex, coupling stripped)
template <typename T> ME_HD spin4<T> row_slash(const spin4<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]);   // J1 + i J2
  const cx<T> jtb = J.c[1] - times_i(J.c[2]);  // J1 - i J2
  spin4<T> o;
  o.c[0] = fma(R.c[3], jt, R.c[2] * jp);
  o.c[1] = fma(R.c[3], jm, R.c[2] * jtb);
  o.c[2] = fnma(R.c[1], jt, R.c[0] * jm);
  o.c[3] = fnma(R.c[0], jtb, R.c[1] * jp);
  return o;
}
template <typename T> ME_HD spin4<T> row_slash_neg(const spin4<T>& R, const vec4<T>& J) {
  spin4<T> o = row_slash(R, J);
#pragma unroll
  for (int i = 0; i < 4; i++) o.c[i] = -o.c[i];
  return o;
}
// R (WLslash P_L + WRslash P_R): a vector boson with chirality-dependent couplings on a fermion line (the boson's
// coupling-weighted current differs for the two chiralities).  In the chiral representation P_L keeps the upper two
// components of the row R gamma^mu, P_R the lower two.
template <typename T> ME_HD spin4<T> row_slash_chiral(const spin4<T>& R, const vec4<T>& WL, const vec4<T>& WR) {
  const spin4<T> a = row_slash(R, WL), b = row_slash(R, WR);
  spin4<T> o;
  o.c[0] = a.c[0]; o.c[1] = a.c[1]; o.c[2] = b.c[2]; o.c[3] = b.c[3];
  return o;
}
// X += R * Jslash
template <typename T> ME_HD void row_slash_add(spin4<T>& X, const spin4<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]);
  const cx<T> jtb = J.c[1] - times_i(J.c[2]);
  X.c[0] = fma(R.c[3], jt, fma(R.c[2], jp, X.c[0]));
  X.c[1] = fma(R.c[3], jm, fma(R.c[2], jtb, X.c[1]));
  X.c[2] = fnma(R.c[1], jt, fma(R.c[0], jm, X.c[2]));
  X.c[3] = fnma(R.c[0], jtb, fma(R.c[1], jp, X.c[3]));
}
// X -= R * Jslash
template <typename T> ME_HD void row_slash_sub(spin4<T>& X, const spin4<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]);
  const cx<T> jtb = J.c[1] - times_i(J.c[2]);
  X.c[0] = X.c[0] - fma(R.c[3], jt, R.c[2] * jp);
  X.c[1] = X.c[1] - fma(R.c[3], jm, R.c[2] * jtb);
  X.c[2] = fma(R.c[1], jt, X.c[2]) - R.c[0] * jm;
  X.c[3] = fma(R.c[0], jtb, X.c[3]) - R.c[1] * jp;
}
// X (qslash + m) * gd,  q real, gd = g / (q^2 - m^2 + i m Gamma)   (propagator of FFV1_2, stripped)
template <typename T> ME_HD spin4<T> row_prop(const spin4<T>& X, mom4<T> q, T m, cx<T> gd) {
  const T qp = q.c[0] + q.c[3], qm = q.c[0] - q.c[3];
  const cx<T> qt = mk<T>(q.c[1], q.c[2]), qtb = mk<T>(q.c[1], -q.c[2]);
  spin4<T> o;
  o.c[0] = fma(X.c[3], qt, fma(qp, X.c[2], m * X.c[0]));
  o.c[1] = fma(qm, X.c[3], fma(X.c[2], qtb, m * X.c[1]));
  o.c[2] = fnma(X.c[1], qt, fma(qm, X.c[0], m * X.c[2]));
  o.c[3] = fnma(X.c[0], qtb, fma(qp, X.c[1], m * X.c[3]));
#pragma unroll
  for (int i = 0; i < 4; i++) o.c[i] = o.c[i] * gd;
  return o;
}
// ---------------------------------------------------------------------------------------------
// Massless quark line of definite chirality: two-component (Weyl) form of the routines above.  In the chiral
// representation a massless row spinor lives in one half (CH = 0: the lower two components, CH = 1: the upper two);
// a vertex R Jslash moves it to the other half and the propagator numerator qslash moves it back, so a line costs half
// the arithmetic and half the registers of the four-component form.
// ---------------------------------------------------------------------------------------------
template <typename T>
struct wsp {  // the two non-zero components
  cx<T> c[2];
};
template <int CH, typename T> ME_HD wsp<T> w_half(const spin4<T>& R) {  // the half a CH line lives in
  wsp<T> r;
  r.c[0] = R.c[CH ? 0 : 2]; r.c[1] = R.c[CH ? 1 : 3];
  return r;
}
// R Jslash: CH = 0 takes (R2, R3) and returns components (0, 1); CH = 1 takes (R0, R1) and returns (2, 3)
template <int CH, typename T> ME_HD wsp<T> w_slash(const wsp<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]), jtb = J.c[1] - times_i(J.c[2]);
  wsp<T> o;
  if (CH == 0) { o.c[0] = fma(R.c[1], jt, R.c[0] * jp); o.c[1] = fma(R.c[1], jm, R.c[0] * jtb); }
  else { o.c[0] = fnma(R.c[1], jt, R.c[0] * jm); o.c[1] = fnma(R.c[0], jtb, R.c[1] * jp); }
  return o;
}
template <int CH, typename T> ME_HD wsp<T> w_slash_neg(const wsp<T>& R, const vec4<T>& J) {
  wsp<T> o = w_slash<CH>(R, J);
  o.c[0] = -o.c[0]; o.c[1] = -o.c[1];
  return o;
}
template <int CH, typename T> ME_HD void w_slash_add(wsp<T>& X, const wsp<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]), jtb = J.c[1] - times_i(J.c[2]);
  if (CH == 0) { X.c[0] = fma(R.c[1], jt, fma(R.c[0], jp, X.c[0])); X.c[1] = fma(R.c[1], jm, fma(R.c[0], jtb, X.c[1])); }
  else { X.c[0] = fnma(R.c[1], jt, fma(R.c[0], jm, X.c[0])); X.c[1] = fnma(R.c[0], jtb, fma(R.c[1], jp, X.c[1])); }
}
template <int CH, typename T> ME_HD void w_slash_sub(wsp<T>& X, const wsp<T>& R, const vec4<T>& J) {
  const cx<T> jp = J.c[0] + J.c[3], jm = J.c[0] - J.c[3];
  const cx<T> jt = J.c[1] + times_i(J.c[2]), jtb = J.c[1] - times_i(J.c[2]);
  if (CH == 0) { X.c[0] = fnma(R.c[1], jt, fnma(R.c[0], jp, X.c[0])); X.c[1] = fnma(R.c[1], jm, fnma(R.c[0], jtb, X.c[1])); }
  else { X.c[0] = fma(R.c[1], jt, fnma(R.c[0], jm, X.c[0])); X.c[1] = fma(R.c[0], jtb, fnma(R.c[1], jp, X.c[1])); }
}
// X qslash / q^2 (massless propagator, gd = 1 / q^2 real): back to the half the line lives in
template <int CH, typename T> ME_HD wsp<T> w_prop(const wsp<T>& X, mom4<T> q, T gd) {
  const T qp = q.c[0] + q.c[3], qm = q.c[0] - q.c[3];
  const cx<T> qt = mk<T>(q.c[1], q.c[2]), qtb = mk<T>(q.c[1], -q.c[2]);
  wsp<T> o;
  if (CH == 0) { o.c[0] = fnma(X.c[1], qt, qm * X.c[0]); o.c[1] = fnma(X.c[0], qtb, qp * X.c[1]); }   // (0,1) -> (2,3)
  else { o.c[0] = fma(X.c[1], qt, qp * X.c[0]); o.c[1] = fma(X.c[0], qtb, qm * X.c[1]); }            // (2,3) -> (0,1)
  o.c[0] = gd * o.c[0]; o.c[1] = gd * o.c[1];
  return o;
}
template <typename T> ME_HD wsp<T> operator+(const wsp<T>& a, const wsp<T>& b) {
  wsp<T> r;
  r.c[0] = a.c[0] + b.c[0]; r.c[1] = a.c[1] + b.c[1];
  return r;
}
// closure with a column spinor: X holds components (0,1) for CH = 0, (2,3) for CH = 1
template <int CH, typename T> ME_HD cx<T> w_col(const wsp<T>& X, const spin4<T>& v) {
  return fma(X.c[1], v.c[CH ? 3 : 1], X.c[0] * v.c[CH ? 2 : 0]);
}

// chiral vector currents of a fermion line, abar gamma^mu P_R b and abar gamma^mu P_L b (upper index):
//   gamma^mu = [[0, sigma^mu], [sigmabar^mu, 0]], P_L = upper two components, P_R = lower two
template <typename T>
ME_HD void chiral_currents(const spin4<T>& a, const spin4<T>& b, vec4<T>& JR, vec4<T>& JL) {
  const cx<T> a0b2 = a.c[0] * b.c[2], a1b3 = a.c[1] * b.c[3], a0b3 = a.c[0] * b.c[3], a1b2 = a.c[1] * b.c[2];
  JR.c[0] = a0b2 + a1b3;
  JR.c[1] = a0b3 + a1b2;
  JR.c[2] = times_i(a1b2 - a0b3);
  JR.c[3] = a0b2 - a1b3;
  const cx<T> a2b0 = a.c[2] * b.c[0], a3b1 = a.c[3] * b.c[1], a2b1 = a.c[2] * b.c[1], a3b0 = a.c[3] * b.c[0];
  JL.c[0] = a2b0 + a3b1;
  JL.c[1] = -(a2b1 + a3b0);
  JL.c[2] = times_i(a2b1 - a3b0);
  JL.c[3] = a3b1 - a2b0;
}
template <typename T> ME_HD cx<T> row_col(const spin4<T>& R, const spin4<T>& v) {
  cx<T> r = R.c[0] * v.c[0];
  r = fma(R.c[1], v.c[1], r);
  r = fma(R.c[2], v.c[2], r);
  r = fma(R.c[3], v.c[3], r);
  return r;
}

}  // namespace me
