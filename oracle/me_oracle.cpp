// me_oracle.cpp -- ORACLE (test infrastructure, NOT the product).
//
// Plain, slow, scalar fp64 CPU evaluation of the tree-level squared matrix element |M|^2 summed
// over helicities and colours ("from the particle momenta, the matrix element (ME) ... is
// computed"; "Feynman diagrams" + "the color matrix quadratic form", PAPER.md:108;
// "different helicity combinations of the particles from each event") for
//     e+ e- -> mu+ mu-      (photon + Z, 2 diagrams)                       BASELINE.json configs[0]
//     g g -> t tbar + (n-2) g,  n = 2..5 gluons (3/16/123/1240 diagrams)   BASELINE.json configs[1..4]
//     g ubar -> tau+ tau- + (n-1) g + ubar, n = 1..3 gluons (photon + Z)    SURVEY.md 8(f) NEXT #4: the mixed
//        EW+QCD workload class of the paper's Table 4 ("g u~ -> tau+ tau- g g u~" is n = 3)
// The paper prints no formula; the definition written out here is the textbook one
// (Route A): literal Feynman rules (Peskin & Schroeder conventions), explicit 4x4
// Dirac matrices in the DIRAC representation, every diagram enumerated and evaluated one by one,
// colour factors reduced to the trace basis with f^{abc} T^c = -i [T^a, T^b], colour matrix from
// explicit Gell-Mann matrices.
//
//   ME = (1/denom) sum_h sum_{sigma,tau} J_sigma(h)^* C_{sigma tau} J_tau(h),  J_sigma = sum_d K_{d sigma} A_d(h)
//
// Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline/reference leg may call this.
// It shares no code, table or constant with the CUDA path (paper_2503_21935_b200/csrc).
// Pins: tests/test_oracle_*.py (closed forms P1-P4, Ward identity P5, Lorentz P6, colour matrix
// P7, diagram counts P8, coupling scaling P9, helicity sums P10, MHV P11, Bose P12, parity P13,
// Berends-Giele Route B and explicit-colour brute force P14).  Selection semantics (good-helicity
// criterion, helicity/colour selection rule) are OUR reading (readings R10, R11): the
// paper is silent, so orc_select is "parity unpinned" against the paper.
//
// Build: g++ -O2 -fopenmp -shared -fPIC me_oracle.cpp -o libme_oracle.so   (oracle/oracle.py does it), and the same
// source with -DORC_COUNT -> libme_oracle_count.so: the operation-counting scalar of "counted mode" (see real_t).

#include <algorithm>
#include <cmath>
#include <complex>
#include <cstdint>
#include <cstring>
#include <map>
#include <mutex>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

// Scalar type of the amplitude arithmetic.  Plain build: double.  Counted build (-DORC_COUNT, "counted mode" of
// SURVEY.md 8(d); BASELINE.json north_star "FLOPs per ME counted by the instrumented oracle"): a double that counts
// every addition/subtraction, multiplication, division and square root it takes part in.  The source is the same,
// so the counted build performs exactly the operations of the plain one.
#ifdef ORC_COUNT
struct OpCount { long add, mul, div, sqrt; };
static OpCount g_ops = {0, 0, 0, 0};  // the counted build is driven single-threaded (orc_count_ops)
struct real_t {
  double v;
  real_t() : v(0.0) {}
  real_t(double x) : v(x) {}
  real_t(int x) : v(x) {}
};
static inline real_t operator+(real_t a, real_t b) { g_ops.add++; return real_t(a.v + b.v); }
static inline real_t operator-(real_t a, real_t b) { g_ops.add++; return real_t(a.v - b.v); }
static inline real_t operator*(real_t a, real_t b) { g_ops.mul++; return real_t(a.v * b.v); }
static inline real_t operator/(real_t a, real_t b) { g_ops.div++; return real_t(a.v / b.v); }
static inline real_t operator-(real_t a) { return real_t(-a.v); }  // sign flip: not an arithmetic operation
static inline real_t& operator+=(real_t& a, real_t b) { a = a + b; return a; }
static inline real_t& operator-=(real_t& a, real_t b) { a = a - b; return a; }
static inline real_t& operator*=(real_t& a, real_t b) { a = a * b; return a; }
static inline real_t& operator/=(real_t& a, real_t b) { a = a / b; return a; }
static inline bool operator==(real_t a, real_t b) { return a.v == b.v; }
static inline bool operator!=(real_t a, real_t b) { return a.v != b.v; }
static inline bool operator<(real_t a, real_t b) { return a.v < b.v; }
static inline bool operator>(real_t a, real_t b) { return a.v > b.v; }
static inline bool operator>=(real_t a, real_t b) { return a.v >= b.v; }
static inline real_t SQRT(real_t a) { g_ops.sqrt++; return real_t(std::sqrt(a.v)); }
static inline double to_double(real_t a) { return a.v; }
#elif defined(ORC_QUAD)
// Quadruple-precision build (-DORC_QUAD -> libme_oracle_quad.so): the same source with a 113-bit scalar (libquadmath).
// The arbiter of the accuracy-tail test: where the fp64 oracle and the fp64 CUDA path disagree beyond the tolerance
// (cancellations in nearly collinear events), this build says which of the two is off.
#include <quadmath.h>
typedef __float128 real_t;
static inline real_t SQRT(real_t a) { return sqrtq(a); }
static inline double to_double(real_t a) { return (double)a; }
#else
typedef double real_t;
static inline double SQRT(double a) { return std::sqrt(a); }
static inline double to_double(double a) { return a; }
#endif
typedef std::complex<real_t> cd;
typedef std::complex<double> cdd;  // colour algebra (Gell-Mann matrices, colour matrix): never counted
// |z|^2 = re^2 + im^2 (what std::norm does for double; written out so that the counted scalar sees it)
static inline real_t cnorm(const cd& z) { return z.real() * z.real() + z.imag() * z.imag(); }
// complex division: the library routine in the plain build, the textbook formula for the counted scalar
static inline cd cdiv(const cd& a, const cd& b) {
#ifdef ORC_COUNT
  real_t n = cnorm(b);
  return cd((a.real() * b.real() + a.imag() * b.imag()) / n, (a.imag() * b.real() - a.real() * b.imag()) / n);
#else
  return a / b;
#endif
}
static const cd I_(0.0, 1.0);

// ----------------------------------------------------------------------------------------------
// Lorentz and Dirac algebra.  Metric (+,-,-,-); 4-vectors carry UPPER indices (v[0]=E or time).
// ----------------------------------------------------------------------------------------------
struct V4 {  // complex 4-vector
  cd c[4];
};
struct Sp {  // 4-component spinor (column u/v or row ubar/vbar, by context)
  cd c[4];
};
struct M4 {  // 4x4 complex matrix
  cd m[4][4];
};

static inline cd mdot(const V4& a, const V4& b) {  // a.b with the metric, no conjugation
  return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3];
}
static inline V4 vreal(const double* p) {
  V4 r;
  for (int i = 0; i < 4; i++) r.c[i] = p[i];
  return r;
}
static inline V4 vadd(const V4& a, const V4& b) {
  V4 r;
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] + b.c[i];
  return r;
}
static inline V4 vsub(const V4& a, const V4& b) {
  V4 r;
  for (int i = 0; i < 4; i++) r.c[i] = a.c[i] - b.c[i];
  return r;
}
static inline V4 vscale(cd s, const V4& a) {
  V4 r;
  for (int i = 0; i < 4; i++) r.c[i] = s * a.c[i];
  return r;
}

// a-slash = gamma^mu a_mu in the Dirac representation, written out:
//   gamma^0 = diag(1,1,-1,-1), gamma^i = [[0, sigma^i], [-sigma^i, 0]]
//   => a-slash = [[ a0*1, -a.sigma ], [ a.sigma, -a0*1 ]],  a.sigma = [[a3, a1 - i a2], [a1 + i a2, -a3]]
// (tests/test_oracle_algebra.py checks this against the Clifford algebra built from Pauli matrices)
static M4 slash(const V4& a) {
  M4 r;
  cd a0 = a.c[0], a1 = a.c[1], a2 = a.c[2], a3 = a.c[3];
  cd s00 = a3, s01 = a1 - I_ * a2, s10 = a1 + I_ * a2, s11 = -a3;
  cd z(0.0, 0.0);
  r.m[0][0] = a0;  r.m[0][1] = z;   r.m[0][2] = -s00; r.m[0][3] = -s01;
  r.m[1][0] = z;   r.m[1][1] = a0;  r.m[1][2] = -s10; r.m[1][3] = -s11;
  r.m[2][0] = s00; r.m[2][1] = s01; r.m[2][2] = -a0;  r.m[2][3] = z;
  r.m[3][0] = s10; r.m[3][1] = s11; r.m[3][2] = z;    r.m[3][3] = -a0;
  return r;
}
static Sp row_times(const Sp& r, const M4& m) {  // (row) * M
  Sp o;
  for (int j = 0; j < 4; j++) {
    cd s(0, 0);
    for (int i = 0; i < 4; i++) s += r.c[i] * m.m[i][j];
    o.c[j] = s;
  }
  return o;
}
static Sp times_col(const M4& m, const Sp& c) {  // M * (column)
  Sp o;
  for (int i = 0; i < 4; i++) {
    cd s(0, 0);
    for (int j = 0; j < 4; j++) s += m.m[i][j] * c.c[j];
    o.c[i] = s;
  }
  return o;
}
static cd row_col(const Sp& r, const Sp& c) {
  cd s(0, 0);
  for (int i = 0; i < 4; i++) s += r.c[i] * c.c[i];
  return s;
}
static M4 madd_mass(const M4& a, real_t m) {  // a + m*1
  M4 r = a;
  for (int i = 0; i < 4; i++) r.m[i][i] += m;
  return r;
}
static Sp bar(const Sp& u) {  // u^dagger gamma^0, gamma^0 = diag(1,1,-1,-1)
  Sp r;
  r.c[0] = std::conj(u.c[0]);
  r.c[1] = std::conj(u.c[1]);
  r.c[2] = -std::conj(u.c[2]);
  r.c[3] = -std::conj(u.c[3]);
  return r;
}
// chirality projectors in the Dirac representation: gamma^5 = [[0,1],[1,0]] (2x2 blocks)
static M4 chiral_coupling(real_t gL, real_t gR) {  // gL*P_L + gR*P_R, P_L/R = (1 -/+ gamma5)/2
  M4 r;
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) r.m[i][j] = 0.0;
  real_t d = 0.5 * (gL + gR), o = 0.5 * (gR - gL);
  for (int i = 0; i < 4; i++) r.m[i][i] = d;
  r.m[0][2] = o; r.m[1][3] = o; r.m[2][0] = o; r.m[3][1] = o;
  return r;
}
static M4 mmul(const M4& a, const M4& b) {
  M4 r;
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) {
      cd s(0, 0);
      for (int k = 0; k < 4; k++) s += a.m[i][k] * b.m[k][j];
      r.m[i][j] = s;
    }
  return r;
}

// ----------------------------------------------------------------------------------------------
// External wavefunctions (lambda = +-1 is the PHYSICAL helicity in the frame
// of the given momenta).  Two-component helicity spinors chi_lambda(p), sigma.phat chi = lambda chi.
// ----------------------------------------------------------------------------------------------
static void chi(const double* p, int lam, cd out[2]) {
  real_t px = p[1], py = p[2], pz = p[3];
  real_t pp = SQRT(px * px + py * py + pz * pz);
  if (pp == 0.0) {  // particle at rest: quantise along +z (reading R9)
    if (lam > 0) { out[0] = 1.0; out[1] = 0.0; } else { out[0] = 0.0; out[1] = 1.0; }
    return;
  }
  if (px == 0.0 && py == 0.0 && pz < 0.0) {  // exactly along -z
    if (lam > 0) { out[0] = 0.0; out[1] = 1.0; } else { out[0] = -1.0; out[1] = 0.0; }
    return;
  }
  real_t n = 1.0 / SQRT(2.0 * pp * (pp + pz));
  if (lam > 0) { out[0] = n * (pp + pz); out[1] = n * cd(px, py); }
  else         { out[0] = n * cd(-px, py); out[1] = n * (pp + pz); }
}
// u(p,lambda): particle spinor, Dirac representation: ( sqrt(E+m) chi ; lambda |p|/sqrt(E+m) chi )
static Sp spinor_u(const double* p, real_t m, int lam) {
  real_t pp = SQRT(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  real_t up = SQRT(p[0] + m), lo = (up > 0.0) ? pp / up : 0.0;
  cd x[2];
  chi(p, lam, x);
  Sp u;
  u.c[0] = up * x[0]; u.c[1] = up * x[1];
  u.c[2] = real_t(lam) * lo * x[0]; u.c[3] = real_t(lam) * lo * x[1];
  return u;
}
// v(p,lambda): antiparticle spinor of physical helicity lambda: ( -lambda |p|/sqrt(E+m) chi_{-lambda} ; sqrt(E+m) chi_{-lambda} )
static Sp spinor_v(const double* p, real_t m, int lam) {
  real_t pp = SQRT(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  real_t up = SQRT(p[0] + m), lo = (up > 0.0) ? pp / up : 0.0;
  cd x[2];
  chi(p, -lam, x);
  Sp v;
  v.c[0] = -real_t(lam) * lo * x[0]; v.c[1] = -real_t(lam) * lo * x[1];
  v.c[2] = up * x[0]; v.c[3] = up * x[1];
  return v;
}
// polarisation vector of a massless vector, helicity lambda: eps = (-lambda*e1 - i e2)/sqrt(2)
static V4 polvec(const double* p, int lam) {
  real_t px = p[1], py = p[2], pz = p[3];
  real_t pt2 = px * px + py * py, pt = SQRT(pt2), pp = SQRT(pt2 + pz * pz);
  real_t e1[3], e2[3];
  if (pt == 0.0) {
    e1[0] = 1; e1[1] = 0; e1[2] = 0;
    e2[0] = 0; e2[1] = (pz >= 0 ? 1.0 : -1.0); e2[2] = 0;
  } else {
    e1[0] = px * pz / (pp * pt); e1[1] = py * pz / (pp * pt); e1[2] = -pt2 / (pp * pt);
    e2[0] = -py / pt; e2[1] = px / pt; e2[2] = 0;
  }
  V4 e;
  e.c[0] = 0.0;
  real_t s = 1.0 / SQRT(2.0);
  for (int i = 0; i < 3; i++) e.c[i + 1] = s * cd(-real_t(lam) * e1[i], -e2[i]);
  return e;
}
static V4 vconj(const V4& a) {
  V4 r;
  for (int i = 0; i < 4; i++) r.c[i] = std::conj(a.c[i]);
  return r;
}

// ----------------------------------------------------------------------------------------------
// Parameters
// ----------------------------------------------------------------------------------------------
struct Params {
  real_t mt, wt, mz, wz, aewm1, gf;
};
static Params params_from(const double* p) {
  Params q;
  if (p) { q.mt = p[0]; q.wt = p[1]; q.mz = p[2]; q.wz = p[3]; q.aewm1 = p[4]; q.gf = p[5]; }
  else { q.mt = 173.0; q.wt = 1.4915; q.mz = 91.188; q.wz = 2.441; q.aewm1 = 132.507; q.gf = 1.16639e-5; }
  return q;
}

// ----------------------------------------------------------------------------------------------
// e+ e- -> mu+ mu-  (particles: 0 = e+ in, 1 = e- in, 2 = mu+ out, 3 = mu- out)
//   M = e^2 [vbar(e+) g^mu u(e-)] [ubar(mu-) g_mu v(mu+)] / s
//     + [vbar(e+) g^mu (gL PL + gR PR) u(e-)] [ubar(mu-) g_mu (gL PL + gR PR) v(mu+)] / (s - MZ^2 + i MZ GZ)
// (alpha, G_F, M_Z) scheme for sin^2 theta_W (reading R5).  The q_mu q_nu / MZ^2 term of the
// Z propagator vanishes for massless leptons.
// ----------------------------------------------------------------------------------------------
static void ew_couplings(const Params& P, real_t& e, real_t& gL, real_t& gR) {
  const real_t pi = M_PI;
  real_t alpha = 1.0 / P.aewm1;
  real_t mz2 = P.mz * P.mz;
  real_t mw2 = 0.5 * mz2 + SQRT(0.25 * mz2 * mz2 - pi * alpha * mz2 / (SQRT(2.0) * P.gf));
  real_t sw2 = 1.0 - mw2 / mz2;
  real_t sw = SQRT(sw2), cw = SQRT(1.0 - sw2);
  e = SQRT(4.0 * pi * alpha);
  gL = e / (sw * cw) * (-0.5 + sw2);
  gR = e / (sw * cw) * sw2;
}
static cd amp_eemumu(const Params& P, const double* mom, const int* hel) {
  real_t e, gL, gR;
  ew_couplings(P, e, gL, gR);
  Sp vb = bar(spinor_v(mom + 0, 0.0, hel[0]));  // incoming e+ : vbar
  Sp u = spinor_u(mom + 4, 0.0, hel[1]);        // incoming e- : u
  Sp v = spinor_v(mom + 8, 0.0, hel[2]);        // outgoing mu+: v
  Sp ub = bar(spinor_u(mom + 12, 0.0, hel[3])); // outgoing mu-: ubar
  real_t q[4];
  for (int i = 0; i < 4; i++) q[i] = mom[i] + mom[4 + i];
  real_t s = q[0] * q[0] - q[1] * q[1] - q[2] * q[2] - q[3] * q[3];
  M4 gz = chiral_coupling(gL, gR);
  // currents J^mu = vbar gamma^mu X u, computed with unit vectors through slash()
  cd amp(0, 0);
  for (int mu = 0; mu < 4; mu++) {
    V4 unit;
    for (int i = 0; i < 4; i++) unit.c[i] = 0.0;
    unit.c[mu] = (mu == 0) ? 1.0 : -1.0;  // slash(unit) = gamma^mu g_{mu mu} * (+-1) -> gamma^mu
    M4 g = slash(unit);
    real_t gmm = (mu == 0) ? 1.0 : -1.0;  // metric for the contraction J1^mu J2_mu
    cd j1g = row_col(vb, times_col(g, u));
    cd j2g = row_col(ub, times_col(g, v));
    cd j1z = row_col(vb, times_col(mmul(g, gz), u));
    cd j2z = row_col(ub, times_col(mmul(g, gz), v));
    amp += gmm * (e * e * j1g * j2g / s + cdiv(j1z * j2z, cd(s - P.mz * P.mz, P.mz * P.wz)));
  }
  return amp;
}

// ----------------------------------------------------------------------------------------------
// g g -> t tbar + (n-2) g : diagram enumeration.
// Particles: 0,1 = incoming g; 2 = t (out); 3 = tbar (out); 4.. = outgoing g.
// Every tree diagram is the quark line from t to tbar with m >= 1 gluon trees attached in order;
// the trees partition the n gluons.  A gluon tree over a leg set S is a leaf (|S| = 1), a
// three-gluon vertex joining trees on a 2-partition of S, or a four-gluon vertex joining trees on a
// 3-partition of S (three colour/Lorentz terms).
// ----------------------------------------------------------------------------------------------
typedef std::complex<int> ci;
typedef std::map<std::vector<int>, ci> ColExp;  // sum of coef * T^{a_s1} T^{a_s2} ... over strings s of legs

static ColExp col_mul(const ColExp& a, const ColExp& b, ci f) {  // f * a.b (string concatenation)
  ColExp r;
  for (auto& x : a)
    for (auto& y : b) {
      std::vector<int> s = x.first;
      s.insert(s.end(), y.first.begin(), y.first.end());
      r[s] += f * x.second * y.second;
    }
  return r;
}
static void col_acc(ColExp& r, const ColExp& a, ci f) {
  for (auto& x : a) r[x.first] += f * x.second;
}
static ColExp col_comm(const ColExp& a, const ColExp& b, ci f) {  // f * [a, b]
  ColExp r = col_mul(a, b, f);
  col_acc(r, col_mul(b, a, f), ci(-1, 0));
  for (auto it = r.begin(); it != r.end();)
    if (it->second == ci(0, 0)) it = r.erase(it); else ++it;
  return r;
}

struct Tree {
  int kind;       // 0 leaf, 3 three-gluon vertex, 4 four-gluon vertex, 5 electroweak boson decaying to the lepton pair
  int term;       // four-gluon vertex: which of the three f.f terms (0,1,2); boson: 0 photon, 1 Z
  int ch[3];      // child tree ids
  int leg;        // leaf: particle index
  unsigned mask;  // set of particle indices below this tree
  ColExp col;     // sum_x (colour tensor)^x T^x expanded on strings
};
struct TrieNode {
  int parent;     // trie node id of the prefix without the last tree (-1 for the root = empty prefix)
  int tree;       // last attached tree
  unsigned mask;  // gluon legs in the prefix
};
struct SubDiagram {
  int prefix;  // trie node: all blocks but the last
  int last;    // tree attached next to tbar
  int diag;    // Feynman diagram number (the three terms of a four-gluon vertex share it)
  std::vector<std::pair<int, ci>> K;  // (colour flow index, coefficient in {+-1, +-i})
};
struct Process {
  int id, npar, ngl, ncomb, ncol, ndiag, denom;
  // fermion line: the row spinor sits at the END of the fermion arrow, the column spinor at its start.
  //   gg -> t tbar + gluons : row = ubar(t) (particle 2, outgoing quark), column = v(tbar) (particle 3), mass m_t
  //   g ubar -> tau+ tau- + gluons + ubar : row = vbar(ubar in) (particle 1, incoming antiquark), column = v(ubar out)
  //   (the last particle), massless; ew = true: one photon / Z -> tau- (3) tau+ (2) is attached to the line
  int row_leg, col_leg, lep_m, lep_p;
  bool ew;
  std::vector<int> gl;  // gluon particle indices
  std::vector<Tree> trees;
  std::map<unsigned, std::vector<int>> trees_of;  // leg set -> tree ids
  std::vector<TrieNode> trie;
  std::vector<SubDiagram> sub;
  std::vector<std::vector<int>> flows;  // [ncol][ngl] gluon particle indices, lexicographic permutations
  std::map<std::vector<int>, int> flow_index;
  std::vector<double> C;  // colour matrix [ncol][ncol]
  long ndiag_counted;
  // multichannel (reading R17): channel = Feynman diagram, numbered by its structural key
  std::vector<std::string> chan_keys;  // [ndiag], sorted
  std::vector<int> chan_of_sub;        // [nsub] channel of every sub-diagram (the terms of a four-gluon vertex share it)
};

static int lowbit(unsigned m) { return __builtin_ctz(m); }

static const std::vector<int>& build_trees(Process& P, unsigned mask) {
  auto it = P.trees_of.find(mask);
  if (it != P.trees_of.end()) return it->second;
  std::vector<int> out;
  if (__builtin_popcount(mask) == 1) {
    Tree t;
    t.kind = 0; t.term = 0; t.leg = lowbit(mask); t.mask = mask; t.ch[0] = t.ch[1] = t.ch[2] = -1;
    t.col[std::vector<int>{t.leg}] = ci(1, 0);
    P.trees.push_back(t);
    out.push_back((int)P.trees.size() - 1);
  } else {
    unsigned lb = 1u << lowbit(mask);
    // three-gluon vertex: unordered 2-partitions {A,B}, A contains the lowest leg
    for (unsigned A = mask; A; A = (A - 1) & mask) {
      if (!(A & lb) || A == mask) continue;
      unsigned B = mask ^ A;
      std::vector<int> ta = build_trees(P, A), tb = build_trees(P, B);
      for (int a : ta)
        for (int b : tb) {
          Tree t;
          t.kind = 3; t.term = 0; t.leg = -1; t.mask = mask; t.ch[0] = a; t.ch[1] = b; t.ch[2] = -1;
          // sum_x f^{abx} T^x = -i [T^a, T^b]
          t.col = col_comm(P.trees[a].col, P.trees[b].col, ci(0, -1));
          P.trees.push_back(t);
          out.push_back((int)P.trees.size() - 1);
        }
    }
    // four-gluon vertex: unordered 3-partitions {A,B,C}, lowest leg in A, lowest of the rest in B
    for (unsigned A = mask; A; A = (A - 1) & mask) {
      if (!(A & lb) || A == mask) continue;
      unsigned rest = mask ^ A;
      unsigned lb2 = 1u << lowbit(rest);
      for (unsigned B = rest; B; B = (B - 1) & rest) {
        if (!(B & lb2) || B == rest) continue;
        unsigned Cm = rest ^ B;
        std::vector<int> ta = build_trees(P, A), tb = build_trees(P, B), tc = build_trees(P, Cm);
        for (int a : ta)
          for (int b : tb)
            for (int c : tc)
              for (int term = 0; term < 3; term++) {
                Tree t;
                t.kind = 4; t.term = term; t.leg = -1; t.mask = mask; t.ch[0] = a; t.ch[1] = b; t.ch[2] = c;
                const ColExp &ca = P.trees[a].col, &cb = P.trees[b].col, &cc = P.trees[c].col;
                // colour of the parent line x (fourth leg d = x):
                //  term 0: f^{abe} f^{cxe}: sum_x T^x (..) = -[[a,b],c]
                //  term 1: f^{ace} f^{bxe}:                 = -[[a,c],b]
                //  term 2: f^{axe} f^{bce}:                 = -[[b,c],a]
                if (term == 0) t.col = col_comm(col_comm(ca, cb, ci(1, 0)), cc, ci(-1, 0));
                if (term == 1) t.col = col_comm(col_comm(ca, cc, ci(1, 0)), cb, ci(-1, 0));
                if (term == 2) t.col = col_comm(col_comm(cb, cc, ci(1, 0)), ca, ci(-1, 0));
                P.trees.push_back(t);
                out.push_back((int)P.trees.size() - 1);
              }
      }
    }
  }
  P.trees_of[mask] = out;
  return P.trees_of[mask];
}

// number of Feynman diagrams of a gluon tree set (a four-gluon vertex counts once)
static long count_tree_diagrams(Process& P, int t) {
  const Tree& T = P.trees[t];
  if (T.kind == 0) return 1;
  long c = 1;
  for (int k = 0; k < 3; k++)
    if (T.ch[k] >= 0) c *= count_tree_diagrams(P, T.ch[k]);
  return c;
}

// the electroweak "trees" of a process with ew = true: the photon and the Z attached to the lepton pair; they carry
// no colour (unit string), their leg set is the lepton pair
static std::vector<int> boson_trees(Process& P) {
  const unsigned lm = (1u << P.lep_m) | (1u << P.lep_p);
  auto it = P.trees_of.find(lm);
  if (it != P.trees_of.end()) return it->second;
  std::vector<int> out;
  for (int b = 0; b < 2; b++) {
    Tree t;
    t.kind = 5; t.term = b; t.leg = -1; t.mask = lm; t.ch[0] = t.ch[1] = t.ch[2] = -1;
    t.col[std::vector<int>()] = ci(1, 0);
    P.trees.push_back(t);
    out.push_back((int)P.trees.size() - 1);
  }
  P.trees_of[lm] = out;
  return out;
}

// remaining: gluon legs not yet attached; boson_left: the electroweak boson is still to be attached
static void enumerate_lines(Process& P, unsigned remaining, bool boson_left, int node, const ColExp& prefix_col, long& ndiag) {
  // choose the next block: any non-empty subset of the remaining gluons with one of its trees, or the boson
  std::vector<std::pair<unsigned, int>> choices;  // (gluon legs used, tree)
  for (unsigned B = remaining; B; B = (B - 1) & remaining)
    for (int t : build_trees(P, B)) choices.push_back(std::make_pair(B, t));
  if (boson_left)
    for (int t : boson_trees(P)) choices.push_back(std::make_pair(0u, t));
  for (auto& ch : choices) {
    const unsigned B = ch.first;
    const int t = ch.second;
    const bool is_boson = (P.trees[t].kind == 5);
    const bool left_after = boson_left && !is_boson;
    {
      ColExp col = col_mul(prefix_col, P.trees[t].col, ci(1, 0));
      if (B == remaining && !left_after) {  // last block: a complete (sub)diagram
        SubDiagram d;
        d.prefix = node;
        d.last = t;
        // diagram numbering: the three terms of each four-gluon vertex belong to one diagram.
        // count 1 for term-0-only trees (a tree whose every V4 has term 0), 0 otherwise.
        bool first_terms = true;
        std::vector<int> stack{t};
        for (int n2 = node; n2 > 0; n2 = P.trie[n2].parent) stack.push_back(P.trie[n2].tree);
        while (!stack.empty()) {
          int x = stack.back();
          stack.pop_back();
          if (P.trees[x].kind == 4 && P.trees[x].term != 0) first_terms = false;
          for (int k = 0; k < 3; k++)
            if (P.trees[x].ch[k] >= 0) stack.push_back(P.trees[x].ch[k]);
        }
        if (first_terms) ndiag++;
        d.diag = (int)ndiag - 1;  // only meaningful for first_terms; others get the running number
        for (auto& s : col) {
          if (s.second == ci(0, 0)) continue;
          auto f = P.flow_index.find(s.first);
          d.K.push_back(std::make_pair(f->second, s.second));
        }
        P.sub.push_back(d);
      } else {
        TrieNode nd;
        nd.parent = node; nd.tree = t; nd.mask = (node >= 0 ? P.trie[node].mask : 0u) | P.trees[t].mask;
        P.trie.push_back(nd);
        enumerate_lines(P, remaining ^ B, left_after, (int)P.trie.size() - 1, col, ndiag);
      }
    }
  }
}

// ---- SU(3): Gell-Mann matrices, T^a = lambda^a/2, f^{abc} = -2i Tr([T^a,T^b] T^c) ----
struct SU3 {
  cdd T[8][3][3];
  double f[8][8][8];
  SU3() {
    memset(T, 0, sizeof(T));
    cdd i(0, 1);
    T[0][0][1] = 1; T[0][1][0] = 1;
    T[1][0][1] = -i; T[1][1][0] = i;
    T[2][0][0] = 1; T[2][1][1] = -1;
    T[3][0][2] = 1; T[3][2][0] = 1;
    T[4][0][2] = -i; T[4][2][0] = i;
    T[5][1][2] = 1; T[5][2][1] = 1;
    T[6][1][2] = -i; T[6][2][1] = i;
    double s3 = 1.0 / std::sqrt(3.0);
    T[7][0][0] = s3; T[7][1][1] = s3; T[7][2][2] = -2.0 * s3;
    for (int a = 0; a < 8; a++)
      for (int r = 0; r < 3; r++)
        for (int c = 0; c < 3; c++) T[a][r][c] *= 0.5;
    for (int a = 0; a < 8; a++)
      for (int b = 0; b < 8; b++)
        for (int c = 0; c < 8; c++) {
          cdd tr(0, 0);
          for (int r = 0; r < 3; r++)
            for (int s = 0; s < 3; s++)
              for (int t = 0; t < 3; t++)
                tr += (T[a][r][s] * T[b][s][t] - T[b][r][s] * T[a][s][t]) * T[c][t][r];
          f[a][b][c] = (cdd(0, -2) * tr).real();
        }
  }
};
static const SU3& su3() {
  static SU3 s;
  return s;
}

struct Mat3 {
  cdd m[3][3];
};
static Mat3 m3mul(const Mat3& a, const Mat3& b) {
  Mat3 r;
  for (int i = 0; i < 3; i++)
    for (int j = 0; j < 3; j++) {
      cdd s(0, 0);
      for (int k = 0; k < 3; k++) s += a.m[i][k] * b.m[k][j];
      r.m[i][j] = s;
    }
  return r;
}

// colour matrix C_{sigma tau} = sum_{a_1..a_n} sum_{ij} (T^{a_s1}..T^{a_sn})_{ij} conj((T^{a_t1}..T^{a_tn})_{ij})
// brute force over all 8^n adjoint assignments with explicit Gell-Mann matrices.
static void build_color_matrix(Process& P) {
  const SU3& S = su3();
  int n = P.ngl, nc = P.ncol;
  P.C.assign((size_t)nc * nc, 0.0);
  long nass = 1;
  for (int k = 0; k < n; k++) nass *= 8;
  std::vector<double> acc((size_t)nc * nc, 0.0);
#pragma omp parallel
  {
    std::vector<double> loc((size_t)nc * nc, 0.0);
    std::vector<Mat3> str(nc);
#pragma omp for schedule(static)
    for (long ass = 0; ass < nass; ass++) {
      int a[8];
      long x = ass;
      for (int k = 0; k < n; k++) { a[k] = (int)(x % 8); x /= 8; }  // a[k]: colour of gluon P.gl[k]
      for (int s = 0; s < nc; s++) {
        Mat3 m;
        for (int i = 0; i < 3; i++)
          for (int j = 0; j < 3; j++) m.m[i][j] = (i == j) ? 1.0 : 0.0;
        for (int k = 0; k < n; k++) {
          int leg = P.flows[s][k];
          int pos = (int)(std::find(P.gl.begin(), P.gl.end(), leg) - P.gl.begin());
          Mat3 t;
          memcpy(t.m, S.T[a[pos]], sizeof(t.m));
          m = m3mul(m, t);
        }
        str[s] = m;
      }
      for (int s = 0; s < nc; s++)
        for (int t = 0; t < nc; t++) {
          cdd tr(0, 0);
          for (int i = 0; i < 3; i++)
            for (int j = 0; j < 3; j++) tr += str[s].m[i][j] * std::conj(str[t].m[i][j]);
          loc[(size_t)s * nc + t] += tr.real();
        }
    }
#pragma omp critical
    for (size_t k = 0; k < loc.size(); k++) acc[k] += loc[k];
  }
  P.C = acc;
}

// Structural key of a gluon tree and of a Feynman diagram (reading R17): a leaf is its particle index, a
// three-gluon vertex "(A,B)" with the lowest leg in A, a four-gluon vertex "[A,B,C]" with the lowest leg in A and the
// lowest of the rest in B; a diagram is the keys of the trees attached to the quark line from t to tbar joined by "|".
// Channels are the distinct keys in increasing (byte-wise) order: the three colour-structure terms of a four-gluon
// vertex belong to one diagram, hence to one channel.
static std::string tree_key(const Process& P, int t) {
  const Tree& T = P.trees[t];
  if (T.kind == 0) return std::to_string(T.leg);
  if (T.kind == 5) return T.term == 0 ? "a" : "z";
  if (T.kind == 3) return "(" + tree_key(P, T.ch[0]) + "," + tree_key(P, T.ch[1]) + ")";
  return "[" + tree_key(P, T.ch[0]) + "," + tree_key(P, T.ch[1]) + "," + tree_key(P, T.ch[2]) + "]";
}
static void build_channels(Process& P) {
  std::vector<std::string> keys(P.sub.size());
  for (size_t d = 0; d < P.sub.size(); d++) {
    std::vector<int> blocks{P.sub[d].last};
    for (int n = P.sub[d].prefix; n > 0; n = P.trie[n].parent) blocks.push_back(P.trie[n].tree);
    std::string k;
    for (size_t i = blocks.size(); i-- > 0;) { k += tree_key(P, blocks[i]); if (i) k += "|"; }
    keys[d] = k;
  }
  P.chan_keys = keys;
  std::sort(P.chan_keys.begin(), P.chan_keys.end());
  P.chan_keys.erase(std::unique(P.chan_keys.begin(), P.chan_keys.end()), P.chan_keys.end());
  P.chan_of_sub.resize(P.sub.size());
  for (size_t d = 0; d < P.sub.size(); d++)
    P.chan_of_sub[d] = (int)(std::lower_bound(P.chan_keys.begin(), P.chan_keys.end(), keys[d]) - P.chan_keys.begin());
}

static Process* build_process(int id) {
  Process* P = new Process();
  P->id = id;
  if (id == 0) {
    P->npar = 4; P->ngl = 0; P->ncomb = 16; P->ncol = 1; P->ndiag = 2; P->denom = 4;
    P->C.assign(1, 1.0);
    P->flows.push_back(std::vector<int>());
    return P;
  }
  int n;  // gluons
  if (id <= 4) {
    n = id + 1;
    P->ngl = n; P->npar = n + 2; P->ncomb = 1 << P->npar;
    P->gl.push_back(0); P->gl.push_back(1);
    for (int k = 4; k < P->npar; k++) P->gl.push_back(k);
    P->row_leg = 2; P->col_leg = 3; P->lep_m = P->lep_p = -1; P->ew = false;
  } else {
    // g ubar -> tau+ tau- + (n-1) g + ubar: 0 = g, 1 = ubar (in), 2 = tau+, 3 = tau-, 4.. = g, last = ubar (out)
    n = id - 4;
    P->ngl = n; P->npar = n + 4; P->ncomb = 1 << P->npar;
    P->gl.push_back(0);
    for (int k = 4; k < P->npar - 1; k++) P->gl.push_back(k);
    P->row_leg = 1; P->col_leg = P->npar - 1; P->lep_p = 2; P->lep_m = 3; P->ew = true;
  }
  // colour flows: permutations of the gluon particle indices in lexicographic order
  std::vector<int> perm = P->gl;
  std::sort(perm.begin(), perm.end());
  do {
    P->flow_index[perm] = (int)P->flows.size();
    P->flows.push_back(perm);
  } while (std::next_permutation(perm.begin(), perm.end()));
  P->ncol = (int)P->flows.size();
  if (id <= 4) {
    // denominators: 2*2 gluon spins, 8*8 gluon colours, (n-2)! identical final-state gluons
    int fact = 1;
    for (int k = 2; k <= n - 2; k++) fact *= k;
    P->denom = 4 * 64 * fact;
  } else {
    // 2*2 initial spins, 8*3 initial colours, (n-1)! identical final-state gluons
    int fact = 1;
    for (int k = 2; k <= n - 1; k++) fact *= k;
    P->denom = 4 * 24 * fact;
  }
  unsigned all = 0;
  for (int g : P->gl) all |= 1u << g;
  TrieNode root;
  root.parent = -1; root.tree = -1; root.mask = 0;
  P->trie.push_back(root);
  ColExp unit;
  unit[std::vector<int>()] = ci(1, 0);
  long nd = 0;
  enumerate_lines(*P, all, P->ew, 0, unit, nd);
  P->ndiag = (int)nd;
  build_color_matrix(*P);
  build_channels(*P);
  return P;
}
static Process* get_process(int id) {
  static Process* cache[8] = {0, 0, 0, 0, 0, 0, 0, 0};
  static std::mutex mtx;
  if (id < 0 || id > 7) return 0;
  std::lock_guard<std::mutex> lock(mtx);
  if (!cache[id]) cache[id] = build_process(id);
  return cache[id];
}

// helicity table: row h, particle k: lambda = +1 if bit (npar-1-k) of h is set, else -1 (reading R7)
static inline int hel_of(int h, int k, int npar) { return ((h >> (npar - 1 - k)) & 1) ? 1 : -1; }

// ----------------------------------------------------------------------------------------------
// Evaluation of all colour-flow amplitudes J_sigma for one event and one helicity.
// Literal Feynman rules (all momenta INCOMING to a vertex; k_i = +p_i for incoming, -p_i for outgoing):
//   quark-gluon vertex   i g_s gamma^mu T^a
//   quark propagator     i (q-slash + m) / (q^2 - m^2 + i m Gamma)       (q along the fermion arrow)
//   gluon propagator     -i g_{mu nu} delta^{ab} / k^2
//   three-gluon vertex   g_s f^{abc} [ g^{mu nu}(k1-k2)^rho + g^{nu rho}(k2-k3)^mu + g^{rho mu}(k3-k1)^nu ]
//   four-gluon vertex    -i g_s^2 [ f^{abe}f^{cde}(g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho})
//                                 + f^{ace}f^{bde}(g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho})
//                                 + f^{ade}f^{bce}(g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma}) ]
//   fermion-photon vertex  i e Q_f gamma^mu              fermion-Z vertex  i gamma^mu (gL_f P_L + gR_f P_R),
//                          gL_f = e (T3_f - Q_f sw^2)/(sw cw), gR_f = -e Q_f sw^2/(sw cw)   (u: Q = 2/3, T3 = 1/2;
//                          tau: Q = -1, T3 = -1/2; (alpha, G_F, M_Z) scheme, reading R5)
//   photon propagator      -i g_{mu nu} / q^2           Z propagator  -i g_{mu nu} / (q^2 - MZ^2 + i MZ GZ)
//                          (the q_mu q_nu term vanishes on the massless lepton current, reading R6)
// external: incoming g eps, outgoing g eps^*, outgoing quark ubar, outgoing antiquark v, incoming antiquark vbar.
// The electroweak boson with its lepton pair enters the quark line like a colourless gluon tree whose "current" is
//   V_B^mu = [ubar(tau-) i gamma^mu c_B^tau v(tau+)] (-i / D_B),   attached with the vertex i gamma_mu c_B^u
// ward_leg >= 0 replaces that gluon's polarisation by its momentum (gauge test); ward_leg = -2 replaces the lepton
// current by the boson momentum (conservation of the quark current, vector and axial for a massless line).
// ----------------------------------------------------------------------------------------------
struct Census {
  long v3, v4, chain, closure, jamp_terms;
};

static void eval_jamps(const Process& P, const Params& par, const double* mom, real_t gs, int h, int ward_leg,
                       std::vector<cd>& jamp, std::vector<cd>* amps, Census* census) {
  const int npar = P.npar;
  // incoming-convention momenta
  real_t k[8][4];
  for (int i = 0; i < npar; i++)
    for (int m = 0; m < 4; m++) k[i][m] = (i < 2 ? 1.0 : -1.0) * mom[4 * i + m];
  // gluon tree currents (upper index, propagator included, colour stripped)
  size_t nt = P.trees.size();
  std::vector<V4> cur(nt);
  std::vector<V4> kk(nt);  // momentum flowing from the tree towards its parent (sum of incoming k of its legs)
  for (size_t t = 0; t < nt; t++) {
    const Tree& T = P.trees[t];
    V4 K;
    for (int m = 0; m < 4; m++) K.c[m] = 0.0;
    for (int i = 0; i < npar; i++)
      if (T.mask & (1u << i))
        for (int m = 0; m < 4; m++) K.c[m] += k[i][m];
    kk[t] = K;
    if (T.kind == 0) {
      int lam = hel_of(h, T.leg, npar);
      if (T.leg == ward_leg) cur[t] = vreal(mom + 4 * T.leg);
      else {
        V4 e = polvec(mom + 4 * T.leg, lam);
        cur[t] = (T.leg < 2) ? e : vconj(e);
      }
      continue;
    }
    if (T.kind == 5) {
      // lepton current of boson B = T.term with its propagator (see the header of this function)
      real_t e, gLl, gRl;
      ew_couplings(par, e, gLl, gRl);
      Sp ubl = bar(spinor_u(mom + 4 * P.lep_m, 0.0, hel_of(h, P.lep_m, npar)));
      Sp vl = spinor_v(mom + 4 * P.lep_p, 0.0, hel_of(h, P.lep_p, npar));
      M4 cl = (T.term == 0) ? chiral_coupling(-e, -e) : chiral_coupling(gLl, gRl);   // Q_tau = -1
      cd s = mdot(K, K);
      cd D = (T.term == 0) ? s : s - par.mz * par.mz + I_ * par.mz * par.wz;
      V4 L;
      for (int mu = 0; mu < 4; mu++) {
        V4 unit;
        for (int i = 0; i < 4; i++) unit.c[i] = 0.0;
        unit.c[mu] = (mu == 0) ? 1.0 : -1.0;  // slash(unit) = gamma^mu (upper index)
        L.c[mu] = I_ * row_col(ubl, times_col(mmul(slash(unit), cl), vl));
      }
      if (ward_leg == -2) L = K;
      cur[t] = vscale(cdiv(-I_, D), L);
      continue;
    }
    V4 k3 = vscale(cd(-1.0), K);  // parent line momentum, incoming to this vertex
    cd k2 = mdot(K, K);
    cd prop = cdiv(-I_, k2);  // -i g_{mu nu} / k^2
    if (T.kind == 3) {
      const V4 &A = cur[T.ch[0]], &B = cur[T.ch[1]];
      const V4 &k1 = kk[T.ch[0]], &k2v = kk[T.ch[1]];
      // W^rho = (A.B)(k1-k2)^rho + B^rho ((k2-k3).A) + A^rho ((k3-k1).B)
      V4 W = vadd(vadd(vscale(mdot(A, B), vsub(k1, k2v)), vscale(mdot(vsub(k2v, k3), A), B)),
                  vscale(mdot(vsub(k3, k1), B), A));
      cur[t] = vscale(prop * gs, W);
      if (census) census->v3++;
    } else {
      const V4 &A = cur[T.ch[0]], &B = cur[T.ch[1]], &Cc = cur[T.ch[2]];
      V4 W;
      if (T.term == 0) W = vsub(vscale(mdot(A, Cc), B), vscale(mdot(B, Cc), A));       // g^{mu rho}g^{nu sigma} - g^{mu sigma}g^{nu rho}
      else if (T.term == 1) W = vsub(vscale(mdot(A, B), Cc), vscale(mdot(B, Cc), A));  // g^{mu nu}g^{rho sigma} - g^{mu sigma}g^{nu rho}
      else W = vsub(vscale(mdot(A, B), Cc), vscale(mdot(A, Cc), B));                   // g^{mu nu}g^{rho sigma} - g^{mu rho}g^{nu sigma}
      cur[t] = vscale(prop * (-I_ * gs * gs), W);
      if (census) census->v4++;
    }
  }
  // quark line
  const real_t mq = P.ew ? real_t(0.0) : par.mt, wq = P.ew ? real_t(0.0) : par.wt;
  const int lrow = hel_of(h, P.row_leg, npar), lcol = hel_of(h, P.col_leg, npar);
  Sp ub = P.ew ? bar(spinor_v(mom + 4 * P.row_leg, mq, lrow))   // incoming antiquark: vbar
               : bar(spinor_u(mom + 4 * P.row_leg, mq, lrow));  // outgoing quark: ubar
  Sp v = spinor_v(mom + 4 * P.col_leg, mq, lcol);               // outgoing antiquark: v
  // vertex of an attached block: i g_s gamma_mu J^mu for a gluon tree, i gamma_mu V^mu c_B^u for the boson
  real_t e_, gLl_, gRl_, gLu = 0.0, gRu = 0.0, eQu = 0.0;
  if (P.ew) {
    ew_couplings(par, e_, gLl_, gRl_);
    // gL_tau = e(-1/2 + sw^2)/(sw cw), gR_tau = e sw^2/(sw cw)  ->  e/(sw cw) = 2 (gR_tau - gL_tau), sw^2 = gR_tau / (e/(sw cw))
    real_t eosc = 2.0 * (gRl_ - gLl_), sw2 = gRl_ / eosc;
    eQu = e_ * (2.0 / 3.0);
    gLu = eosc * (0.5 - (2.0 / 3.0) * sw2);
    gRu = eosc * (-(2.0 / 3.0) * sw2);
  }
  auto attach = [&](const Sp& r, int tree) {
    const Tree& T = P.trees[tree];
    Sp x;
    if (T.kind == 5) {
      M4 cq = (T.term == 0) ? chiral_coupling(eQu, eQu) : chiral_coupling(gLu, gRu);
      x = row_times(r, mmul(slash(cur[tree]), cq));
      for (int i = 0; i < 4; i++) x.c[i] *= I_;
    } else {
      x = row_times(r, slash(cur[tree]));
      for (int i = 0; i < 4; i++) x.c[i] *= I_ * gs;
    }
    return x;
  };
  size_t nn = P.trie.size();
  std::vector<Sp> chain(nn);
  chain[0] = ub;
  for (size_t n = 1; n < nn; n++) {
    const TrieNode& N = P.trie[n];
    Sp x = attach(chain[N.parent], N.tree);
    // propagator: fermion-arrow momentum q = -(k_row + sum_prefix k) (k: incoming convention)
    V4 q;
    for (int m = 0; m < 4; m++) {
      real_t s = k[P.row_leg][m];
      for (int i = 0; i < npar; i++)
        if (N.mask & (1u << i)) s += k[i][m];
      q.c[m] = -s;
    }
    cd den = mdot(q, q) - mq * mq + I_ * mq * wq;
    Sp y = row_times(x, madd_mass(slash(q), mq));
    for (int i = 0; i < 4; i++) y.c[i] *= cdiv(I_, den);
    chain[n] = y;
    if (census) census->chain++;
  }
  jamp.assign(P.ncol, cd(0, 0));
  if (amps) amps->assign(P.sub.size(), cd(0, 0));
  for (size_t d = 0; d < P.sub.size(); d++) {
    const SubDiagram& D = P.sub[d];
    cd A = row_col(attach(chain[D.prefix], D.last), v);
    if (amps) (*amps)[d] = A;
    if (census) { census->closure++; census->jamp_terms += (long)D.K.size(); }
    for (auto& kc : D.K) jamp[kc.first] += cd(kc.second.real(), kc.second.imag()) * A;
  }
}

// |M_h|^2 = sum_{sigma,tau} conj(J_sigma) C_{sigma tau} J_tau  (plain real_t sum)
static real_t color_sum(const Process& P, const std::vector<cd>& J) {
  cd s(0, 0);
  for (int a = 0; a < P.ncol; a++)
    for (int b = 0; b < P.ncol; b++) s += std::conj(J[a]) * real_t(P.C[(size_t)a * P.ncol + b]) * J[b];
  return s.real();
}

// ----------------------------------------------------------------------------------------------
// C interface (ctypes).  proc: 0 ee_mumu, 1 gg_tt, 2 gg_ttg, 3 gg_ttgg, 4 gg_ttggg, 5/6/7 g ubar -> tau+ tau- ubar + 0/1/2 g.
// ----------------------------------------------------------------------------------------------
extern "C" {

int orc_info(int proc, int* npar, int* ncomb, int* ncol, int* ndiag, int* denom) {
  Process* P = get_process(proc);
  if (!P) return -1;
  *npar = P->npar; *ncomb = P->ncomb; *ncol = P->ncol; *ndiag = P->ndiag; *denom = P->denom;
  return 0;
}
int orc_counts(int proc, long* ntrees, long* ntrie, long* nsub) {
  Process* P = get_process(proc);
  if (!P) return -1;
  *ntrees = (long)P->trees.size(); *ntrie = (long)P->trie.size(); *nsub = (long)P->sub.size();
  return 0;
}
int orc_helicity_table(int proc, int8_t* out) {
  Process* P = get_process(proc);
  if (!P) return -1;
  for (int h = 0; h < P->ncomb; h++)
    for (int k = 0; k < P->npar; k++) out[h * P->npar + k] = (int8_t)hel_of(h, k, P->npar);
  return 0;
}
int orc_color_table(int proc, int8_t* out) {
  Process* P = get_process(proc);
  if (!P) return -1;
  for (int c = 0; c < P->ncol; c++)
    for (int k = 0; k < P->ngl; k++) out[c * P->ngl + k] = (int8_t)P->flows[c][k];
  return 0;
}
int orc_color_matrix(int proc, double* out) {
  Process* P = get_process(proc);
  if (!P) return -1;
  memcpy(out, P->C.data(), sizeof(double) * P->C.size());
  return 0;
}

// per-event, per-helicity |M_h|^2 (NOT divided by denom) and per-(helicity,colour) |J_c(h)|^2
//   mhel  [nevt][ncomb]      (required)
//   jamp2 [nevt][ncomb][ncol] or NULL
// mask[ncomb] (or NULL = all): helicities with mask 0 are skipped and reported as 0.
int orc_me_helicities(int proc, const double* params, const double* mom, const double* gs, int64_t nevt,
                      const uint8_t* mask, double* mhel, double* jamp2, int nthreads) {
  Process* P = get_process(proc);
  if (!P) return -1;
  Params par = params_from(params);
  const int npar = P->npar, ncomb = P->ncomb, ncol = P->ncol;
  // threads of THIS call only (no omp_set_num_threads: it would change the process-wide setting)
#ifdef _OPENMP
  const int nt = (nthreads > 0) ? nthreads : omp_get_max_threads();
#else
  const int nt = 1;
#endif
  (void)nt;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
  for (int64_t e = 0; e < nevt; e++) {
    const double* pm = mom + (size_t)e * npar * 4;
    std::vector<cd> J;
    for (int h = 0; h < ncomb; h++) {
      real_t v = 0.0;
      if (!mask || mask[h]) {
        if (proc == 0) {
          int hel[4];
          for (int k = 0; k < 4; k++) hel[k] = hel_of(h, k, 4);
          cd a = amp_eemumu(par, pm, hel);
          v = cnorm(a);
          if (jamp2) jamp2[((size_t)e * ncomb + h) * ncol] = to_double(v);
        } else {
          eval_jamps(*P, par, pm, gs[e], h, -1, J, 0, 0);
          v = color_sum(*P, J);
          if (jamp2)
            for (int c = 0; c < ncol; c++) jamp2[((size_t)e * ncomb + h) * ncol + c] = to_double(cnorm(J[c]));
        }
      } else if (jamp2) {
        for (int c = 0; c < ncol; c++) jamp2[((size_t)e * ncomb + h) * ncol + c] = 0.0;
      }
      mhel[(size_t)e * ncomb + h] = to_double(v);
    }
  }
  return 0;
}

// colour-flow amplitudes of one event and one helicity: jamp[ncol] as (re,im) pairs;
// amps (or NULL): [nsub] sub-diagram amplitudes (re,im); ward_leg = -1 or a gluon particle index.
int orc_jamps(int proc, const double* params, const double* mom, double gs, int h, int ward_leg, double* jamp,
              double* amps) {
  Process* P = get_process(proc);
  if (!P || proc == 0) return -1;
  Params par = params_from(params);
  std::vector<cd> J, A;
  eval_jamps(*P, par, mom, gs, h, ward_leg, J, amps ? &A : 0, 0);
  for (int c = 0; c < P->ncol; c++) { jamp[2 * c] = to_double(J[c].real()); jamp[2 * c + 1] = to_double(J[c].imag()); }
  if (amps)
    for (size_t d = 0; d < A.size(); d++) { amps[2 * d] = to_double(A[d].real()); amps[2 * d + 1] = to_double(A[d].imag()); }
  return 0;
}

// Counted mode (BASELINE.json north_star "FLOPs per ME counted by the instrumented oracle"): the
// arithmetic operations the oracle performs for ONE event over the helicities of mask (NULL = all), every distinct
// gluon-tree current and quark-line prefix evaluated once per helicity (eval_jamps memoises them), colour sum as the
// plain double sum.  out4 = {additions+subtractions, multiplications, divisions, square roots}; *me_raw = sum of
// |M_h|^2 (not divided by denom).  Only the -DORC_COUNT build counts; the plain build returns -2.
int orc_count_ops(int proc, const double* params, const double* mom, double gs, const uint8_t* mask, long* out4,
                  double* me_raw) {
#ifdef ORC_COUNT
  Process* P = get_process(proc);
  if (!P) return -1;
  std::vector<double> mhel(P->ncomb, 0.0);
  g_ops = OpCount{0, 0, 0, 0};
  int rc = orc_me_helicities(proc, params, mom, &gs, 1, mask, mhel.data(), 0, 1);
  out4[0] = g_ops.add; out4[1] = g_ops.mul; out4[2] = g_ops.div; out4[3] = g_ops.sqrt;
  double s = 0.0;
  for (int h = 0; h < P->ncomb; h++) s += mhel[h];
  *me_raw = s;
  return rc;
#else
  (void)proc; (void)params; (void)mom; (void)gs; (void)mask; (void)out4; (void)me_raw;
  return -2;
#endif
}

// Multichannel weights ("events from different channels"; reading R17): for every
// event and channel d (= Feynman diagram), num[e][d] = sum over the helicities of mask and over the colour-structure
// terms t of the diagram of |A_{d,t}(h)|^2, with A the Feynman-rule value of the (sub)diagram evaluated by eval_jamps.
// The single-diagram-enhancement weight of channel d is num[e][d] / sum_d' num[e][d'].
int orc_multichannel(int proc, const double* params, const double* mom, const double* gs, int64_t nevt,
                     const uint8_t* mask, double* num, int nthreads) {
  Process* P = get_process(proc);
  if (!P || proc == 0) return -1;
  Params par = params_from(params);
  const int npar = P->npar, ncomb = P->ncomb, nch = (int)P->chan_keys.size();
#ifdef _OPENMP
  const int nt = (nthreads > 0) ? nthreads : omp_get_max_threads();
#else
  const int nt = 1;
#endif
  (void)nt;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
  for (int64_t e = 0; e < nevt; e++) {
    std::vector<cd> J, A;
    double* out = num + (size_t)e * nch;
    for (int d = 0; d < nch; d++) out[d] = 0.0;
    for (int h = 0; h < ncomb; h++) {
      if (mask && !mask[h]) continue;
      eval_jamps(*P, par, mom + (size_t)e * npar * 4, gs[e], h, -1, J, &A, 0);
      for (size_t d = 0; d < A.size(); d++) out[P->chan_of_sub[d]] += to_double(cnorm(A[d]));
    }
  }
  return 0;
}
// number of channels, and (buf != NULL) their keys separated by newlines; returns the bytes needed
int orc_channel_keys(int proc, char* buf, int cap) {
  Process* P = get_process(proc);
  if (!P || proc == 0) return -1;
  std::string all;
  for (auto& k : P->chan_keys) { all += k; all += "\n"; }
  if (buf && cap > (int)all.size()) memcpy(buf, all.c_str(), all.size() + 1);
  return (int)all.size() + 1;
}
// allowed[ndiag][ncol]: 1 iff the diagram contributes to the colour flow (some term has K != 0)
int orc_channel_flows(int proc, uint8_t* allowed) {
  Process* P = get_process(proc);
  if (!P || proc == 0) return -1;
  const int nch = (int)P->chan_keys.size();
  memset(allowed, 0, (size_t)nch * P->ncol);
  for (size_t d = 0; d < P->sub.size(); d++)
    for (auto& kc : P->sub[d].K) allowed[(size_t)P->chan_of_sub[d] * P->ncol + kc.first] = 1;
  return nch;
}

// operation census of ONE helicity: number of three-/four-gluon currents, quark-line chain steps,
// diagram closures and jamp accumulation terms, every distinct current evaluated once.
int orc_census(int proc, long* out5) {
  Process* P = get_process(proc);
  if (!P || proc == 0) return -1;
  Params par = params_from(0);
  std::vector<double> mom(P->npar * 4, 0.0);
  // any valid-looking momenta: census does not depend on values
  for (int i = 0; i < P->npar; i++) { mom[4 * i] = 100.0 + i; mom[4 * i + 1] = 10.0 * (i + 1); mom[4 * i + 2] = 7.0 * i + 1; mom[4 * i + 3] = 20.0 - 3 * i; }
  Census c = {0, 0, 0, 0, 0};
  std::vector<cd> J;
  eval_jamps(*P, par, mom.data(), 1.2, 0, -1, J, 0, &c);
  out5[0] = c.v3; out5[1] = c.v4; out5[2] = c.chain; out5[3] = c.closure; out5[4] = c.jamp_terms;
  return 0;
}

// explicit-colour brute force for one event and helicity: sum over all 8^n * 9 colour assignments of
// | sum_d colourtensor_d(a_1..a_n; i, j) A_d |^2, colour tensors built from Gell-Mann matrices and
// f^{abc} directly (NO trace-basis decomposition, NO colour matrix).  n <= 4.
#ifndef ORC_COUNT
int orc_brute_color(int proc, const double* params, const double* mom, double gs, int h, double* out) {
  Process* P = get_process(proc);
  if (!P || proc == 0 || P->ngl > 4 || P->ew) return -1;
  const SU3& S = su3();
  Params par = params_from(params);
  std::vector<cd> J, A;
  eval_jamps(*P, par, mom, gs, h, -1, J, &A, 0);
  int n = P->ngl;
  long nass = 1;
  for (int k = 0; k < n; k++) nass *= 8;
  double total = 0.0;
#pragma omp parallel for reduction(+ : total) schedule(static)
  for (long ass = 0; ass < nass; ass++) {
    int col_of_leg[8];
    long x = ass;
    for (int k = 0; k < n; k++) { col_of_leg[P->gl[k]] = (int)(x % 8); x /= 8; }
    // colour vector (adjoint index x) of every tree
    std::vector<std::vector<double>> cv(P->trees.size(), std::vector<double>(8, 0.0));
    for (size_t t = 0; t < P->trees.size(); t++) {
      const Tree& T = P->trees[t];
      if (T.kind == 0) cv[t][col_of_leg[T.leg]] = 1.0;
      else if (T.kind == 3) {
        for (int a = 0; a < 8; a++)
          for (int b = 0; b < 8; b++) {
            double w = cv[T.ch[0]][a] * cv[T.ch[1]][b];
            if (w == 0.0) continue;
            for (int xx = 0; xx < 8; xx++) cv[t][xx] += S.f[a][b][xx] * w;
          }
      } else {
        for (int a = 0; a < 8; a++)
          for (int b = 0; b < 8; b++)
            for (int c = 0; c < 8; c++) {
              double w = cv[T.ch[0]][a] * cv[T.ch[1]][b] * cv[T.ch[2]][c];
              if (w == 0.0) continue;
              for (int xx = 0; xx < 8; xx++)
                for (int e = 0; e < 8; e++) {
                  double ff;
                  if (T.term == 0) ff = S.f[a][b][e] * S.f[c][xx][e];
                  else if (T.term == 1) ff = S.f[a][c][e] * S.f[b][xx][e];
                  else ff = S.f[a][xx][e] * S.f[b][c][e];
                  cv[t][xx] += ff * w;
                }
            }
      }
    }
    // quark-line colour matrices along the trie
    std::vector<Mat3> cm(P->trie.size());
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) cm[0].m[i][j] = (i == j) ? 1.0 : 0.0;
    auto tree_matrix = [&](int t) {
      Mat3 m;
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) {
          cdd s(0, 0);
          for (int xx = 0; xx < 8; xx++) s += cv[t][xx] * S.T[xx][i][j];
          m.m[i][j] = s;
        }
      return m;
    };
    for (size_t nd = 1; nd < P->trie.size(); nd++) cm[nd] = m3mul(cm[P->trie[nd].parent], tree_matrix(P->trie[nd].tree));
    Mat3 M;
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) M.m[i][j] = 0.0;
    for (size_t d = 0; d < P->sub.size(); d++) {
      Mat3 c = m3mul(cm[P->sub[d].prefix], tree_matrix(P->sub[d].last));
      for (int i = 0; i < 3; i++)
        for (int j = 0; j < 3; j++) M.m[i][j] += c.m[i][j] * cdd(to_double(A[d].real()), to_double(A[d].imag()));
    }
    double s = 0.0;
    for (int i = 0; i < 3; i++)
      for (int j = 0; j < 3; j++) s += std::norm(M.m[i][j]);
    total += s;
  }
  *out = total;
  return 0;
}
#endif

// external wavefunctions for the algebra tests.  kind: 0 u, 1 v, 2 ubar, 3 vbar, 4 eps (upper index).
int orc_wavefunction(int kind, const double* p, double m, int lam, double* out8) {
  cd r[4];
  if (kind == 4) { V4 e = polvec(p, lam); for (int i = 0; i < 4; i++) r[i] = e.c[i]; }
  else {
    Sp s = (kind == 0 || kind == 2) ? spinor_u(p, m, lam) : spinor_v(p, m, lam);
    if (kind >= 2) s = bar(s);
    for (int i = 0; i < 4; i++) r[i] = s.c[i];
  }
  for (int i = 0; i < 4; i++) { out8[2 * i] = to_double(r[i].real()); out8[2 * i + 1] = to_double(r[i].imag()); }
  return 0;
}
// slash(a) for a complex 4-vector a given as 8 doubles -> 16 complex (32 doubles), row-major
int orc_slash(const double* a8, double* out32) {
  V4 a;
  for (int i = 0; i < 4; i++) a.c[i] = cd(a8[2 * i], a8[2 * i + 1]);
  M4 m = slash(a);
  for (int i = 0; i < 4; i++)
    for (int j = 0; j < 4; j++) { out32[2 * (4 * i + j)] = to_double(m.m[i][j].real()); out32[2 * (4 * i + j) + 1] = to_double(m.m[i][j].imag()); }
  return 0;
}
int orc_num_threads() {
#ifdef _OPENMP
  return omp_get_max_threads();
#else
  return 1;
#endif
}

}  // extern "C"
