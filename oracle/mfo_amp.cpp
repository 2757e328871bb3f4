// mfo_amp.cpp -- ORACLE (test infrastructure, not the product): squared matrix elements.
// PAPER.md:47 (external wavefunctions, vertices, propagators evaluated by ALOHA/HELAS routines),
// PAPER.md:67 (smatrix "loops over initial and final state particle helicities and aggregates"),
// PAPER.md:69 (conditionals in the wavefunctions).  The paper prints no Feynman rule; the set used
// is DESIGN.md reading O6 (HELAS helicity basis, chiral gamma matrices, Peskin-Schroeder rules).
// Everything is done with explicit 4x4 complex matrices and explicit SU(3) generators: slow and
// checkable by eye.  Shares nothing with the CUDA path.
#include "mfo.h"
#include <complex>
#include <cmath>
#include <cstring>
#include <map>
#include <vector>
#include <array>
#include <algorithm>
#include <mutex>
#include <functional>

typedef std::complex<double> cd;
static const cd I_(0.0, 1.0);
struct V4 { cd c[4]; };   // complex 4-vector, upper index (E,x,y,z)
struct Sp { cd c[4]; };   // Dirac spinor (column) or adjoint spinor (row)
struct M4 { cd m[4][4]; };

// ---- O6.1 Dirac algebra, chiral representation, metric (+,-,-,-) ------------------------------
static M4 GAM[4];
static std::once_flag gamma_once;
static void init_gamma_impl();
static void init_gamma() { std::call_once(gamma_once, init_gamma_impl); }
static void init_gamma_impl() {
  cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};   // Pauli
  for (int mu = 0; mu < 4; ++mu) for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) GAM[mu].m[r][c] = 0;
  for (int a = 0; a < 2; ++a) { GAM[0].m[a][2 + a] = 1; GAM[0].m[2 + a][a] = 1; }   // [[0,1],[1,0]]
  for (int i = 0; i < 3; ++i) for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) {
    GAM[1 + i].m[a][2 + b] = s[i][a][b];        // [[0, sigma],[-sigma, 0]]
    GAM[1 + i].m[2 + a][b] = -s[i][a][b];
  }
}
extern "C" void mfo_gamma(double out[128]) {
  init_gamma();
  for (int mu = 0; mu < 4; ++mu) for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) {
    out[((mu * 4 + r) * 4 + c) * 2] = GAM[mu].m[r][c].real();
    out[((mu * 4 + r) * 4 + c) * 2 + 1] = GAM[mu].m[r][c].imag();
  }
}
static inline cd mdot(const V4 &a, const V4 &b) { return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3]; }
static inline V4 vadd(const V4 &a, const V4 &b) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] + b.c[i]; return r; }
static inline V4 vsub(const V4 &a, const V4 &b) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] - b.c[i]; return r; }
static inline V4 vscale(cd s, const V4 &a) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = s * a.c[i]; return r; }
static inline V4 vreal(const double *p) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = p[i]; return r; }
// slash(v) = gamma^mu v_mu = gamma^0 v^0 - gamma^i v^i
static M4 slash(const V4 &v) {
  M4 r;
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b)
    r.m[a][b] = GAM[0].m[a][b] * v.c[0] - GAM[1].m[a][b] * v.c[1] - GAM[2].m[a][b] * v.c[2] - GAM[3].m[a][b] * v.c[3];
  return r;
}
static Sp matvec(const M4 &A, const Sp &x) { Sp r; for (int a = 0; a < 4; ++a) { r.c[a] = 0; for (int b = 0; b < 4; ++b) r.c[a] += A.m[a][b] * x.c[b]; } return r; }
static Sp adjoint(const Sp &u) {   // ubar = u^dagger gamma^0
  Sp r; for (int b = 0; b < 4; ++b) { r.c[b] = 0; for (int a = 0; a < 4; ++a) r.c[b] += std::conj(u.c[a]) * GAM[0].m[a][b]; } return r;
}
static cd rowcol(const Sp &row, const Sp &col) { cd s = 0; for (int a = 0; a < 4; ++a) s += row.c[a] * col.c[a]; return s; }

// ---- O6.2 external wavefunctions (HELAS helicity basis) ------------------------------------------
static void chi(const double p[4], cd chip[2], cd chim[2]) {
  double pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  double pt2 = p[1] * p[1] + p[2] * p[2];
  if (pabs < 1e-12 * std::fabs(p[0]) || (pt2 == 0.0 && p[3] < 0)) {   // p_z = -|p| branch (O6.2)
    chip[0] = 0; chip[1] = 1; chim[0] = -1; chim[1] = 0; return;
  }
  double ppz = (p[3] >= 0) ? pabs + p[3] : pt2 / (pabs - p[3]);   // |p|+pz without cancellation
  double N = 1.0 / std::sqrt(2.0 * pabs * ppz);
  chip[0] = N * ppz; chip[1] = N * cd(p[1], p[2]);
  chim[0] = N * cd(-p[1], p[2]); chim[1] = N * ppz;
}
// kind 0: u(p,lambda); kind 1: v(p,lambda)
static Sp wf_fermion(int kind, const double p[4], double m, int lam) {
  double pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  double wp = std::sqrt(p[0] + pabs);
  double wm = (m == 0.0) ? 0.0 : m / wp;       // sqrt(E-|p|) = m / sqrt(E+|p|)
  cd cp[2], cm[2]; chi(p, cp, cm);
  auto om = [&](int s) { return s > 0 ? wp : wm; };
  Sp r;
  if (kind == 0) {           // u = (omega_{-lam} chi_lam ; omega_lam chi_lam)
    const cd *c = lam > 0 ? cp : cm;
    r.c[0] = om(-lam) * c[0]; r.c[1] = om(-lam) * c[1]; r.c[2] = om(lam) * c[0]; r.c[3] = om(lam) * c[1];
  } else {                   // v = (-lam omega_lam chi_{-lam} ; lam omega_{-lam} chi_{-lam})
    const cd *c = lam > 0 ? cm : cp;
    double l = (double)lam;
    r.c[0] = -l * om(lam) * c[0]; r.c[1] = -l * om(lam) * c[1]; r.c[2] = l * om(-lam) * c[0]; r.c[3] = l * om(-lam) * c[1];
  }
  return r;
}
// eps(p,lam) = (-lam eps1 - i eps2)/sqrt2
static V4 wf_vector(const double p[4], int lam) {
  double pt = std::sqrt(p[1] * p[1] + p[2] * p[2]);
  double pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  double e1[4], e2[4];
  if (pt == 0.0) { e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0; e2[0] = 0; e2[1] = 0; e2[2] = (p[3] >= 0 ? 1.0 : -1.0); e2[3] = 0; }
  else {
    e1[0] = 0; e1[1] = p[1] * p[3] / (pabs * pt); e1[2] = p[2] * p[3] / (pabs * pt); e1[3] = -pt / pabs;
    e2[0] = 0; e2[1] = -p[2] / pt; e2[2] = p[1] / pt; e2[3] = 0;
  }
  V4 r; double l = (double)lam;
  for (int i = 0; i < 4; ++i) r.c[i] = (-l * e1[i] - I_ * e2[i]) / std::sqrt(2.0);
  return r;
}
extern "C" void mfo_wf_fermion(int kind, const double p[4], double m, int lambda, double out[8]) {
  init_gamma(); Sp s = wf_fermion(kind, p, m, lambda);
  for (int i = 0; i < 4; ++i) { out[2 * i] = s.c[i].real(); out[2 * i + 1] = s.c[i].imag(); }
}
extern "C" void mfo_wf_vector(const double p[4], int lambda, double out[8]) {
  V4 v = wf_vector(p, lambda);
  for (int i = 0; i < 4; ++i) { out[2 * i] = v.c[i].real(); out[2 * i + 1] = v.c[i].imag(); }
}

// ---- SU(3): Gell-Mann matrices, T^a = lambda^a/2, f^{abc} = -2i Tr([T^a,T^b]T^c) (O6.3) ----------
struct C3 { cd m[3][3]; };
static C3 TA[8]; static double FABC[8][8][8];
static C3 c3mul(const C3 &a, const C3 &b) { C3 r; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { r.m[i][j] = 0; for (int k = 0; k < 3; ++k) r.m[i][j] += a.m[i][k] * b.m[k][j]; } return r; }
static cd c3trace(const C3 &a) { return a.m[0][0] + a.m[1][1] + a.m[2][2]; }
static std::once_flag su3_once;
static void init_su3() {
  std::call_once(su3_once, [] {
    for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) TA[a].m[i][j] = 0;
    TA[0].m[0][1] = 0.5; TA[0].m[1][0] = 0.5;
    TA[1].m[0][1] = -0.5 * I_; TA[1].m[1][0] = 0.5 * I_;
    TA[2].m[0][0] = 0.5; TA[2].m[1][1] = -0.5;
    TA[3].m[0][2] = 0.5; TA[3].m[2][0] = 0.5;
    TA[4].m[0][2] = -0.5 * I_; TA[4].m[2][0] = 0.5 * I_;
    TA[5].m[1][2] = 0.5; TA[5].m[2][1] = 0.5;
    TA[6].m[1][2] = -0.5 * I_; TA[6].m[2][1] = 0.5 * I_;
    double s3 = 1.0 / std::sqrt(3.0);
    TA[7].m[0][0] = 0.5 * s3; TA[7].m[1][1] = 0.5 * s3; TA[7].m[2][2] = -s3;
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
      C3 ab = c3mul(TA[a], TA[b]), ba = c3mul(TA[b], TA[a]), comm;
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) comm.m[i][j] = ab.m[i][j] - ba.m[i][j];
      cd v = -2.0 * I_ * c3trace(c3mul(comm, TA[c]));
      FABC[a][b][c] = std::fabs(v.real()) < 1e-14 ? 0.0 : v.real();
    }
    init_gamma();
  });
}
extern "C" void mfo_su3(double *T, double *f) {
  init_su3();
  for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) {
    T[((a * 3 + i) * 3 + j) * 2] = TA[a].m[i][j].real(); T[((a * 3 + i) * 3 + j) * 2 + 1] = TA[a].m[i][j].imag();
  }
  for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) f[(a * 8 + b) * 8 + c] = FABC[a][b][c];
}

// V3^{mu nu rho}(k,p,q) A_nu B_rho = A^mu ((k-p).B) + (p-q)^mu (A.B) + B^mu ((q-k).A)   (O6.3)
static V4 v3contract(const V4 &k, const V4 &p, const V4 &q, const V4 &A, const V4 &B) {
  cd c1 = mdot(vsub(k, p), B), c2 = mdot(A, B), c3 = mdot(vsub(q, k), A);
  V4 pq = vsub(p, q), r;
  for (int i = 0; i < 4; ++i) r.c[i] = A.c[i] * c1 + pq.c[i] * c2 + B.c[i] * c3;
  return r;
}

// ---- process description ---------------------------------------------------------------------------
// gg -> t tbar + (ng-2) g.  Gluon legs g = 0..ng-1: legs 0,1 incoming (momenta mom[0], mom[1]),
// legs 2.. outgoing (mom[4], mom[5]); top = mom[2] (ubar), antitop = mom[3] (v).  All-incoming
// gluon momenta K_g = +k (initial), -k (final); polarisation eps (initial), eps^* (final).
struct Ext {
  int ng; double mt, gs;
  V4 K[4], e[4];          // all-incoming momenta and polarisations of the gluon legs
  V4 p3, p4; Sp ubar3, v4;
};
static int process_ng(int process) { return process == MFO_GG_TT ? 2 : process == MFO_GG_TTG ? 3 : process == MFO_GG_TTGG ? 4 : -1; }
static void fill_ext(Ext &X, int ng, const double *mom, double mt, double alpha_s, const int *hel, int ward_leg) {
  X.ng = ng; X.mt = mt; X.gs = std::sqrt(4.0 * M_PI * alpha_s);
  for (int g = 0; g < ng; ++g) {
    const double *k = (g < 2) ? mom + 4 * g : mom + 4 * (2 + g);
    int lam = (g < 2) ? hel[g] : hel[2 + g];
    V4 eps = wf_vector(k, lam);
    if (g < 2) { X.K[g] = vreal(k); X.e[g] = eps; }
    else { X.K[g] = vscale(-1.0, vreal(k)); for (int i = 0; i < 4; ++i) X.e[g].c[i] = std::conj(eps.c[i]); }
    if (g == ward_leg) X.e[g] = X.K[g];
  }
  X.p3 = vreal(mom + 8); X.p4 = vreal(mom + 12);
  X.ubar3 = adjoint(wf_fermion(0, mom + 8, mt, hel[2]));
  X.v4 = wf_fermion(1, mom + 12, mt, hel[3]);
}
static V4 subset_momentum(const Ext &X, unsigned S) { V4 P; for (int i = 0; i < 4; ++i) P.c[i] = 0; for (int g = 0; g < X.ng; ++g) if (S >> g & 1) P = vadd(P, X.K[g]); return P; }
// quark propagator i (qslash + m)/(q^2 - m^2) applied to a spinor
static Sp quark_prop(const V4 &q, double m, const Sp &x) {
  M4 qs = slash(q); Sp r = matvec(qs, x); cd den = mdot(q, q) - m * m;
  for (int a = 0; a < 4; ++a) r.c[a] = I_ * (r.c[a] + m * x.c[a]) / den;
  return r;
}

// ================================================================================================
// Algorithm B -- the literal colour-dressed recursion (O6.5): the definition.
// ================================================================================================
struct GC { V4 a[8]; };                 // gluon current with adjoint colour index
struct QC { Sp i[3]; };                 // quark current with fundamental colour index
static cd amp_literal(const Ext &X, const int *col_g, int c3, int c4) {
  const int ng = X.ng; const unsigned full = (1u << ng) - 1;
  std::vector<GC> J(full + 1); std::vector<V4> P(full + 1);
  for (unsigned S = 1; S <= full; ++S) P[S] = subset_momentum(X, S);
  for (unsigned S = 1; S <= full; ++S) {
    GC &j = J[S];
    for (int a = 0; a < 8; ++a) for (int i = 0; i < 4; ++i) j.a[a].c[i] = 0;
    if (__builtin_popcount(S) == 1) { int g = __builtin_ctz(S); j.a[col_g[g]] = X.e[g]; continue; }
  }
  // subsets in order of size so that parts are ready
  std::vector<unsigned> order; for (int sz = 2; sz <= ng; ++sz) for (unsigned S = 1; S <= full; ++S) if (__builtin_popcount(S) == sz) order.push_back(S);
  for (unsigned S : order) {
    GC acc; for (int a = 0; a < 8; ++a) for (int i = 0; i < 4; ++i) acc.a[a].c[i] = 0;
    unsigned low = S & (~S + 1);
    V4 mP = vscale(-1.0, P[S]);
    // cubic: unordered {A,B}, A contains the lowest leg
    for (unsigned A = S; A; A = (A - 1) & S) {
      unsigned B = S & ~A; if (!(A & low) || !B) continue;
      for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {
        if (FABC[a][b][c] == 0.0) continue;
        V4 t = v3contract(mP, P[A], P[B], J[A].a[b], J[B].a[c]);
        acc.a[a] = vadd(acc.a[a], vscale(X.gs * FABC[a][b][c], t));
      }
    }
    // quartic: unordered {A,B,C}
    for (unsigned A = S; A; A = (A - 1) & S) {
      if (!(A & low)) continue; unsigned R = S & ~A; if (!R) continue; unsigned lowR = R & (~R + 1);
      for (unsigned B = R; B; B = (B - 1) & R) {
        unsigned C = R & ~B; if (!(B & lowR) || !C) continue;
        for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) for (int d = 0; d < 8; ++d) {
          const V4 &JA = J[A].a[b], &JB = J[B].a[c], &JC = J[C].a[d];
          cd ab = mdot(JA, JB), ac = mdot(JA, JC), bc = mdot(JB, JC);
          if (ab == 0.0 && ac == 0.0 && bc == 0.0) continue;
          for (int a = 0; a < 8; ++a) {
            double f1 = 0, f2 = 0, f3 = 0;
            for (int e = 0; e < 8; ++e) { f1 += FABC[a][b][e] * FABC[c][d][e]; f2 += FABC[a][c][e] * FABC[b][d][e]; f3 += FABC[a][d][e] * FABC[b][c][e]; }
            if (f1 == 0 && f2 == 0 && f3 == 0) continue;
            cd pref = -I_ * X.gs * X.gs;
            for (int i = 0; i < 4; ++i)
              acc.a[a].c[i] += pref * (f1 * (JB.c[i] * ac - JC.c[i] * ab) + f2 * (JA.c[i] * bc - JC.c[i] * ab) + f3 * (JA.c[i] * bc - JB.c[i] * ac));
          }
        }
      }
    }
    cd prop = -I_ / mdot(P[S], P[S]);
    for (int a = 0; a < 8; ++a) J[S].a[a] = vscale(prop, acc.a[a]);
  }
  // quark line: psi(empty) = delta_{i c4} v; psi(S) = S_F(q_S) sum_A (i gs) T^a Jslash^a(A) psi(S\A)
  std::vector<QC> psi(full + 1);
  auto attach = [&](unsigned S) {          // sum over nonempty A subset of S, no propagator
    QC r; for (int i = 0; i < 3; ++i) for (int al = 0; al < 4; ++al) r.i[i].c[al] = 0;
    for (unsigned A = S; A; A = (A - 1) & S) {
      const QC &rest = psi[S & ~A];
      for (int a = 0; a < 8; ++a) {
        M4 js = slash(J[A].a[a]);
        for (int j = 0; j < 3; ++j) {
          Sp t = matvec(js, rest.i[j]);
          for (int i = 0; i < 3; ++i) { cd w = I_ * X.gs * TA[a].m[i][j]; if (w == 0.0) continue; for (int al = 0; al < 4; ++al) r.i[i].c[al] += w * t.c[al]; }
        }
      }
    }
    return r;
  };
  for (int i = 0; i < 3; ++i) for (int al = 0; al < 4; ++al) psi[0].i[i].c[al] = (i == c4) ? X.v4.c[al] : cd(0);
  std::vector<unsigned> qorder; for (int sz = 1; sz < ng; ++sz) for (unsigned S = 1; S <= full; ++S) if (__builtin_popcount(S) == sz) qorder.push_back(S);
  for (unsigned S : qorder) {
    QC r = attach(S); V4 q = vsub(P[S], X.p4);
    for (int i = 0; i < 3; ++i) psi[S].i[i] = quark_prop(q, X.mt, r.i[i]);
  }
  QC last = attach(full);
  return rowcol(X.ubar3, last.i[c3]);       // = iM
}

// ================================================================================================
// Algorithm A -- diagram list with colour flows (O6.5), built at run time by enumeration.
// ================================================================================================
typedef std::map<std::vector<int>, cd> Word;   // colour word: sum of coeff * T^{a_l1} T^{a_l2} ...
static Word wmul(const Word &a, const Word &b) { Word r; for (auto &x : a) for (auto &y : b) { std::vector<int> w = x.first; w.insert(w.end(), y.first.begin(), y.first.end()); r[w] += x.second * y.second; } return r; }
static Word wlin(cd ca, const Word &a, cd cb, const Word &b) { Word r; for (auto &x : a) r[x.first] += ca * x.second; for (auto &y : b) r[y.first] += cb * y.second; return r; }
static Word wcomm(const Word &a, const Word &b) { return wlin(1.0, wmul(a, b), -1.0, wmul(b, a)); }
static Word wscale(cd c, const Word &a) { Word r; for (auto &x : a) r[x.first] = c * x.second; return r; }

struct Tree { int kind; unsigned mask; int ch[3]; int which; Word T; int topo; };  // kind 0 leaf,1 cubic,2 quartic
struct Diagram { std::vector<int> clusters; std::vector<std::pair<int, cd>> flows; };  // tree ids along the quark line
struct Table {
  int ng = 0; std::vector<Tree> trees; std::vector<std::vector<int>> by_mask;   // tree ids per subset
  std::vector<Diagram> diags; std::vector<std::vector<int>> perms; uint32_t ndiag = 0, nsub = 0;
  std::vector<double> C; double cden = 1;     // colour matrix (real) [nf][nf]
};
static Table TAB[5]; static std::once_flag tab_once[5];

static void build_colour_matrix(Table &t) {
  // C_{s s'} = sum_a Tr(T^{a_s(1)}...T^{a_s(n)} (T^{a_s'(1)}...T^{a_s'(n)})^dagger), brute force
  int ng = t.ng, nf = (int)t.perms.size(); t.C.assign((size_t)nf * nf, 0.0);
  int ncol = 1; for (int i = 0; i < ng; ++i) ncol *= 8;
  std::vector<cd> acc((size_t)nf * nf, 0.0);
  for (int code = 0; code < ncol; ++code) {
    int a[4], c = code; for (int g = 0; g < ng; ++g) { a[g] = c % 8; c /= 8; }
    std::vector<C3> W(nf);
    for (int s = 0; s < nf; ++s) { C3 m = TA[a[t.perms[s][0]]]; for (int k = 1; k < ng; ++k) m = c3mul(m, TA[a[t.perms[s][k]]]); W[s] = m; }
    for (int s = 0; s < nf; ++s) for (int s2 = 0; s2 < nf; ++s2) {
      cd tr = 0; for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) tr += W[s].m[i][j] * std::conj(W[s2].m[i][j]);
      acc[(size_t)s * nf + s2] += tr;
    }
  }
  for (size_t i = 0; i < acc.size(); ++i) t.C[i] = acc[i].real();
  t.cden = (ng == 2) ? 3.0 : (ng == 3) ? 9.0 : 54.0;
}

static void build_table(int ng) {
  init_su3();
  Table &t = TAB[ng]; t.ng = ng; const unsigned full = (1u << ng) - 1;
  t.by_mask.assign(full + 1, {});
  for (int sz = 1; sz <= ng; ++sz) for (unsigned S = 1; S <= full; ++S) {
    if (__builtin_popcount(S) != sz) continue;
    if (sz == 1) { Tree tr{0, S, {-1, -1, -1}, 0, {}, 0}; int g = __builtin_ctz(S); tr.T[{g}] = 1.0; t.by_mask[S].push_back((int)t.trees.size()); t.trees.push_back(tr); continue; }
    unsigned low = S & (~S + 1);
    // topology id of a node = index of (kind, child subsets, child topology ids): the three colour
    // structures of one four-gluon vertex share it, so that "diagrams" count the vertex once
    std::map<std::array<int, 7>, int> topo_ids;
    auto topo_of = [&](int kind, int ta, int tb, int tc) {
      std::array<int, 7> key = {kind, (int)t.trees[ta].mask, t.trees[ta].topo, (int)t.trees[tb].mask, t.trees[tb].topo,
                                tc >= 0 ? (int)t.trees[tc].mask : 0, tc >= 0 ? t.trees[tc].topo : 0};
      auto it = topo_ids.find(key); if (it != topo_ids.end()) return it->second;
      int id = (int)topo_ids.size(); topo_ids[key] = id; return id;
    };
    for (unsigned A = S; A; A = (A - 1) & S) {       // cubic nodes, T = -i [T_A, T_B]
      unsigned B = S & ~A; if (!(A & low) || !B) continue;
      for (int ta : t.by_mask[A]) for (int tb : t.by_mask[B]) {
        Tree tr{1, S, {ta, tb, -1}, 0, wscale(-I_, wcomm(t.trees[ta].T, t.trees[tb].T)), topo_of(1, ta, tb, -1)};
        t.by_mask[S].push_back((int)t.trees.size()); t.trees.push_back(tr);
      }
    }
    for (unsigned A = S; A; A = (A - 1) & S) {       // quartic nodes, three colour structures each
      if (!(A & low)) continue; unsigned R = S & ~A; if (!R) continue; unsigned lowR = R & (~R + 1);
      for (unsigned B = R; B; B = (B - 1) & R) {
        unsigned Cc = R & ~B; if (!(B & lowR) || !Cc) continue;
        for (int ta : t.by_mask[A]) for (int tb : t.by_mask[B]) for (int tc : t.by_mask[Cc]) {
          const Word &WA = t.trees[ta].T, &WB = t.trees[tb].T, &WC = t.trees[tc].T;
          Word w[3] = {wscale(-1.0, wcomm(WA, wcomm(WB, WC))), wscale(-1.0, wcomm(WB, wcomm(WA, WC))), wscale(-1.0, wcomm(WC, wcomm(WA, WB)))};
          int tp = topo_of(2, ta, tb, tc);
          for (int k = 0; k < 3; ++k) { Tree tr{2, S, {ta, tb, tc}, k, w[k], tp}; t.by_mask[S].push_back((int)t.trees.size()); t.trees.push_back(tr); }
        }
      }
    }
  }
  // permutations of the gluon legs in lexicographic order = colour flows
  std::vector<int> p(ng); for (int i = 0; i < ng; ++i) p[i] = i;
  do t.perms.push_back(p); while (std::next_permutation(p.begin(), p.end()));
  std::map<std::vector<int>, int> perm_index; for (size_t s = 0; s < t.perms.size(); ++s) perm_index[t.perms[s]] = (int)s;
  // diagrams: ordered set partitions (C1..Cm) of the legs x one tree per cluster
  std::vector<std::vector<unsigned>> parts;
  std::vector<unsigned> cur;
  std::function<void(unsigned)> rec = [&](unsigned rest) {
    if (!rest) { parts.push_back(cur); return; }
    for (unsigned A = rest; A; A = (A - 1) & rest) { cur.push_back(A); rec(rest & ~A); cur.pop_back(); }
  };
  rec(full);
  // a "diagram" counts a quartic node once: sub-terms with identical topology ids in every cluster
  std::map<std::vector<std::pair<unsigned, int>>, int> topo_seen;
  for (auto &pt : parts) {
    std::vector<int> idx(pt.size(), 0);
    while (true) {
      Diagram d; Word w; w[{}] = 1.0; std::vector<std::pair<unsigned, int>> sig;
      for (size_t c = 0; c < pt.size(); ++c) {
        int id = t.by_mask[pt[c]][idx[c]]; d.clusters.push_back(id); w = wmul(w, t.trees[id].T);
        sig.push_back({pt[c], t.trees[id].topo});
      }
      for (auto &x : w) if (std::abs(x.second) > 1e-14) d.flows.push_back({perm_index.at(x.first), x.second});
      t.diags.push_back(d); topo_seen[sig]++;
      size_t c = 0; for (; c < pt.size(); ++c) { if (++idx[c] < (int)t.by_mask[pt[c]].size()) break; idx[c] = 0; }
      if (c == pt.size()) break;
    }
  }
  t.nsub = (uint32_t)t.diags.size(); t.ndiag = (uint32_t)topo_seen.size();
  build_colour_matrix(t);
}

static const Table &table(int ng) { std::call_once(tab_once[ng], build_table, ng); return TAB[ng]; }

// current of every tree node for one helicity assignment (children precede parents in the table)
static void eval_trees(const Table &t, const Ext &X, std::vector<V4> &J, std::vector<V4> &P) {
  const unsigned full = (1u << t.ng) - 1;
  P.resize(full + 1); for (unsigned S = 1; S <= full; ++S) P[S] = subset_momentum(X, S);
  J.resize(t.trees.size());
  for (size_t id = 0; id < t.trees.size(); ++id) {
    const Tree &tr = t.trees[id];
    if (tr.kind == 0) { J[id] = X.e[__builtin_ctz(tr.mask)]; continue; }
    const V4 &PS = P[tr.mask]; cd prop = -I_ / mdot(PS, PS);
    if (tr.kind == 1) {     // (-i/P^2) gs V3(-P, P_A, P_B) J_A J_B
      const Tree &a = t.trees[tr.ch[0]], &b = t.trees[tr.ch[1]];
      V4 v = v3contract(vscale(-1.0, PS), P[a.mask], P[b.mask], J[tr.ch[0]], J[tr.ch[1]]);
      J[id] = vscale(prop * X.gs, v);
    } else {                // (-i/P^2)(-i gs^2) x one of the three Lorentz structures
      const V4 &A = J[tr.ch[0]], &B = J[tr.ch[1]], &C = J[tr.ch[2]];
      cd ab = mdot(A, B), ac = mdot(A, C), bc = mdot(B, C); V4 v;
      for (int i = 0; i < 4; ++i)
        v.c[i] = tr.which == 0 ? B.c[i] * ac - C.c[i] * ab : tr.which == 1 ? A.c[i] * bc - C.c[i] * ab : A.c[i] * bc - B.c[i] * ac;
      J[id] = vscale(prop * (-I_ * X.gs * X.gs), v);
    }
  }
}

// jamp_sigma = sum_D coeff_{sigma,D} A_D,  A_D = ubar (i gs Jslash(C1)) S(q2) (i gs Jslash(C2)) ... v
static void eval_jamps(const Table &t, const Ext &X, std::vector<cd> &jamp) {
  std::vector<V4> J, P; eval_trees(t, X, J, P);
  jamp.assign(t.perms.size(), cd(0));
  for (const Diagram &d : t.diags) {
    Sp psi = X.v4; int m = (int)d.clusters.size();
    V4 q = vscale(-1.0, X.p4);
    for (int j = m - 1; j >= 0; --j) {
      const Tree &tr = t.trees[d.clusters[j]];
      Sp t1 = matvec(slash(J[d.clusters[j]]), psi);
      for (int a = 0; a < 4; ++a) t1.c[a] *= I_ * X.gs;
      q = vadd(q, P[tr.mask]);                 // q_j = sum_{l>=j} P_{C_l} - p4
      psi = (j > 0) ? quark_prop(q, X.mt, t1) : t1;
    }
    cd A = rowcol(X.ubar3, psi);
    for (auto &f : d.flows) jamp[f.first] += f.second * A;
  }
}
static double colour_form(const Table &t, const std::vector<cd> &jamp) {
  size_t nf = t.perms.size(); long double s = 0;
  for (size_t a = 0; a < nf; ++a) for (size_t b = 0; b < nf; ++b)
    s += (long double)t.C[a * nf + b] * (jamp[a].real() * jamp[b].real() + jamp[a].imag() * jamp[b].imag());
  return (double)s;
}

// O6.4  e+ e- -> mu+ mu-: M = e^2 [vbar(pb) gamma^mu u(pa)] [ubar(p1) gamma_mu v(p2)] / s
static double me2_eemumu(const double *mom, double alpha_em) {
  init_su3();
  double e2 = 4.0 * M_PI * alpha_em;
  double s = (mom[0] + mom[4]) * (mom[0] + mom[4]) - (mom[1] + mom[5]) * (mom[1] + mom[5]) -
             (mom[2] + mom[6]) * (mom[2] + mom[6]) - (mom[3] + mom[7]) * (mom[3] + mom[7]);
  long double tot = 0;
  for (int h = 0; h < 16; ++h) {
    int la = (h & 1) ? 1 : -1, lb = (h & 2) ? 1 : -1, l1 = (h & 4) ? 1 : -1, l2 = (h & 8) ? 1 : -1;
    Sp ua = wf_fermion(0, mom, 0.0, la);                   // incoming e-
    Sp vbb = adjoint(wf_fermion(1, mom + 4, 0.0, lb));     // incoming e+
    Sp ub1 = adjoint(wf_fermion(0, mom + 8, 0.0, l1));     // outgoing mu-
    Sp v2 = wf_fermion(1, mom + 12, 0.0, l2);              // outgoing mu+
    V4 L, R;
    for (int mu = 0; mu < 4; ++mu) { L.c[mu] = rowcol(vbb, matvec(GAM[mu], ua)); R.c[mu] = rowcol(ub1, matvec(GAM[mu], v2)); }
    cd M = e2 * mdot(L, R) / s;
    tot += std::norm(M);
  }
  return (double)(tot / 4.0L);
}

// O6q  q q~ -> t t~: M = g_s^2 T^a_{ji} T^a_{kl} [vbar(pb) gamma^mu u(pa)] [ubar(k1) gamma_mu v(k2)] / shat;
// sum over the helicities and over the colours i, j (incoming) and k, l (outgoing) of |M|^2, averaged over the
// 4 helicities and 9 colours of the incoming pair.  The colour sum is taken literally from the Gell-Mann matrices.
static double me2_qqtt(const double *mom, double m_top, double alpha_s) {
  init_su3();
  double g2 = 4.0 * M_PI * alpha_s;
  double s = (mom[0] + mom[4]) * (mom[0] + mom[4]) - (mom[1] + mom[5]) * (mom[1] + mom[5]) -
             (mom[2] + mom[6]) * (mom[2] + mom[6]) - (mom[3] + mom[7]) * (mom[3] + mom[7]);
  long double col = 0;                                     // sum_{ijkl} |sum_a T^a_{ji} T^a_{kl}|^2
  for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int k = 0; k < 3; ++k) for (int l = 0; l < 3; ++l) {
    cd c = 0;
    for (int a = 0; a < 8; ++a) c += TA[a].m[j][i] * TA[a].m[k][l];
    col += std::norm(c);
  }
  long double tot = 0;
  for (int h = 0; h < 16; ++h) {
    int la = (h & 1) ? 1 : -1, lb = (h & 2) ? 1 : -1, l1 = (h & 4) ? 1 : -1, l2 = (h & 8) ? 1 : -1;
    Sp ua = wf_fermion(0, mom, 0.0, la);                   // incoming q
    Sp vbb = adjoint(wf_fermion(1, mom + 4, 0.0, lb));     // incoming q~
    Sp ub1 = adjoint(wf_fermion(0, mom + 8, m_top, l1));   // outgoing t
    Sp v2 = wf_fermion(1, mom + 12, m_top, l2);            // outgoing t~
    V4 L, R;
    for (int mu = 0; mu < 4; ++mu) { L.c[mu] = rowcol(vbb, matvec(GAM[mu], ua)); R.c[mu] = rowcol(ub1, matvec(GAM[mu], v2)); }
    cd M = g2 * mdot(L, R) / s;
    tot += std::norm(M);
  }
  return (double)(tot * col / 36.0L);
}

static void hel_from_index(int h, int nleg, int *hel) { for (int l = 0; l < nleg; ++l) hel[l] = (h >> l & 1) ? 1 : -1; }

extern "C" int mfo_me2(int process, const double *mom, double m_top, double alpha_s, double alpha_em, double *out) {
  if (process == MFO_EE_MUMU) { *out = me2_eemumu(mom, alpha_em); return MFO_OK; }
  if (process == MFO_QQ_TT) { *out = me2_qqtt(mom, m_top, alpha_s); return MFO_OK; }
  if (process == MFO_QQ_TTG || process == MFO_QG_TTQ) return mfo_me2_2q(process, mom, m_top, alpha_s, 0, out);
  int ng = process_ng(process); if (ng < 0) return MFO_EINVAL;
  const Table &t = table(ng); int nleg = ng + 2; long double tot = 0;
  std::vector<cd> jamp;
  for (int h = 0; h < (1 << nleg); ++h) {
    int hel[6]; hel_from_index(h, nleg, hel);
    Ext X; fill_ext(X, ng, mom, m_top, alpha_s, hel, -1);
    eval_jamps(t, X, jamp);
    tot += colour_form(t, jamp);
  }
  *out = (double)(tot / 256.0L);     // 1/4 helicities x 1/64 colours of the incoming gluons (A12)
  return MFO_OK;
}

extern "C" int mfo_jamps(int process, const double *mom, double m_top, double alpha_s, const int *hel,
                         int ward_leg, double *jamp_out, double *me2_hel) {
  int ng = process_ng(process); if (ng < 0) return MFO_EINVAL;
  const Table &t = table(ng);
  Ext X; fill_ext(X, ng, mom, m_top, alpha_s, hel, ward_leg);
  std::vector<cd> jamp; eval_jamps(t, X, jamp);
  if (jamp_out) for (size_t s = 0; s < jamp.size(); ++s) { jamp_out[2 * s] = jamp[s].real(); jamp_out[2 * s + 1] = jamp[s].imag(); }
  if (me2_hel) *me2_hel = colour_form(t, jamp);
  return MFO_OK;
}

extern "C" int mfo_amp_literal(int process, const double *mom, double m_top, double alpha_s, const int *hel,
                               const int *col_g, int c3, int c4, int ward_leg, double out[2]) {
  int ng = process_ng(process); if (ng < 0) return MFO_EINVAL;
  init_su3();
  Ext X; fill_ext(X, ng, mom, m_top, alpha_s, hel, ward_leg);
  cd A = amp_literal(X, col_g, c3, c4); out[0] = A.real(); out[1] = A.imag();
  return MFO_OK;
}

extern "C" int mfo_me2_literal(int process, const double *mom, double m_top, double alpha_s, int hel_only, double *out) {
  int ng = process_ng(process); if (ng < 0) return MFO_EINVAL;
  init_su3();
  int nleg = ng + 2, ncol = 1; for (int g = 0; g < ng; ++g) ncol *= 8;
  long double tot = 0;
  for (int h = 0; h < (1 << nleg); ++h) {
    if (hel_only >= 0 && h != hel_only) continue;
    int hel[6]; hel_from_index(h, nleg, hel);
    Ext X; fill_ext(X, ng, mom, m_top, alpha_s, hel, -1);
    for (int code = 0; code < ncol; ++code) {
      int col[4], c = code; for (int g = 0; g < ng; ++g) { col[g] = c % 8; c /= 8; }
      for (int c3 = 0; c3 < 3; ++c3) for (int c4 = 0; c4 < 3; ++c4) tot += std::norm(amp_literal(X, col, c3, c4));
    }
  }
  *out = (double)(hel_only >= 0 ? tot : tot / 256.0L);
  return MFO_OK;
}

extern "C" int mfo_colour_matrix(uint32_t ng, double *numer, double *denom) {
  if (ng < 2 || ng > 4) return MFO_EINVAL;
  const Table &t = table((int)ng); size_t nf = t.perms.size();
  for (size_t i = 0; i < nf * nf; ++i) numer[i] = t.C[i] * t.cden;
  *denom = t.cden; return MFO_OK;
}
extern "C" int mfo_diagram_counts(uint32_t ng, uint32_t *ndiag, uint32_t *nsub, uint32_t *nflow) {
  if (ng < 2 || ng > 4) return MFO_EINVAL;
  const Table &t = table((int)ng); *ndiag = t.ndiag; *nsub = t.nsub; *nflow = (uint32_t)t.perms.size(); return MFO_OK;
}
