// mfo_amp2q.cpp -- ORACLE (test infrastructure, not the product): squared matrix elements of the LO channels with a
// second (light, massless) quark line and one gluon ("any process generated (at LO)"):
//   MFO_QQ_TTG  q(pa) q~(pb) -> t(k1) t~(k2) g(k3)      MFO_QG_TTQ  q(pa) g(pb) -> t(k1) t~(k2) q(k3)
// Five Feynman diagrams each, written out one by one from the rules of DESIGN.md reading O6.3 (Peskin-Schroeder, Feynman
// gauge): quark-gluon vertex i g gamma^mu T^a, quark propagator i (pslash + m)/(p^2 - m^2), gluon propagator
// -i g_{mu nu} delta^{ab} / p^2, three-gluon vertex g f^{abc} [g^{mu nu}(k-p)^rho + g^{nu rho}(p-q)^mu + g^{rho mu}(q-k)^nu]
// (all momenta incoming).  Explicit 4x4 gamma matrices, explicit Gell-Mann generators, the colour sum taken literally
// over all 3^4 x 8 colour assignments.  The file is self-contained on purpose (its own gamma matrices, generators and
// wavefunctions, restated from the same readings O6.1-O6.3): it shares no line with the CUDA path.
//
// Both processes are one amplitude with different external lines.  The LIGHT quark line runs from a column spinor `lcol`
// (all-incoming momentum pc flows into the line) to a row spinor `lrow` (all-incoming momentum pr):
//   q q~ -> t t~ g:  lcol = u(pa), pc = pa;  lrow = vbar(pb), pr = pb;   gluon outgoing: K = -k3, e = eps^*(k3)
//   q g  -> t t~ q:  lcol = u(pa), pc = pa;  lrow = ubar(k3), pr = -k3;  gluon incoming: K = pb,  e = eps(pb)
// (an overall sign from crossing a fermion does not matter in |M|^2).  The HEAVY line runs from v(k2) to ubar(k1).
// With  JL^mu  = (-i / PL^2) lrow (i g gamma^mu) lcol,  PL = pc + pr          (the light line's off-shell gluon, colour T^b_{ji})
// the five diagrams, as i M = sum_d L_d t_d(colours), are
//   d1  gluon off the heavy line next to the top:      L1 = ubar (i g eslash) S(PL - k2) (i g JLslash) v      t1 = (T^a T^b)_{c3 c4} T^b_{ji}
//   d2  gluon off the heavy line next to the antitop:  L2 = ubar (i g JLslash) S(K - k2) (i g eslash) v       t2 = (T^b T^a)_{c3 c4} T^b_{ji}
//   d3  gluon off the light line next to lcol:  J3^mu = (-i/P^2) lrow (i g gamma^mu) S0(pc + K) (i g eslash) lcol, L3 = ubar (i g J3slash) v,  t3 = T^b_{c3 c4} (T^b T^a)_{ji}
//   d4  gluon off the light line next to lrow:  J4^mu = (-i/P^2) lrow (i g eslash) S0(-pr - K) (i g gamma^mu) lcol, L4 = ubar (i g J4slash) v, t4 = T^b_{c3 c4} (T^a T^b)_{ji}
//   d5  three-gluon vertex:  J5^mu = (-i/P^2) g V3^{mu nu rho}(-P, PL, K) JL_nu e_rho,  L5 = ubar (i g J5slash) v,   t5 = f^{c b a} T^c_{c3 c4} T^b_{ji}
// with P = PL + K = k1 + k2 the momentum of the gluon that enters the heavy line, S(q) = i (qslash + m_t)/(q^2 - m_t^2),
// S0(q) = i qslash / q^2, j (i) the colour at the row (column) end of the light line, a the colour of the external gluon.
//   |M|^2 = (1/avg) sum_hel sum_{d d'} L_d conj(L_d') CC_{d d'},   CC_{d d'} = sum_colours t_d conj(t_d'),
// avg = 4 x 9 (q q~) or 4 x 24 (q g: 3 x 8 colours).  `ward` replaces e by K (the sum must vanish).
#include "mfo.h"
#include <complex>
#include <cmath>
#include <mutex>

namespace {
typedef std::complex<double> cd;
const cd I_(0.0, 1.0);
struct V4 { cd c[4]; };
struct Sp { cd c[4]; };
struct M4 { cd m[4][4]; };
M4 GAM[4];
cd TA[8][3][3];
double FABC[8][8][8];
cd CC[5][5];
std::once_flag once;

void init() {
  std::call_once(once, [] {
    const cd s[3][2][2] = {{{0, 1}, {1, 0}}, {{0, -I_}, {I_, 0}}, {{1, 0}, {0, -1}}};       // Pauli matrices
    for (int mu = 0; mu < 4; ++mu) for (int r = 0; r < 4; ++r) for (int c = 0; c < 4; ++c) GAM[mu].m[r][c] = 0;
    for (int a = 0; a < 2; ++a) { GAM[0].m[a][2 + a] = 1; GAM[0].m[2 + a][a] = 1; }         // chiral representation (O6.1)
    for (int i = 0; i < 3; ++i) for (int a = 0; a < 2; ++a) for (int b = 0; b < 2; ++b) { GAM[1 + i].m[a][2 + b] = s[i][a][b]; GAM[1 + i].m[2 + a][b] = -s[i][a][b]; }
    for (int a = 0; a < 8; ++a) for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) TA[a][i][j] = 0;   // T^a = lambda^a / 2
    TA[0][0][1] = 0.5; TA[0][1][0] = 0.5; TA[1][0][1] = -0.5 * I_; TA[1][1][0] = 0.5 * I_; TA[2][0][0] = 0.5; TA[2][1][1] = -0.5;
    TA[3][0][2] = 0.5; TA[3][2][0] = 0.5; TA[4][0][2] = -0.5 * I_; TA[4][2][0] = 0.5 * I_;
    TA[5][1][2] = 0.5; TA[5][2][1] = 0.5; TA[6][1][2] = -0.5 * I_; TA[6][2][1] = 0.5 * I_;
    const double s3 = 1.0 / std::sqrt(3.0);
    TA[7][0][0] = 0.5 * s3; TA[7][1][1] = 0.5 * s3; TA[7][2][2] = -s3;
    auto mul = [](const cd (*A)[3], const cd (*B)[3], cd (*R)[3]) { for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) { R[i][j] = 0; for (int k = 0; k < 3; ++k) R[i][j] += A[i][k] * B[k][j]; } };
    for (int a = 0; a < 8; ++a) for (int b = 0; b < 8; ++b) for (int c = 0; c < 8; ++c) {   // f^{abc} = -2i Tr([T^a, T^b] T^c)
      cd ab[3][3], ba[3][3], cm[3][3], x[3][3];
      mul(TA[a], TA[b], ab); mul(TA[b], TA[a], ba);
      for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) cm[i][j] = ab[i][j] - ba[i][j];
      mul(cm, TA[c], x);
      const cd v = -2.0 * I_ * (x[0][0] + x[1][1] + x[2][2]);
      FABC[a][b][c] = std::fabs(v.real()) < 1e-14 ? 0.0 : v.real();
    }
    // colour tensors of the five diagrams for every assignment (i, j, c3, c4, a), and their literal sums
    for (int d = 0; d < 5; ++d) for (int e = 0; e < 5; ++e) CC[d][e] = 0;
    for (int i = 0; i < 3; ++i) for (int j = 0; j < 3; ++j) for (int c3 = 0; c3 < 3; ++c3) for (int c4 = 0; c4 < 3; ++c4) for (int a = 0; a < 8; ++a) {
      cd t[5] = {0, 0, 0, 0, 0};
      for (int b = 0; b < 8; ++b) {
        cd ab[3][3], ba[3][3];
        mul(TA[a], TA[b], ab); mul(TA[b], TA[a], ba);
        t[0] += ab[c3][c4] * TA[b][j][i];
        t[1] += ba[c3][c4] * TA[b][j][i];
        t[2] += TA[b][c3][c4] * ba[j][i];
        t[3] += TA[b][c3][c4] * ab[j][i];
        for (int c = 0; c < 8; ++c) t[4] += FABC[c][b][a] * TA[c][c3][c4] * TA[b][j][i];
      }
      for (int d = 0; d < 5; ++d) for (int e = 0; e < 5; ++e) CC[d][e] += t[d] * std::conj(t[e]);
    }
  });
}

cd mdot(const V4 &a, const V4 &b) { return a.c[0] * b.c[0] - a.c[1] * b.c[1] - a.c[2] * b.c[2] - a.c[3] * b.c[3]; }
V4 vadd(const V4 &a, const V4 &b) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] + b.c[i]; return r; }
V4 vsub(const V4 &a, const V4 &b) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = a.c[i] - b.c[i]; return r; }
V4 vscale(cd s, const V4 &a) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = s * a.c[i]; return r; }
V4 vreal(const double *p, double sign) { V4 r; for (int i = 0; i < 4; ++i) r.c[i] = sign * p[i]; return r; }
M4 slash(const V4 &v) {           // gamma^mu v_mu
  M4 r;
  for (int a = 0; a < 4; ++a) for (int b = 0; b < 4; ++b)
    r.m[a][b] = GAM[0].m[a][b] * v.c[0] - GAM[1].m[a][b] * v.c[1] - GAM[2].m[a][b] * v.c[2] - GAM[3].m[a][b] * v.c[3];
  return r;
}
Sp matvec(const M4 &A, const Sp &x) { Sp r; for (int a = 0; a < 4; ++a) { r.c[a] = 0; for (int b = 0; b < 4; ++b) r.c[a] += A.m[a][b] * x.c[b]; } return r; }
Sp sscale(cd s, const Sp &x) { Sp r; for (int a = 0; a < 4; ++a) r.c[a] = s * x.c[a]; return r; }
cd rowcol(const Sp &row, const Sp &col) { cd s = 0; for (int a = 0; a < 4; ++a) s += row.c[a] * col.c[a]; return s; }
Sp adjoint(const Sp &u) { Sp r; for (int b = 0; b < 4; ++b) { r.c[b] = 0; for (int a = 0; a < 4; ++a) r.c[b] += std::conj(u.c[a]) * GAM[0].m[a][b]; } return r; }
// quark propagator i (qslash + m)/(q^2 - m^2) applied to a column spinor
Sp prop(const V4 &q, double m, const Sp &x) {
  Sp r = matvec(slash(q), x); const cd den = mdot(q, q) - m * m;
  for (int a = 0; a < 4; ++a) r.c[a] = I_ * (r.c[a] + m * x.c[a]) / den;
  return r;
}

// O6.2 external wavefunctions (HELAS helicity basis), restated
void chi(const double p[4], cd cp[2], cd cm[2]) {
  const double pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]), pt2 = p[1] * p[1] + p[2] * p[2];
  if (pabs < 1e-12 * std::fabs(p[0]) || (pt2 == 0.0 && p[3] < 0)) { cp[0] = 0; cp[1] = 1; cm[0] = -1; cm[1] = 0; return; }
  const double ppz = (p[3] >= 0) ? pabs + p[3] : pt2 / (pabs - p[3]);
  const double N = 1.0 / std::sqrt(2.0 * pabs * ppz);
  cp[0] = N * ppz; cp[1] = N * cd(p[1], p[2]); cm[0] = N * cd(-p[1], p[2]); cm[1] = N * ppz;
}
Sp wf_fermion(int kind, const double p[4], double m, int lam) {      // kind 0: u(p, lam); 1: v(p, lam)
  const double pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  const double wp = std::sqrt(p[0] + pabs), wm = (m == 0.0) ? 0.0 : m / wp;
  cd cp[2], cm[2]; chi(p, cp, cm);
  auto om = [&](int s) { return s > 0 ? wp : wm; };
  Sp r;
  if (kind == 0) { const cd *c = lam > 0 ? cp : cm; r.c[0] = om(-lam) * c[0]; r.c[1] = om(-lam) * c[1]; r.c[2] = om(lam) * c[0]; r.c[3] = om(lam) * c[1]; }
  else { const cd *c = lam > 0 ? cm : cp; const double l = lam; r.c[0] = -l * om(lam) * c[0]; r.c[1] = -l * om(lam) * c[1]; r.c[2] = l * om(-lam) * c[0]; r.c[3] = l * om(-lam) * c[1]; }
  return r;
}
V4 wf_vector(const double p[4], int lam) {                            // eps(p, lam) = (-lam eps1 - i eps2)/sqrt2
  const double pt = std::sqrt(p[1] * p[1] + p[2] * p[2]), pabs = std::sqrt(p[1] * p[1] + p[2] * p[2] + p[3] * p[3]);
  double e1[4], e2[4];
  if (pt == 0.0) { e1[0] = 0; e1[1] = 1; e1[2] = 0; e1[3] = 0; e2[0] = 0; e2[1] = 0; e2[2] = (p[3] >= 0 ? 1.0 : -1.0); e2[3] = 0; }
  else { e1[0] = 0; e1[1] = p[1] * p[3] / (pabs * pt); e1[2] = p[2] * p[3] / (pabs * pt); e1[3] = -pt / pabs; e2[0] = 0; e2[1] = -p[2] / pt; e2[2] = p[1] / pt; e2[3] = 0; }
  V4 r; const double l = lam;
  for (int i = 0; i < 4; ++i) r.c[i] = (-l * e1[i] - I_ * e2[i]) / std::sqrt(2.0);
  return r;
}
// V3^{mu nu rho}(k,p,q) A_nu B_rho = A^mu ((k-p).B) + (p-q)^mu (A.B) + B^mu ((q-k).A)
V4 v3contract(const V4 &k, const V4 &p, const V4 &q, const V4 &A, const V4 &B) {
  const cd c1 = mdot(vsub(k, p), B), c2 = mdot(A, B), c3 = mdot(vsub(q, k), A);
  const V4 pq = vsub(p, q); V4 r;
  for (int i = 0; i < 4; ++i) r.c[i] = A.c[i] * c1 + pq.c[i] * c2 + B.c[i] * c3;
  return r;
}
// the open Lorentz index of a fermion bilinear: row (i g gamma^mu) col, upper index
V4 current(const Sp &row, const Sp &col, double gs) {
  V4 r; for (int mu = 0; mu < 4; ++mu) r.c[mu] = I_ * gs * rowcol(row, matvec(GAM[mu], col)); return r;
}
}  // namespace

// mom: [5][4] = pa, pb, k1 (t), k2 (t~), k3 (gluon, or the outgoing light quark); partonic frame of the caller's choice
extern "C" int mfo_me2_2q(int process, const double *mom, double m_top, double alpha_s, int ward, double *out) {
  if (process != MFO_QQ_TTG && process != MFO_QG_TTQ) return MFO_EINVAL;
  init();
  const double gs = std::sqrt(4.0 * M_PI * alpha_s);
  const double *pa = mom, *pb = mom + 4, *k1 = mom + 8, *k2 = mom + 12, *k3 = mom + 16;
  const bool qq = process == MFO_QQ_TTG;
  const V4 pc = vreal(pa, 1.0), pr = qq ? vreal(pb, 1.0) : vreal(k3, -1.0);
  const V4 K = qq ? vreal(k3, -1.0) : vreal(pb, 1.0);
  const V4 q2 = vreal(k2, 1.0), PL = vadd(pc, pr), P = vadd(PL, K);
  long double tot = 0;
  for (int h = 0; h < 32; ++h) {
    const int lc = (h & 1) ? 1 : -1, lr = (h & 2) ? 1 : -1, l1 = (h & 4) ? 1 : -1, l2 = (h & 8) ? 1 : -1, lg = (h & 16) ? 1 : -1;
    const Sp lcol = wf_fermion(0, pa, 0.0, lc);
    const Sp lrow = qq ? adjoint(wf_fermion(1, pb, 0.0, lr)) : adjoint(wf_fermion(0, k3, 0.0, lr));
    const Sp ub = adjoint(wf_fermion(0, k1, m_top, l1));
    const Sp v = wf_fermion(1, k2, m_top, l2);
    V4 e = wf_vector(qq ? k3 : pb, lg);
    if (qq) for (int i = 0; i < 4; ++i) e.c[i] = std::conj(e.c[i]);             // outgoing gluon: eps^*
    if (ward) e = K;
    const M4 es = slash(e);
    const V4 JL = vscale(-I_ / mdot(PL, PL), current(lrow, lcol, gs));
    cd L[5];
    // d1, d2: the external gluon on the heavy line
    L[0] = rowcol(ub, sscale(I_ * gs, matvec(es, prop(vsub(PL, q2), m_top, sscale(I_ * gs, matvec(slash(JL), v))))));
    L[1] = rowcol(ub, sscale(I_ * gs, matvec(slash(JL), prop(vsub(K, q2), m_top, sscale(I_ * gs, matvec(es, v))))));
    // d3, d4: on the light line
    const cd gp = -I_ / mdot(P, P);
    const V4 J3 = vscale(gp, current(lrow, prop(vadd(pc, K), 0.0, sscale(I_ * gs, matvec(es, lcol))), gs));
    Sp rowe;                                                                      // lrow (i g eslash): a row times a matrix
    for (int b = 0; b < 4; ++b) { rowe.c[b] = 0; for (int a = 0; a < 4; ++a) rowe.c[b] += lrow.c[a] * es.m[a][b]; rowe.c[b] *= I_ * gs; }
    V4 J4;
    {
      const V4 q = vscale(-1.0, vadd(pr, K));
      for (int mu = 0; mu < 4; ++mu) J4.c[mu] = gp * rowcol(rowe, prop(q, 0.0, sscale(I_ * gs, matvec(GAM[mu], lcol))));
    }
    L[2] = rowcol(ub, sscale(I_ * gs, matvec(slash(J3), v)));
    L[3] = rowcol(ub, sscale(I_ * gs, matvec(slash(J4), v)));
    // d5: three-gluon vertex, colour index of the new current first: f^{c b a} (b: light line, a: external gluon)
    const V4 J5 = vscale(gp * gs, v3contract(vscale(-1.0, P), PL, K, JL, e));
    L[4] = rowcol(ub, sscale(I_ * gs, matvec(slash(J5), v)));
    cd s = 0;
    for (int d = 0; d < 5; ++d) for (int f = 0; f < 5; ++f) s += L[d] * std::conj(L[f]) * CC[d][f];
    tot += s.real();
  }
  *out = (double)(tot / (qq ? 36.0L : 96.0L));          // 1/4 helicities x 1/9 (q q~) or 1/24 (q g) colours of the incoming pair
  return MFO_OK;
}
