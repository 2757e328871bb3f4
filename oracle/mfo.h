/* mfo.h -- C API of the ORACLE (test infrastructure, NOT the product).
 *
 * Plain, slow, fp64 CPU restatement of the MadFlow leading-order integrand hot path
 * (arxiv 2105.10529; PAPER.md:29,59 pipeline "random numbers -> phase space -> matrix element ->
 * histogram accumulation", PAPER.md:47,67,69 structure of the matrix element).  The paper prints no
 * formulas; every step follows the reading listed in DESIGN.md ("Readings", items O1-O11 / A1-A24,
 * taken from SURVEY.md section 8(c)).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use
 * anything under oracle/.  It shares no code, header, table or constant generator with the CUDA
 * path (paper_2105_10529_b200/csrc); the struct definitions below are the oracle's own.
 *
 * Pins (what the functions below are checked against, other than themselves): tests/test_oracle_core.py,
 * tests/test_oracle_me.py, tests/test_oracle_crosscheck.py and the fixtures in tests/golden/ -- listed in
 * DESIGN.md section 4.  Parity unpinned: none of the functions; of the RESULTS, the absolute cross
 * sections of configs 2 and 3 (no closed form, no value in the paper) are pinned factor by factor and,
 * as a whole, only within the Monte Carlo error of the independent-generator cross-check (2.7 % / 12 %).
 *
 * All pointers are HOST pointers.  All functions return 0 on success, <0 on error.
 */
#ifndef MFO_H
#define MFO_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { MFO_OK = 0, MFO_EINVAL = -1, MFO_ENOMEM = -2, MFO_ESTATE = -4, MFO_EUNSUPPORTED = -5 };
enum { MFO_EE_MUMU = 0, MFO_GG_TT = 1, MFO_GG_TTG = 2, MFO_GG_TTGG = 3,
       MFO_QQ_TT = 4,          /* q q~ -> t t~ summed over the five light flavours     */
       MFO_PP_TT = 5,          /* p p -> t t~ at LO: the sum of the subprocesses g g -> t t~ and q q~ -> t t~   */
       MFO_QQ_TTG = 6,         /* p p -> t t~ g through q q~ -> t t~ g (five diagrams), five flavours, both beam orientations   */
       MFO_QG_TTQ = 7 };       /* p p -> t t~ + quark jet through q g, g q, q~ g, g q~ -> t t~ q (five diagrams each)      */

typedef struct {
  int32_t  process;            /* MFO_*                                                          */
  uint64_t seed;               /* Philox key (O1)                                                */
  uint32_t n_bins;             /* VEGAS bins per dimension (50)                                  */
  double   alpha_damp;         /* VEGAS damping exponent (1.5)                                   */
  double   sqrt_s, m_top, alpha_s, alpha_em, mu_f;
  double   ptmin_g, etamax_g, drmin_gg;   /* cuts; <= 0 disables                                 */
  double   gev2_to_pb;         /* 0.3894e9                                                       */
  const double *pdf_xf;        /* host [nx][nq] row-major table of x*g(x,Q^2); must not be NULL  */
  uint32_t pdf_nx, pdf_nq;
  double   pdf_xmin, pdf_xmax, pdf_qmin, pdf_qmax;
  uint32_t generator;          /* MFO_GEN_* flags; 0 = the generators of the configs   */
  uint32_t pdf_nf;             /* flavour tables in pdf_xf: 0 or 1 = the gluon table [nx][nq] (processes 1-3);
                                * 11 = [11][nx][nq], flavour index = PDG id + 5 (b~ c~ s~ u~ d~ g d u s c b),
                                * required by MFO_QQ_TT (flavour-summed PDFs)                  */
} mfo_config_t;
/* MFO_QQ_TT ("any process generated (at LO)"): one diagram, s-channel gluon,
 *   M = g_s^2 T^a_{ji} T^a_{kl} [vbar(pb) gamma^mu u(pa)] [ubar(k1) gamma_mu v(k2)] / shat,
 * averaged over 4 helicities x 9 colours of the incoming pair (O6q).  Same 2-body kinematics and VEGAS
 * dimensions as MFO_GG_TT.  The parton luminosity is summed over flavours and both beam orientations:
 *   F = J_V J_x [sum_{q=1..5} f_q(x1) f_q~(x2) + f_q~(x1) f_q(x2)] |M|^2 W_PS K / (2 shat)
 * (|M|^2 is symmetric under the exchange of the beams); the per-event record pdf[2] holds the two sums
 * sum_q xf_q(x1) xf_q~(x2) and sum_q xf_q~(x1) xf_q(x2).  Selectable generators apply as for process 1.   */
/* selectable generators (processes 1-3):
 *  MFO_GEN_CLASSIC_RAMBO  textbook RAMBO (Kleiss, Stirling, Ellis 1986) with 4n uniforms instead of the 3n-4-random
 *                         sequential form; VEGAS dimensions d = 2 + 4n (mfo_rambo_classic)
 *  MFO_GEN_LINEAR_TAU     tau = tau0 + (1 - tau0) y0 instead of tau = tau0^(1-y0) (mfo_x_map_linear)     */
enum { MFO_GEN_CLASSIC_RAMBO = 1, MFO_GEN_LINEAR_TAU = 2 };

/* MFO_PP_TT: both subprocesses in one integrand on the 11-flavour grid,
 *   F = J_V J_x [ xg(x1) xg(x2) |M_gg|^2 + (L12 + L21) |M_qq|^2 ] / (x1 x2) W_PS K / (2 shat),
 * L12, L21 the flavour sums of MFO_QQ_TT, the gluon density from table 5.  Per-event record: pdf[2] =
 * { xg(x1) xg(x2), L12 + L21 } (the two x1 x2-weighted luminosities), me2 = their luminosity-weighted mean |M|^2. */
typedef struct {               /* host buffers owned by the caller; NULL = skip                  */
  double  *weight;             /* [n]  F_i = w_i f_i  (t_i * N)                                  */
  double  *x;                  /* [n][d]  VEGAS points                                           */
  uint8_t *bins;               /* [n][d]                                                         */
  double  *momenta;            /* [n][2+n_final][4] (E,px,py,pz), partonic CM frame              */
  double  *me2;                /* [n]  |M|^2 averaged/summed, before the symmetry factor         */
  double  *pdf;                /* [n][2]  xg(x1), xg(x2)                                         */
  uint8_t *pass;               /* [n]  1 if the event passed the cuts                            */
} mfo_eval_out_t;

typedef struct { double integral, sigma; uint64_t n_events, n_pass, n_nonfinite; } mfo_iter_t;
typedef struct { double integral, sigma, chi2_dof; uint32_t n_iter; } mfo_result_t;
typedef struct mfo_vegas mfo_vegas_t;

/* MFO_QQ_TTG, MFO_QG_TTQ ("q q~ -> t t~ (g), q g -> t t~ q").  Kinematics, VEGAS dimensions, cuts
 * (on the third final particle: the gluon, resp. the light-quark jet) and generators of MFO_GG_TTG; 11-flavour grid.
 *   MFO_QQ_TTG: F = J_V J_x [L12 |M(q(p1) q~(p2))|^2 + L21 |M(q~(p1) q(p2))|^2] / (x1 x2) W_PS K / (2 shat), L12, L21 the
 *     flavour sums of MFO_QQ_TT; the two |M|^2 differ (charge asymmetry): the second is the first with the beams exchanged.
 *     Record: pdf[2] = {L12, L21}, me2 = their luminosity-weighted mean |M|^2.
 *   MFO_QG_TTQ: F = J_V J_x [Lqg |M(q g)|^2 + Lgq |M(g q)|^2 + Lq~g |M(q~ g)|^2 + Lgq~ |M(g q~)|^2] / (x1 x2) W_PS K / (2 shat),
 *     Lqg = sum_q xf_q(x1) xg(x2), Lgq = xg(x1) sum_q xf_q(x2), Lq~g, Lgq~ with the antiquark tables; |M(g q)|^2 = |M(q g)|^2
 *     with the beams exchanged, |M(q~ g -> t t~ q~)|^2 = |M(q g -> t t~ q)|^2 with t and t~ exchanged (charge conjugation).
 *     Record: pdf[2] = {Lqg + Lq~g, Lgq + Lgq~}, me2 = the luminosity-weighted mean of the four |M|^2.
 * mfo_me2 returns the basic |M|^2 (q along mom[0]): averaged over 4 helicities and 9 (q q~) / 24 (q g) colours.            */
int mfo_me2_2q(int process, const double *mom /* [5][4]: pa, pb, k1 (t), k2 (t~), k3 */, double m_top, double alpha_s,
               int ward /* != 0: the gluon's polarisation replaced by its momentum (must give 0) */, double *out);

/* ---- the path (same calls as the product's C-ABI, on host memory) ---------------------------- */
int mfo_vegas_create(const mfo_config_t *cfg, mfo_vegas_t **out);
int mfo_vegas_destroy(mfo_vegas_t *h);
int mfo_ndim(const mfo_vegas_t *h, uint32_t *d, uint32_t *n_final);
int mfo_integrand_eval(mfo_vegas_t *h, uint32_t iteration, uint64_t first_event, uint64_t n_events,
                       const mfo_eval_out_t *out, int n_threads);
int mfo_vegas_iterate(mfo_vegas_t *h, uint64_t n_events, int n_threads, mfo_iter_t *out);
int mfo_result(mfo_vegas_t *h, mfo_result_t *out);
int mfo_get_grid(mfo_vegas_t *h, double *edges /* [d][n_bins+1] */);
int mfo_set_grid(mfo_vegas_t *h, const double *edges);
/* raw sums of the last iteration: acc[0]=sum t, acc[1]=sum t^2, acc[2+j*nb+k]=H[j][k] (O9) */
int mfo_get_accum(mfo_vegas_t *h, double *acc /* [2 + d*n_bins] */);
/* accumulate events [first, first+n) of an iteration of n_total events into acc (adds; O9);
 * counts[0] += n_pass, counts[1] += n_nonfinite.  Used by the sharding tests. */
int mfo_vegas_accumulate(mfo_vegas_t *h, uint32_t iteration, uint64_t first_event, uint64_t n_events,
                         uint64_t n_total, int n_threads, double *acc, uint64_t *counts);
/* finish an iteration from raw sums (O10): record (I, sigma), refine the grid */
int mfo_vegas_finalize(mfo_vegas_t *h, const double *acc, uint64_t n_total, uint64_t n_pass,
                       uint64_t n_nonfinite, mfo_iter_t *out);
/* Observable histograms filled in the same pass as the integral ("histogram accumulation";
 * the differential cross section in the top-quark pT is the paper's physics plot; SURVEY
 * section 8(f) item 1).  Plain definition: for every event i of [first, first+n) with weight F_i != 0,
 * t_i = F_i / n_total, the observable v_i is computed from the final-state momenta (partonic CM frame;
 * all kinds are invariant under the boost along the beam) and
 *   b = n_bins      if v < lo        (underflow slot)
 *   b = n_bins + 1  if v >= hi       (overflow slot)
 *   b = floor((v - lo) / (hi - lo) * n_bins)  otherwise (clamped to n_bins - 1),
 *   sum[o][b] += t_i,  sum2[o][b] += t_i^2          (long double sums; arrays [n_obs][n_bins + 2], ADDED to).
 * kinds: 0 = pT of final particle 1 (top / mu-), 1 = pT of final particle 2 (antitop / mu+),
 *        2 = invariant mass of particles 1+2, 3 = pT of final particle 3 (first gluon; processes 2, 3). */
enum { MFO_OBS_PT_1 = 0, MFO_OBS_PT_2 = 1, MFO_OBS_M_12 = 2, MFO_OBS_PT_3 = 3 };
typedef struct { int32_t kind; uint32_t n_bins; double lo, hi; } mfo_observable_t;
int mfo_observable_hist(mfo_vegas_t *h, uint32_t iteration, uint64_t first_event, uint64_t n_events,
                        uint64_t n_total, int n_threads, const mfo_observable_t *obs, uint32_t n_obs,
                        double *sum, double *sum2);
int mfo_max_threads(void);

/* ---- single steps, exported so that the tests can pin each one ------------------------------- */
/* O1 */
void mfo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
void mfo_uniforms(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t d, double *u);
/* O2 */
void mfo_vegas_map(const double *edges, uint32_t d, uint32_t nb, const double *u,
                   double *x, uint8_t *bins, double *jac);
/* O10 refinement of one set of edges [d][nb+1] from H [d][nb] */
void mfo_refine(const double *edges_in, const double *H, uint32_t d, uint32_t nb, double alpha,
                double *edges_out);
/* O11 */
void mfo_combine(const double *I, const double *sig, uint32_t n, mfo_result_t *out);
/* O3: y0,y1 -> x1,x2,shat,Jx */
void mfo_x_map(double y0, double y1, double s, double shat_min, double *x1, double *x2,
               double *shat, double *jx);
/* O3': linear-tau variant: tau = tau0 + (1 - tau0) y0, x1 = tau^y1, x2 = tau/x1, Jx = (1 - tau0)(-ln tau) */
void mfo_x_map_linear(double y0, double y1, double s, double shat_min, double *x1, double *x2,
                      double *shat, double *jx);
/* O4': textbook RAMBO.  rs[4n] uniforms, particle i uses rs[4i..4i+3]: c = 2 r0 - 1, phi = 2 pi r1,
 * q0 = -ln(r2 r3), q = q0 (1, s cos phi, s sin phi, c); Q = sum q, M = sqrt(Q^2), b = -Qvec/M, x = sqrt(shat)/M,
 * gamma = Q0/M, a = 1/(1+gamma); p0_i = x (gamma q0 + b.q), pvec_i = x (qvec + b q0 + a (b.q) b).
 * Output: massless momenta p0 [n][4] in the CM frame, flat in phase space: the weight is the constant mfo_w0.  */
void mfo_rambo_classic(uint32_t n, double shat, const double *rs, double *p0);
/* O4.4: RAMBO's massive rescaling of massless CM momenta p0 [n][4]: xi with sum sqrt(m^2 + xi^2 E^2) = sqrt(shat)
 * (Newton, A7), k [n][4] massive momenta, out2 = {Wm, xi}; returns the Newton steps (step 4 of mfo_phase_space) */
int mfo_massive_rescale(uint32_t n, double shat, const double *masses, const double *p0, double *k, double *out2);
/* O4: n-body phase space from 3n-4 numbers. p0: massless momenta [n][4], k: massive [n][4],
 * Mint[n] intermediate masses (Mint[0]=sqrt(shat)), out3 = {W0, Wm, xi}; returns Newton steps */
int mfo_phase_space(uint32_t n, double shat, const double *masses, const double *rs,
                    double *p0, double *k, double *Mint, double *out3);
/* O5 */
double mfo_pdf_interp(const double *xf, uint32_t nx, uint32_t nq, double xmin, double xmax,
                      double qmin, double qmax, double x, double q2);
/* O6.2: kind 0 = u (incoming fermion), 1 = v (outgoing antifermion); out = 4 complex (re,im) */
void mfo_wf_fermion(int kind, const double p[4], double m, int lambda, double out[8]);
/* polarisation vector eps(p,lambda) (not conjugated); out = 4 complex, upper index */
void mfo_wf_vector(const double p[4], int lambda, double out[8]);
/* gamma^mu in the chiral representation, out[mu][r][c] complex -> [4][4][4][2] */
void mfo_gamma(double out[128]);
/* O6.6: colour matrix numerators over the common denominator, [nf][nf], nf = ng! */
int mfo_colour_matrix(uint32_t ng, double *numer, double *denom);
/* SU(3): T^a (a=0..7) as [8][3][3][2] and f^{abc} as [8][8][8] */
void mfo_su3(double *T, double *f);
/* O6.5 counts: diagrams, colour-stripped sub-amplitudes, flows */
int mfo_diagram_counts(uint32_t ng, uint32_t *ndiag, uint32_t *nsub, uint32_t *nflow);
/* O6: |M|^2 averaged over initial and summed over final helicities/colours (before S_f) at the
 * given momenta [2+n_final][4] (incoming k1,k2 then final), algorithm A (diagram list + flows) */
int mfo_me2(int process, const double *mom, double m_top, double alpha_s, double alpha_em,
            double *out);
/* same with the literal colour-dressed recursion (algorithm B) and explicit colour sum;
 * hel_only >= 0 restricts the helicity sum to that single combination index                    */
int mfo_me2_literal(int process, const double *mom, double m_top, double alpha_s, int hel_only,
                    double *out);
/* algorithm A for one helicity combination hel[2+n_final] (+-1): jamp[nf] complex, and the
 * colour-summed |M|^2 of that helicity (no averaging).  ward_leg >= 0 replaces that gluon leg's
 * polarisation by its momentum (P19).                                                          */
int mfo_jamps(int process, const double *mom, double m_top, double alpha_s, const int *hel,
              int ward_leg, double *jamp /* [nf][2] */, double *me2_hel);
/* algorithm B amplitude iM for explicit colours: col_g[ng] in 0..7, c3,c4 in 0..2 */
int mfo_amp_literal(int process, const double *mom, double m_top, double alpha_s, const int *hel,
                    const int *col_g, int c3, int c4, int ward_leg, double out[2]);
/* O7: cuts on final gluons in the lab frame; obs = {pt_i, eta_i (per gluon)..., dR} */
int mfo_cuts(uint32_t n_gluons, const double *kg /* [n_gluons][4] */, double x1, double x2,
             double ptmin, double etamax, double drmin, double *obs);
/* O4.3 */
double mfo_w0(uint32_t n, double shat);
const char *mfo_last_error(void);

#ifdef __cplusplus
}
#endif
#endif
