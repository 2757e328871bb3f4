// mf_params.h -- host-side validation of mf_config_t and derivation of the kernel constants
// (MfParams).  Used by the C-ABI (mf_api.cu); the test harness includes it as well.
#pragma once
#include "../../include/madflow_b200.h"
#include "mf_event.cuh"
#include <string>

static_assert(MFD_GEN_CLASSIC == MF_GEN_CLASSIC_RAMBO && MFD_GEN_LINEAR == MF_GEN_LINEAR_TAU, "device flags follow the header");

static inline int mf_process_shape(int process, uint32_t generator, int* d, int* n_final, int* ng) {
  static const int nf[8] = {2, 2, 3, 4, 2, 2, 3, 3};
  if (process < 0 || process > 7) return -1;
  *n_final = nf[process];
  *d = (process == MF_EE_MUMU) ? 2 : 2 + 3 * nf[process] - 4;
  if (generator & MF_GEN_CLASSIC_RAMBO) *d = 2 + 4 * nf[process];       // O4': 4n uniforms
  *ng = (process == MF_EE_MUMU) ? 0 : nf[process];      // gluon legs of gg -> t t~ + (n_final-2) g (= powers of g_s^2; 2 for q q~ -> t t~)
  return 0;
}

// device copy of the 11-flavour grid (processes 4 and 5): host [11][nx][nq] (index = PDG id + 5) -> flavour-innermost,
// rows pdf_iq0 .. pdf_iq0 + pdf_nqs - 1 only: out[nx][pdf_nqs * MF_NFL + MF_XPAD] (P.pdf_smem doubles, zeroed by the caller:
// the pad entries are never read), slot = PDG id + 5.
static inline void mf_flavour_slice(const MfParams& P, const double* pdf11, double* out) {
  const size_t ntab = (size_t)P.pdf_nx * P.pdf_nq;
  for (int f = 0; f < MF_NFL; ++f)
    for (int ix = 0; ix < P.pdf_nx; ++ix)
      for (int r = 0; r < P.pdf_nqs; ++r)
        out[(size_t)ix * (P.pdf_nqs * MF_NFL + MF_XPAD) + r * MF_NFL + f] = pdf11[(size_t)f * ntab + (size_t)ix * P.pdf_nq + P.pdf_iq0 + r];
}

// returns MF_OK or MF_EINVAL / MF_EUNSUPPORTED with a message in err
static inline int mf_fill_params(const mf_config_t* c, MfParams* P, std::string& err) {
  if (!c) { err = "cfg is NULL"; return MF_EINVAL; }
  if (c->struct_size != sizeof(mf_config_t)) { err = "struct_size mismatch (ABI)"; return MF_EINVAL; }
  int d, nfin, ng;
  if (c->generator & ~(uint32_t)(MF_GEN_CLASSIC_RAMBO | MF_GEN_LINEAR_TAU)) { err = "unknown generator flag"; return MF_EINVAL; }
  if (mf_process_shape(c->process, c->generator, &d, &nfin, &ng)) { err = "unknown process"; return MF_EINVAL; }
  if (c->generator && c->process == MF_EE_MUMU) { err = "generator variants apply to processes 1-3"; return MF_EINVAL; }
  if (c->precision != 64 && !(c->precision == 32 && c->process == MF_GG_TTG)) {
    err = "precision must be 64 (32: the fp32 |M|^2 variant exists for gg -> tt~g only)"; return MF_EUNSUPPORTED;
  }
  if (c->n_bins < 1 || c->n_bins > MF_NBMAX) { err = "n_bins must be in 1..64"; return MF_EINVAL; }
  if (!(c->sqrt_s > 0.0)) { err = "sqrt_s must be positive"; return MF_EINVAL; }
  if (!(c->alpha_damp >= 0.0)) { err = "alpha_damp must be >= 0"; return MF_EINVAL; }
  if (!(c->gev2_to_pb > 0.0)) { err = "gev2_to_pb must be positive"; return MF_EINVAL; }
  MfParams p = {};
  p.process = c->process; p.d = d; p.n_final = nfin; p.nb = (int)c->n_bins; p.gen = (int32_t)c->generator;
  p.key0 = (uint32_t)c->seed; p.key1 = (uint32_t)(c->seed >> 32);
  p.s = c->sqrt_s * c->sqrt_s; p.m_top = c->m_top;
  p.ptmin = c->ptmin_g; p.etamax = c->etamax_g; p.drmin = c->drmin_gg;
  p.tanh_etamax = c->etamax_g > 0.0 ? tanh(c->etamax_g) : 1.0;
  const double PI = 3.14159265358979323846;
  if (c->process == MF_EE_MUMU) {
    if (!(c->alpha_em > 0.0)) { err = "alpha_em must be positive"; return MF_EINVAL; }
    const double e2 = 4.0 * PI * c->alpha_em;
    p.me_pref = e2 * e2 * MF_ME2_EE_MUMU_SCALE;         // e^4 / 4 (spin average, A12)
    p.wconst = c->gev2_to_pb / 2.0;
    p.ltau0 = 0.0;
  } else {
    if (!(c->m_top > 0.0) || !(c->alpha_s > 0.0)) { err = "m_top and alpha_s must be positive"; return MF_EINVAL; }
    if (!c->pdf_xf || c->pdf_nx < 2 || c->pdf_nq < 2) { err = "pdf grid required"; return MF_EINVAL; }
    const uint32_t nfl = c->pdf_nf ? c->pdf_nf : 1;
    if (nfl != 1 && nfl != 11) { err = "pdf_nf must be 0, 1 or 11"; return MF_EINVAL; }
    if ((c->process >= MF_QQ_TT) != (nfl == 11)) { err = "processes 4-7 need the 11-flavour grid, processes 1-3 the gluon table"; return MF_EINVAL; }
    if ((uint64_t)c->pdf_nx * c->pdf_nq * 8ull > 160ull * 1024ull) { err = "pdf table larger than 160 KB"; return MF_EINVAL; }
    if (!(c->pdf_xmin > 0.0 && c->pdf_xmax > c->pdf_xmin && c->pdf_qmin > 0.0 && c->pdf_qmax > c->pdf_qmin)) { err = "bad pdf ranges"; return MF_EINVAL; }
    const int ngl = nfin - 2;
    const double thr = 2.0 * c->m_top + ngl * (c->ptmin_g > 0.0 ? c->ptmin_g : 0.0);   // O3: shat_min
    const double tau0 = thr * thr / p.s;
    if (!(tau0 < 1.0) || tau0 < c->pdf_xmin || c->mu_f < c->pdf_qmin || c->mu_f > c->pdf_qmax) {
      err = "kinematics outside the PDF grid"; return MF_EINVAL;
    }
    p.ltau0 = log(tau0); p.tau0 = tau0;
    double gs2n = 1.0;
    for (int i = 0; i < ng; ++i) gs2n *= 4.0 * PI * c->alpha_s;
    const double scale = (c->process == MF_GG_TT) ? MF_ME2_GG_TT_SCALE : (c->process == MF_GG_TTG) ? MF_ME2_GG_TTG_SCALE : MF_ME2_GG_TTGG_LANES_SCALE;
    p.me_pref = gs2n / 256.0 * scale;                   // 1/4 helicities x 1/64 colours (A12)
    if (c->process == MF_PP_TT) p.me_pref = gs2n / 256.0 * MF_ME2_GG_TT_SCALE;         // its g g -> t t~ subprocess
    p.me_pref_qq = gs2n * (2.0 / 9.0) * MF_ME2_EE_MUMU_SCALE;                           // O6q: colour sum 2 / 9 colours, 1/4 spins
    if (c->process == MF_QQ_TT) p.me_pref = p.me_pref_qq;
    if (c->process == MF_QQ_TTG) p.me_pref = gs2n * MF_ME2_QQ_TTG_SCALE;               // g_s^6 / (9 colour denominator x 36)
    if (c->process == MF_QG_TTQ) p.me_pref = gs2n * MF_ME2_QG_TTQ_SCALE;               // ... x 96
    p.wconst = (ngl == 2 ? 0.5 : 1.0) * c->gev2_to_pb / 2.0;
    p.pdf_nx = (int)c->pdf_nx; p.pdf_nq = (int)c->pdf_nq;
    p.pdf_lx0 = log(c->pdf_xmin);
    p.pdf_ihx = (double)(c->pdf_nx - 1) / (log(c->pdf_xmax) - p.pdf_lx0);
    p.pdf_lq0 = log(c->pdf_qmin * c->pdf_qmin);
    p.pdf_ihq = (double)(c->pdf_nq - 1) / (log(c->pdf_qmax * c->pdf_qmax) - p.pdf_lq0);
    p.pdf_lq = log(c->mu_f * c->mu_f);
    p.pdf_smem = p.pdf_nx * p.pdf_nq; p.pdf_iq0 = 0; p.pdf_nqs = p.pdf_nq;
    if (nfl == 11) {                                   // flavour grid: keep the Q^2 rows the stencil of mu_F touches (mf_pdf_strided)
      int iq = (int)floor((p.pdf_lq - p.pdf_lq0) * p.pdf_ihq);
      iq = iq < 0 ? 0 : (iq > p.pdf_nq - 2 ? p.pdf_nq - 2 : iq);
      const int lo = iq - 1 < 0 ? 0 : iq - 1, hi = iq + 2 > p.pdf_nq - 1 ? p.pdf_nq - 1 : iq + 2;
      p.pdf_iq0 = lo; p.pdf_nqs = hi - lo + 1;
      p.pdf_smem = p.pdf_nx * (p.pdf_nqs * MF_NFL + MF_XPAD);
    }
  }
  *P = p;
  return MF_OK;
}
