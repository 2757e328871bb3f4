// mfo_integrand.cpp -- ORACLE (test infrastructure, not the product): the event weight, the
// reductions, the iteration result and the handle-level calls (O8-O11 of DESIGN.md; PAPER.md:59
// pipeline, PAPER.md:31 VegasFlow integrator).  Plain loops; host threads only split the event range.
#include "mfo.h"
#include <cmath>
#include <cstring>
#include <string>
#include <vector>
#include <new>
#include <thread>
#include <functional>

static thread_local std::string g_err;
extern "C" const char *mfo_last_error(void) { return g_err.c_str(); }
extern "C" int mfo_max_threads(void) { unsigned n = std::thread::hardware_concurrency(); return n ? (int)n : 1; }
// static split of [0,n) over nt host threads (events are independent: counter-based RNG)
static void parallel_ranges(uint64_t n, int nt, const std::function<void(int, uint64_t, uint64_t)> &fn) {
  if (nt <= 1) { fn(0, 0, n); return; }
  std::vector<std::thread> th;
  for (int t = 0; t < nt; ++t) th.emplace_back(fn, t, n * (uint64_t)t / nt, n * (uint64_t)(t + 1) / nt);
  for (auto &x : th) x.join();
}

struct mfo_vegas {
  mfo_config_t cfg; std::vector<double> pdf;
  uint32_t d, n_final; std::vector<double> edges; std::vector<double> masses;
  double shat_min, sym;
  uint32_t iteration; std::vector<double> I, sig; std::vector<double> acc;
};

extern "C" int mfo_vegas_create(const mfo_config_t *cfg, mfo_vegas_t **out) {
  if (!cfg || !out) { g_err = "null argument"; return MFO_EINVAL; }
  if (cfg->process < 0 || cfg->process > 7) { g_err = "unknown process"; return MFO_EINVAL; }
  if (cfg->n_bins < 1 || cfg->n_bins > 255) { g_err = "n_bins out of range"; return MFO_EINVAL; }
  if (!(cfg->sqrt_s > 0)) { g_err = "sqrt_s must be positive"; return MFO_EINVAL; }
  mfo_vegas *h = new (std::nothrow) mfo_vegas(); if (!h) return MFO_ENOMEM;
  h->cfg = *cfg;
  static const uint32_t nfin[8] = {2, 2, 3, 4, 2, 2, 3, 3};
  h->n_final = nfin[cfg->process];
  h->d = (cfg->process == MFO_EE_MUMU) ? 2 : 2 + 3 * h->n_final - 4;
  if (cfg->generator & ~(uint32_t)(MFO_GEN_CLASSIC_RAMBO | MFO_GEN_LINEAR_TAU)) { g_err = "unknown generator flag"; delete h; return MFO_EINVAL; }
  if (cfg->generator && cfg->process == MFO_EE_MUMU) { g_err = "generator variants apply to processes 1-3"; delete h; return MFO_EINVAL; }
  if (cfg->generator & MFO_GEN_CLASSIC_RAMBO) h->d = 2 + 4 * h->n_final;               // O4': 4n uniforms
  h->masses.assign(h->n_final, 0.0);
  h->sym = 1.0; h->shat_min = 0;
  if (cfg->process != MFO_EE_MUMU) {
    if (!cfg->pdf_xf || cfg->pdf_nx < 2 || cfg->pdf_nq < 2) { g_err = "pdf grid required"; delete h; return MFO_EINVAL; }
    const uint32_t nf = cfg->pdf_nf ? cfg->pdf_nf : 1;
    if (nf != 1 && nf != 11) { g_err = "pdf_nf must be 0, 1 or 11"; delete h; return MFO_EINVAL; }
    if ((cfg->process >= MFO_QQ_TT) != (nf == 11)) { g_err = "processes 4-7 need the 11-flavour grid, processes 1-3 the gluon table"; delete h; return MFO_EINVAL; }
    h->pdf.assign(cfg->pdf_xf, cfg->pdf_xf + (size_t)nf * cfg->pdf_nx * cfg->pdf_nq); h->cfg.pdf_xf = h->pdf.data();
    h->masses[0] = h->masses[1] = cfg->m_top;
    uint32_t ngl = h->n_final - 2;
    double thr = 2.0 * cfg->m_top + ngl * (cfg->ptmin_g > 0 ? cfg->ptmin_g : 0.0);   // O3: shat_min = (sum m + sum pTmin)^2
    h->shat_min = thr * thr;
    if (ngl == 2) h->sym = 0.5;                                                      // A12
    double tau0 = h->shat_min / (cfg->sqrt_s * cfg->sqrt_s);
    if (!(tau0 < 1.0) || tau0 < cfg->pdf_xmin || cfg->mu_f < cfg->pdf_qmin || cfg->mu_f > cfg->pdf_qmax) { g_err = "kinematics outside the PDF grid"; delete h; return MFO_EINVAL; }
  }
  uint32_t nb = cfg->n_bins; h->edges.resize((size_t)h->d * (nb + 1));
  for (uint32_t j = 0; j < h->d; ++j) for (uint32_t k = 0; k <= nb; ++k) h->edges[(size_t)j * (nb + 1) + k] = (double)k / (double)nb;
  h->iteration = 0; h->acc.assign(2 + (size_t)h->d * nb, 0.0);
  *out = h; return MFO_OK;
}
extern "C" int mfo_vegas_destroy(mfo_vegas_t *h) { delete h; return MFO_OK; }
extern "C" int mfo_ndim(const mfo_vegas_t *h, uint32_t *d, uint32_t *nf) { if (!h) return MFO_EINVAL; if (d) *d = h->d; if (nf) *nf = h->n_final; return MFO_OK; }
extern "C" int mfo_get_grid(mfo_vegas_t *h, double *e) { if (!h || !e) return MFO_EINVAL; std::memcpy(e, h->edges.data(), h->edges.size() * sizeof(double)); return MFO_OK; }
extern "C" int mfo_set_grid(mfo_vegas_t *h, const double *e) {
  if (!h || !e) return MFO_EINVAL; uint32_t nb = h->cfg.n_bins;
  for (uint32_t j = 0; j < h->d; ++j) for (uint32_t k = 0; k < nb; ++k) if (!(e[(size_t)j * (nb + 1) + k + 1] > e[(size_t)j * (nb + 1) + k])) { g_err = "edges not increasing"; return MFO_EINVAL; }
  std::memcpy(h->edges.data(), e, h->edges.size() * sizeof(double)); return MFO_OK;
}
extern "C" int mfo_get_accum(mfo_vegas_t *h, double *acc) { if (!h || !acc) return MFO_EINVAL; std::memcpy(acc, h->acc.data(), h->acc.size() * sizeof(double)); return MFO_OK; }

// One event, O1 -> O8.  Returns F = w f (the weight before the 1/N), fills the optional records.
struct EventRec { double x[24]; uint8_t bins[24]; double mom[6 * 4]; double me2; double pdf[2]; int pass; };
static double one_event(const mfo_vegas *h, uint32_t iteration, uint64_t ev, EventRec &R) {
  const mfo_config_t &c = h->cfg; const uint32_t d = h->d, nb = c.n_bins, n = h->n_final;
  double u[24], JV;
  mfo_uniforms(c.seed, iteration, ev, d, u);                              // O1
  mfo_vegas_map(h->edges.data(), d, nb, u, R.x, R.bins, &JV);             // O2
  double s = c.sqrt_s * c.sqrt_s, shat = s, x1 = 1, x2 = 1, Jx = 1;
  const double *rs = R.x;
  if (c.process != MFO_EE_MUMU) {                                         // O3 / O3'
    if (c.generator & MFO_GEN_LINEAR_TAU) mfo_x_map_linear(R.x[0], R.x[1], s, h->shat_min, &x1, &x2, &shat, &Jx);
    else mfo_x_map(R.x[0], R.x[1], s, h->shat_min, &x1, &x2, &shat, &Jx);
    rs = R.x + 2;
  }
  double p0[16], k[16], Mint[4], w3[3];
  if (c.generator & MFO_GEN_CLASSIC_RAMBO) {                              // O4': textbook RAMBO, then O4.4
    mfo_rambo_classic(n, shat, rs, p0);
    w3[0] = mfo_w0(n, shat);
    mfo_massive_rescale(n, shat, h->masses.data(), p0, k, w3 + 1);
  } else {
    mfo_phase_space(n, shat, h->masses.data(), rs, p0, k, Mint, w3);      // O4
  }
  double rts = std::sqrt(shat);
  double *m = R.mom;                                                      // O4.5 incoming momenta
  m[0] = rts / 2; m[1] = 0; m[2] = 0; m[3] = rts / 2; m[4] = rts / 2; m[5] = 0; m[6] = 0; m[7] = -rts / 2;
  std::memcpy(m + 8, k, sizeof(double) * 4 * n);
  R.pass = 1; R.me2 = 0; R.pdf[0] = R.pdf[1] = 0;
  if (c.process == MFO_EE_MUMU) {                                         // O8, config 0
    mfo_me2(c.process, m, 0.0, 0.0, c.alpha_em, &R.me2);
    return JV * R.me2 * (1.0 / (8.0 * M_PI)) * c.gev2_to_pb / (2.0 * s);
  }
  uint32_t ngl = n - 2;
  if (ngl > 0) R.pass = mfo_cuts(ngl, k + 8, x1, x2, c.ptmin_g, c.etamax_g, c.drmin_gg, nullptr);   // O7
  double q2 = c.mu_f * c.mu_f;
  if (c.process == MFO_QQ_TTG || c.process == MFO_QG_TTQ) {               // O5q / O6q with a second quark line and a gluon
    const size_t tab = (size_t)c.pdf_nx * c.pdf_nq;                       // table of PDG id f at index f + 5
    auto xf = [&](int id, double x) { return mfo_pdf_interp(c.pdf_xf + (5 + id) * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x, q2); };
    auto me2_of = [&](int i0, int i1, int i2, int i3) {                   // |M|^2 with the legs (pa, pb, k1, k2) taken from m[i0], m[i1], m[i2], m[i3]
      double mm[20], r;
      std::memcpy(mm, m + 4 * i0, 32); std::memcpy(mm + 4, m + 4 * i1, 32); std::memcpy(mm + 8, m + 4 * i2, 32);
      std::memcpy(mm + 12, m + 4 * i3, 32); std::memcpy(mm + 16, m + 16, 32);
      mfo_me2(c.process, mm, c.m_top, c.alpha_s, c.alpha_em, &r);
      return r;
    };
    long double lum[4] = {0, 0, 0, 0};
    double me[4] = {0, 0, 0, 0};
    int nch;
    if (c.process == MFO_QQ_TTG) {
      nch = 2;
      for (int f = 1; f <= 5; ++f) { lum[0] += (long double)xf(f, x1) * xf(-f, x2); lum[1] += (long double)xf(-f, x1) * xf(f, x2); }
      R.pdf[0] = (double)lum[0]; R.pdf[1] = (double)lum[1];
      if (R.pass) { me[0] = me2_of(0, 1, 2, 3); me[1] = me2_of(1, 0, 2, 3); }            // q along beam 1 / along beam 2
    } else {
      nch = 4;
      const double g1 = xf(0, x1), g2 = xf(0, x2);
      long double q1 = 0, a1 = 0, q2s = 0, a2 = 0;
      for (int f = 1; f <= 5; ++f) { q1 += xf(f, x1); a1 += xf(-f, x1); q2s += xf(f, x2); a2 += xf(-f, x2); }
      lum[0] = q1 * g2; lum[1] = g1 * q2s; lum[2] = a1 * g2; lum[3] = g1 * a2;            // q g, g q, q~ g, g q~
      R.pdf[0] = (double)(lum[0] + lum[2]); R.pdf[1] = (double)(lum[1] + lum[3]);
      if (R.pass) {
        me[0] = me2_of(0, 1, 2, 3); me[1] = me2_of(1, 0, 2, 3);                          // quark along beam 1 / beam 2
        me[2] = me2_of(0, 1, 3, 2); me[3] = me2_of(1, 0, 3, 2);                          // antiquarks: charge conjugation = t <-> t~
      }
    }
    if (!R.pass) return 0.0;
    long double sum = 0, ltot = 0;
    for (int i = 0; i < nch; ++i) { sum += lum[i] * me[i]; ltot += lum[i]; }
    R.me2 = (double)(sum / ltot);
    return JV * Jx * ((double)sum / (x1 * x2)) * h->sym * w3[0] * w3[1] * c.gev2_to_pb / (2.0 * shat);
  }
  if (c.process == MFO_QQ_TT || c.process == MFO_PP_TT) {                 // O5q: flavour-summed luminosity
    const size_t tab = (size_t)c.pdf_nx * c.pdf_nq;                       // table of PDG id f at index f + 5
    long double l12 = 0, l21 = 0;
    for (int f = 1; f <= 5; ++f) {
      double q1 = mfo_pdf_interp(c.pdf_xf + (5 + f) * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x1, q2);
      double a1 = mfo_pdf_interp(c.pdf_xf + (5 - f) * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x1, q2);
      double q2_ = mfo_pdf_interp(c.pdf_xf + (5 + f) * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x2, q2);
      double a2 = mfo_pdf_interp(c.pdf_xf + (5 - f) * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x2, q2);
      l12 += (long double)q1 * a2; l21 += (long double)a1 * q2_;
    }
    if (c.process == MFO_PP_TT) {                                         // both subprocesses in one integrand
      double g1 = mfo_pdf_interp(c.pdf_xf + 5 * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x1, q2);
      double g2 = mfo_pdf_interp(c.pdf_xf + 5 * tab, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x2, q2);
      double mgg, mqq;
      mfo_me2(MFO_GG_TT, m, c.m_top, c.alpha_s, c.alpha_em, &mgg);       // O6
      mfo_me2(MFO_QQ_TT, m, c.m_top, c.alpha_s, c.alpha_em, &mqq);       // O6q
      R.pdf[0] = g1 * g2; R.pdf[1] = (double)(l12 + l21);
      double sum = R.pdf[0] * mgg + R.pdf[1] * mqq;
      R.me2 = sum / (R.pdf[0] + R.pdf[1]);
      return JV * Jx * (sum / (x1 * x2)) * h->sym * w3[0] * w3[1] * c.gev2_to_pb / (2.0 * shat);
    }
    R.pdf[0] = (double)l12; R.pdf[1] = (double)l21;
    mfo_me2(c.process, m, c.m_top, c.alpha_s, c.alpha_em, &R.me2);        // O6q
    return JV * Jx * ((R.pdf[0] + R.pdf[1]) / (x1 * x2)) * R.me2 * h->sym * w3[0] * w3[1] * c.gev2_to_pb / (2.0 * shat);
  }
  R.pdf[0] = mfo_pdf_interp(c.pdf_xf, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x1, q2);   // O5
  R.pdf[1] = mfo_pdf_interp(c.pdf_xf, c.pdf_nx, c.pdf_nq, c.pdf_xmin, c.pdf_xmax, c.pdf_qmin, c.pdf_qmax, x2, q2);
  if (!R.pass) return 0.0;
  mfo_me2(c.process, m, c.m_top, c.alpha_s, c.alpha_em, &R.me2);          // O6
  // O8: F = JV Jx f(x1) f(x2) |M|^2 S_f W0 Wm K / (2 shat),  f(x) = xf/x
  return JV * Jx * (R.pdf[0] / x1) * (R.pdf[1] / x2) * R.me2 * h->sym * w3[0] * w3[1] * c.gev2_to_pb / (2.0 * shat);
}

extern "C" int mfo_integrand_eval(mfo_vegas_t *h, uint32_t iteration, uint64_t first, uint64_t n_events,
                                  const mfo_eval_out_t *out, int n_threads) {
  if (!h || !out) { g_err = "null argument"; return MFO_EINVAL; }
  const uint32_t d = h->d, nl = 2 + h->n_final;
  if (n_threads < 1) n_threads = 1;
  parallel_ranges(n_events, n_threads, [&](int, uint64_t lo, uint64_t hi) {
  for (uint64_t i = lo; i < hi; ++i) {
    EventRec R; double F = one_event(h, iteration, first + (uint64_t)i, R);
    if (!std::isfinite(F)) F = 0.0;
    if (out->weight) out->weight[i] = F;
    if (out->x) std::memcpy(out->x + (size_t)i * d, R.x, sizeof(double) * d);
    if (out->bins) std::memcpy(out->bins + (size_t)i * d, R.bins, d);
    if (out->momenta) std::memcpy(out->momenta + (size_t)i * nl * 4, R.mom, sizeof(double) * nl * 4);
    if (out->me2) out->me2[i] = R.me2;
    if (out->pdf) { out->pdf[2 * i] = R.pdf[0]; out->pdf[2 * i + 1] = R.pdf[1]; }
    if (out->pass) out->pass[i] = (uint8_t)R.pass;
  }
  });
  return MFO_OK;
}

// O9: I = sum t, S2 = sum t^2, H[j][k] = sum_{i in bin k of dim j} t^2, t = F/N; long double sums
extern "C" int mfo_vegas_accumulate(mfo_vegas_t *h, uint32_t iteration, uint64_t first, uint64_t n_events,
                                    uint64_t n_total, int n_threads, double *acc, uint64_t *counts) {
  if (!h || !acc || n_total == 0) { g_err = "bad argument"; return MFO_EINVAL; }
  const uint32_t d = h->d, nb = h->cfg.n_bins; const size_t na = 2 + (size_t)d * nb;
  if (n_threads < 1) n_threads = 1;
  std::vector<std::vector<long double>> part(n_threads, std::vector<long double>(na, 0.0L));
  std::vector<uint64_t> npass(n_threads, 0), nbad(n_threads, 0);
  parallel_ranges(n_events, n_threads, [&](int tid, uint64_t lo, uint64_t hi) {
    std::vector<long double> &a = part[tid];
    for (uint64_t i = lo; i < hi; ++i) {
      EventRec R; double F = one_event(h, iteration, first + i, R);
      if (!std::isfinite(F)) { F = 0.0; nbad[tid]++; }
      if (R.pass) npass[tid]++;
      long double t = (long double)F / (long double)n_total, t2 = t * t;
      a[0] += t; a[1] += t2;
      for (uint32_t j = 0; j < d; ++j) a[2 + (size_t)j * nb + R.bins[j]] += t2;
    }
  });
  for (size_t q = 0; q < na; ++q) { long double s = acc[q]; for (int t = 0; t < n_threads; ++t) s += part[t][q]; acc[q] = (double)s; }
  if (counts) for (int t = 0; t < n_threads; ++t) { counts[0] += npass[t]; counts[1] += nbad[t]; }
  return MFO_OK;
}

// Observable histograms ("histogram accumulation"): the plain definition of mfo.h
static double observable(int kind, const double *k /* final momenta [n][4] */) {
  switch (kind) {
    case MFO_OBS_PT_1: return std::sqrt(k[1] * k[1] + k[2] * k[2]);
    case MFO_OBS_PT_2: return std::sqrt(k[5] * k[5] + k[6] * k[6]);
    case MFO_OBS_PT_3: return std::sqrt(k[9] * k[9] + k[10] * k[10]);
    default: {
      const double E = k[0] + k[4], px = k[1] + k[5], py = k[2] + k[6], pz = k[3] + k[7];
      const double m2 = E * E - px * px - py * py - pz * pz;
      return m2 > 0.0 ? std::sqrt(m2) : 0.0;
    }
  }
}
extern "C" int mfo_observable_hist(mfo_vegas_t *h, uint32_t iteration, uint64_t first, uint64_t n_events,
                                   uint64_t n_total, int n_threads, const mfo_observable_t *obs, uint32_t n_obs,
                                   double *sum, double *sum2) {
  if (!h || !obs || !sum || !sum2 || n_total == 0) { g_err = "bad argument"; return MFO_EINVAL; }
  std::vector<size_t> off(n_obs + 1, 0);
  for (uint32_t o = 0; o < n_obs; ++o) {
    if (obs[o].kind < 0 || obs[o].kind > 3 || obs[o].n_bins < 1 || !(obs[o].hi > obs[o].lo)) { g_err = "bad observable"; return MFO_EINVAL; }
    if (obs[o].kind == MFO_OBS_PT_3 && h->n_final < 3) { g_err = "no third final particle"; return MFO_EINVAL; }
    off[o + 1] = off[o] + obs[o].n_bins + 2;
  }
  if (n_threads < 1) n_threads = 1;
  const size_t tot = off[n_obs];
  std::vector<std::vector<long double>> p1(n_threads, std::vector<long double>(tot, 0.0L)), p2 = p1;
  parallel_ranges(n_events, n_threads, [&](int tid, uint64_t lo, uint64_t hi) {
    for (uint64_t i = lo; i < hi; ++i) {
      EventRec R; double F = one_event(h, iteration, first + i, R);
      if (!std::isfinite(F) || F == 0.0) continue;
      const long double t = (long double)F / (long double)n_total;
      for (uint32_t o = 0; o < n_obs; ++o) {
        const double v = observable(obs[o].kind, R.mom + 8);
        size_t b;
        if (v < obs[o].lo) b = obs[o].n_bins;
        else if (v >= obs[o].hi) b = obs[o].n_bins + 1;
        else { b = (size_t)std::floor((v - obs[o].lo) / (obs[o].hi - obs[o].lo) * obs[o].n_bins); if (b > obs[o].n_bins - 1) b = obs[o].n_bins - 1; }
        p1[tid][off[o] + b] += t; p2[tid][off[o] + b] += t * t;
      }
    }
  });
  for (size_t q = 0; q < tot; ++q) {
    long double a = sum[q], b = sum2[q];
    for (int t = 0; t < n_threads; ++t) { a += p1[t][q]; b += p2[t][q]; }
    sum[q] = (double)a; sum2[q] = (double)b;
  }
  return MFO_OK;
}

// O10: sigma_I^2 = max(0, (N S2 - I^2)/(N-1)); refine every iteration; keep every iteration (A2)
extern "C" int mfo_vegas_finalize(mfo_vegas_t *h, const double *acc, uint64_t n_total, uint64_t n_pass,
                                  uint64_t n_nonfinite, mfo_iter_t *out) {
  if (!h || !acc || n_total < 2) { g_err = "bad argument"; return MFO_EINVAL; }
  const uint32_t d = h->d, nb = h->cfg.n_bins;
  std::memcpy(h->acc.data(), acc, h->acc.size() * sizeof(double));
  long double I = acc[0], S2 = acc[1], N = (long double)n_total;
  long double var = (N * S2 - I * I) / (N - 1.0L); if (var < 0) var = 0;
  h->I.push_back((double)I); h->sig.push_back((double)sqrtl(var));
  std::vector<double> ne(h->edges.size());
  mfo_refine(h->edges.data(), acc + 2, d, nb, h->cfg.alpha_damp, ne.data());
  h->edges = ne; h->iteration++;
  if (out) { out->integral = (double)I; out->sigma = (double)sqrtl(var); out->n_events = n_total; out->n_pass = n_pass; out->n_nonfinite = n_nonfinite; }
  return MFO_OK;
}

extern "C" int mfo_vegas_iterate(mfo_vegas_t *h, uint64_t n_events, int n_threads, mfo_iter_t *out) {
  if (!h) return MFO_EINVAL;
  std::vector<double> acc(h->acc.size(), 0.0); uint64_t counts[2] = {0, 0};
  int rc = mfo_vegas_accumulate(h, h->iteration, 0, n_events, n_events, n_threads, acc.data(), counts);
  if (rc) return rc;
  return mfo_vegas_finalize(h, acc.data(), n_events, counts[0], counts[1], out);
}

extern "C" int mfo_result(mfo_vegas_t *h, mfo_result_t *out) {
  if (!h || !out) return MFO_EINVAL;
  if (h->I.empty()) { g_err = "no iteration yet"; return MFO_ESTATE; }
  mfo_combine(h->I.data(), h->sig.data(), (uint32_t)h->I.size(), out); return MFO_OK;
}
