// mfo_core.cpp -- ORACLE (test infrastructure, not the product): RNG, VEGAS map/refinement,
// parton fractions, phase space, PDF interpolation, cuts.  Plain fp64 C++, one function per step,
// each citing the passage / DESIGN.md reading it follows.  Shares nothing with the CUDA path.
#include "mfo.h"
#include <cmath>
#include <cstring>
#include <vector>
#include <algorithm>

// ------------------------------------------------------------------------------------------------
// O1  Random numbers ("generation of random numbers"; reading A1)
// Philox4x32-10, Salmon et al. SC'11.  Pinned by the three known-answer vectors (tests/golden).
// ------------------------------------------------------------------------------------------------
extern "C" void mfo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  const uint32_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u, W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3], k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) { k0 += W0; k1 += W1; }
    uint64_t p0 = (uint64_t)M0 * c0, p1 = (uint64_t)M1 * c2;
    uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    uint32_t n0 = hi1 ^ c1 ^ k0, n1 = lo1, n2 = hi0 ^ c3 ^ k1, n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// key = (seed lo, seed hi); counter = (event lo, event hi, block j, iteration); block j gives
// dimensions 2j (from words o1:o0) and 2j+1 (from o3:o2); u = ((X >> 12) + 0.5) * 2^-52  (A1).
extern "C" void mfo_uniforms(uint64_t seed, uint32_t iteration, uint64_t event, uint32_t d,
                             double *u) {
  uint32_t key[2] = {(uint32_t)seed, (uint32_t)(seed >> 32)};
  for (uint32_t j = 0; 2 * j < d; ++j) {
    uint32_t ctr[4] = {(uint32_t)event, (uint32_t)(event >> 32), j, iteration}, o[4];
    mfo_philox4x32_10(ctr, key, o);
    uint64_t X0 = ((uint64_t)o[1] << 32) | o[0], X1 = ((uint64_t)o[3] << 32) | o[2];
    u[2 * j] = ((double)(X0 >> 12) + 0.5) * 0x1p-52;
    if (2 * j + 1 < d) u[2 * j + 1] = ((double)(X1 >> 12) + 0.5) * 0x1p-52;
  }
}

// ------------------------------------------------------------------------------------------------
// O2  VEGAS map (Lepage's VEGAS as used by VegasFlow, ref [8] PAPER.md:110; A2)
// t = u*Nb; k = min(floor t, Nb-1); y = e_k + (t-k)(e_{k+1}-e_k); J = prod Nb (e_{k+1}-e_k)
// ------------------------------------------------------------------------------------------------
extern "C" void mfo_vegas_map(const double *edges, uint32_t d, uint32_t nb, const double *u,
                              double *x, uint8_t *bins, double *jac) {
  double J = 1.0;
  for (uint32_t j = 0; j < d; ++j) {
    const double *e = edges + (size_t)j * (nb + 1);
    double t = u[j] * (double)nb;
    uint32_t k = (uint32_t)std::floor(t);
    if (k > nb - 1) k = nb - 1;
    double delta = e[k + 1] - e[k];
    x[j] = e[k] + (t - (double)k) * delta;
    bins[j] = (uint8_t)k;
    J *= (double)nb * delta;
  }
  *jac = J;
}

// ------------------------------------------------------------------------------------------------
// O10  Grid refinement (Lepage's classic VEGAS; A2, A3): smooth, normalise, compress with
// r = ((s-1)/ln s)^alpha, re-bin so that every new bin holds the same share of sum r.
// ------------------------------------------------------------------------------------------------
extern "C" void mfo_refine(const double *edges_in, const double *H, uint32_t d, uint32_t nb,
                           double alpha, double *edges_out) {
  for (uint32_t j = 0; j < d; ++j) {
    const double *e = edges_in + (size_t)j * (nb + 1);
    const double *h = H + (size_t)j * nb;
    double *eo = edges_out + (size_t)j * (nb + 1);
    std::vector<double> s(nb), r(nb);
    // 1. smooth
    for (uint32_t k = 0; k < nb; ++k) {
      if (nb == 1) s[k] = h[k];
      else if (k == 0) s[k] = (h[0] + h[1]) / 2.0;
      else if (k == nb - 1) s[k] = (h[nb - 2] + h[nb - 1]) / 2.0;
      else s[k] = (h[k - 1] + h[k] + h[k + 1]) / 3.0;
    }
    // 2. normalise
    long double tot = 0.0L;
    for (uint32_t k = 0; k < nb; ++k) tot += s[k];
    if (!(tot > 0.0L)) { std::memcpy(eo, e, sizeof(double) * (nb + 1)); continue; }
    for (uint32_t k = 0; k < nb; ++k) { s[k] = (double)(s[k] / tot); if (s[k] < 1e-30) s[k] = 1e-30; }
    // 3. compress
    long double rtot = 0.0L;
    for (uint32_t k = 0; k < nb; ++k) {
      r[k] = (s[k] == 1.0) ? 1.0 : std::pow((s[k] - 1.0) / std::log(s[k]), alpha);
      rtot += r[k];
    }
    // 4. re-bin: C(e_k) = sum_{l<k} r_l / rtot piecewise linear on the old edges; e'_m = C^-1(m/Nb)
    eo[0] = 0.0; eo[nb] = 1.0;
    long double cum = 0.0L;   // sum_{l<k} r_l
    uint32_t k = 0;
    for (uint32_t m = 1; m < nb; ++m) {
      long double target = rtot * (long double)m / (long double)nb;
      while (k < nb - 1 && cum + r[k] < target) { cum += r[k]; ++k; }
      long double frac = (target - cum) / r[k];
      if (frac < 0.0L) frac = 0.0L;
      if (frac > 1.0L) frac = 1.0L;
      eo[m] = (double)(e[k] + frac * ((long double)e[k + 1] - e[k]));
    }
  }
}

// ------------------------------------------------------------------------------------------------
// O11  Combination over iterations (inverse-variance weighted mean; VegasFlow / Lepage)
// ------------------------------------------------------------------------------------------------
extern "C" void mfo_combine(const double *I, const double *sig, uint32_t n, mfo_result_t *out) {
  out->n_iter = n; out->integral = 0; out->sigma = 0; out->chi2_dof = 0;
  if (n == 0) return;
  bool any_zero = false;
  for (uint32_t j = 0; j < n; ++j) if (!(sig[j] > 0.0)) any_zero = true;
  if (any_zero) {
    long double m = 0; for (uint32_t j = 0; j < n; ++j) m += I[j];
    out->integral = (double)(m / n);
    long double v = 0; for (uint32_t j = 0; j < n; ++j) v += (long double)sig[j] * sig[j];
    out->sigma = (double)(sqrtl(v) / n);
    return;
  }
  long double sw = 0, swi = 0;
  for (uint32_t j = 0; j < n; ++j) { long double w = 1.0L / ((long double)sig[j] * sig[j]); sw += w; swi += w * I[j]; }
  long double mean = swi / sw;
  out->integral = (double)mean;
  out->sigma = (double)(1.0L / sqrtl(sw));
  if (n > 1) {
    long double c = 0;
    for (uint32_t j = 0; j < n; ++j) { long double dlt = I[j] - mean; c += dlt * dlt / ((long double)sig[j] * sig[j]); }
    out->chi2_dof = (double)(c / (n - 1));
  }
}

// ------------------------------------------------------------------------------------------------
// O3  Parton momentum fractions (paper silent, reading A4):
// tau = tau0^(1-y0), x1 = tau^y1, x2 = tau/x1, shat = tau s, Jx = tau (-ln tau0)(-ln tau)
// ------------------------------------------------------------------------------------------------
extern "C" void mfo_x_map(double y0, double y1, double s, double shat_min, double *x1, double *x2,
                          double *shat, double *jx) {
  double tau0 = shat_min / s;
  double ltau0 = std::log(tau0);
  double ltau = (1.0 - y0) * ltau0;
  double tau = std::exp(ltau);
  *x1 = std::exp(y1 * ltau);
  *x2 = tau / *x1;
  *shat = tau * s;
  *jx = tau * (-ltau0) * (-ltau);
}

// O3': tau linear in y0; x1 = tau^y1 as in O3, so dx1 dx2 = (1 - tau0)(-ln tau) dy0 dy1
extern "C" void mfo_x_map_linear(double y0, double y1, double s, double shat_min, double *x1, double *x2,
                                 double *shat, double *jx) {
  double tau0 = shat_min / s;
  double tau = tau0 + (1.0 - tau0) * y0;
  double ltau = std::log(tau);
  *x1 = std::exp(y1 * ltau);
  *x2 = tau / *x1;
  *shat = tau * s;
  *jx = (1.0 - tau0) * (-ltau);
}

// ------------------------------------------------------------------------------------------------
// O4  Phase space (reading A5: 3n-4-random sequential-decay RAMBO with the
// standard RAMBO massive rescaling; A6 particle order = generation order; A7 Newton)
// ------------------------------------------------------------------------------------------------
static double factorial(uint32_t n) { double f = 1; for (uint32_t i = 2; i <= n; ++i) f *= i; return f; }

// W0(n, shat) = (pi/2)^(n-1) shat^(n-2) / ((n-1)!(n-2)!) * (2 pi)^(4-3n)
extern "C" double mfo_w0(uint32_t n, double shat) {
  return std::pow(M_PI / 2.0, (double)n - 1.0) * std::pow(shat, (double)n - 2.0) /
         (factorial(n - 1) * factorial(n - 2)) * std::pow(2.0 * M_PI, 4.0 - 3.0 * (double)n);
}

// solve r = (k+1) u^(2k) - k u^(2k+2) for u in (0,1), k = n-i >= 1.  The left side rises
// monotonically from 0 to 1, so plain bisection (to the last bit) is used: no closed form here.
static double solve_mass_fraction(uint32_t k, double r) {
  auto f = [k](double u) { return (k + 1.0) * std::pow(u, 2.0 * k) - k * std::pow(u, 2.0 * k + 2.0); };
  double lo = 0.0, hi = 1.0;
  for (int it = 0; it < 200; ++it) {
    double mid = 0.5 * (lo + hi);
    if (mid == lo || mid == hi) break;
    if (f(mid) < r) lo = mid; else hi = mid;
  }
  double u = 0.5 * (lo + hi);
  // a few Newton steps on the polynomial to remove the residual left by evaluating f in fp64
  for (int it = 0; it < 3; ++it) {
    double fp = 2.0 * k * (k + 1.0) * (std::pow(u, 2.0 * k - 1.0) - std::pow(u, 2.0 * k + 1.0));
    if (fp > 0) { double un = u - (f(u) - r) / fp; if (un > 0.0 && un < 1.0) u = un; }
  }
  return u;
}

// boost p from the rest frame of Q (mass M known analytically) to the frame where Q is given
static void boost_from_rest(const double Q[4], double M, const double p[4], double out[4]) {
  double Ep = (Q[0] * p[0] + Q[1] * p[1] + Q[2] * p[2] + Q[3] * p[3]) / M;
  double f = (p[0] + Ep) / (Q[0] + M);
  out[0] = Ep; out[1] = p[1] + Q[1] * f; out[2] = p[2] + Q[2] * f; out[3] = p[3] + Q[3] * f;
}

extern "C" int mfo_massive_rescale(uint32_t n, double shat, const double *masses, const double *p0, double *kk,
                                   double *out2) {
  double rts = std::sqrt(shat);
  // massive rescaling (O4.4): sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt(shat), Newton from
  //    xi0 = sqrt(1 - (sum m / sqrt shat)^2), stop |dxi| <= 1e-14 xi, cap 50 (A7)
  double summ = 0; bool massless = true;
  for (uint32_t i = 0; i < n; ++i) { summ += masses[i]; if (masses[i] != 0.0) massless = false; }
  double xi = 1.0; int steps = 0;
  if (!massless) {
    xi = std::sqrt(1.0 - (summ / rts) * (summ / rts));
    for (steps = 0; steps < 50;) {
      long double F = -(long double)rts, dF = 0;
      for (uint32_t i = 0; i < n; ++i) {
        double e0 = p0[4 * i];
        double E = std::sqrt(masses[i] * masses[i] + xi * xi * e0 * e0);
        F += E; dF += (long double)xi * e0 * e0 / E;
      }
      double dxi = (double)(F / dF);
      xi -= dxi; ++steps;
      if (std::fabs(dxi) <= 1e-14 * xi) break;
    }
  }
  double prod = 1.0, den = 0.0;
  for (uint32_t i = 0; i < n; ++i) {
    double e0 = p0[4 * i];
    double kabs = xi * e0;
    double E = std::sqrt(masses[i] * masses[i] + kabs * kabs);
    kk[4 * i] = E; kk[4 * i + 1] = xi * p0[4 * i + 1]; kk[4 * i + 2] = xi * p0[4 * i + 2]; kk[4 * i + 3] = xi * p0[4 * i + 3];
    prod *= kabs / E; den += kabs * kabs / E;
  }
  double Wm = massless ? 1.0 : std::pow(xi, 2.0 * n - 3.0) * prod * rts / den;
  out2[0] = Wm; out2[1] = xi;
  return steps;
}

// O4': textbook RAMBO (Kleiss, Stirling, Ellis 1986), the steps in the order of mfo.h
extern "C" void mfo_rambo_classic(uint32_t n, double shat, const double *rs, double *p0) {
  double rts = std::sqrt(shat);
  std::vector<double> q(4 * (size_t)n);
  double Q[4] = {0, 0, 0, 0};
  for (uint32_t i = 0; i < n; ++i) {
    double c = 2.0 * rs[4 * i] - 1.0, phi = 2.0 * M_PI * rs[4 * i + 1];
    double q0 = -std::log(rs[4 * i + 2] * rs[4 * i + 3]);
    double st = std::sqrt(1.0 - c * c);
    q[4 * i] = q0; q[4 * i + 1] = q0 * st * std::cos(phi); q[4 * i + 2] = q0 * st * std::sin(phi); q[4 * i + 3] = q0 * c;
    for (int m = 0; m < 4; ++m) Q[m] += q[4 * i + m];
  }
  double M = std::sqrt(Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3]);
  double b[3] = {-Q[1] / M, -Q[2] / M, -Q[3] / M};
  double x = rts / M, gam = Q[0] / M, a = 1.0 / (1.0 + gam);
  for (uint32_t i = 0; i < n; ++i) {
    const double *qi = &q[4 * i];
    double bq = b[0] * qi[1] + b[1] * qi[2] + b[2] * qi[3];
    p0[4 * i] = x * (gam * qi[0] + bq);
    for (int m = 0; m < 3; ++m) p0[4 * i + 1 + m] = x * (qi[1 + m] + b[m] * qi[0] + a * bq * b[m]);
  }
}

extern "C" int mfo_phase_space(uint32_t n, double shat, const double *masses, const double *rs,
                               double *p0, double *kk, double *Mint, double *out3) {
  double rts = std::sqrt(shat);
  std::vector<double> M(n + 1);
  // 1. intermediate masses M_1 = sqrt(shat), M_n = 0, M_i = u_i M_{i-1} (i = 2..n-1), rs[i-2]
  M[1] = rts; M[n] = 0.0;
  for (uint32_t i = 2; i + 1 <= n; ++i) M[i] = solve_mass_fraction(n - i, rs[i - 2]) * M[i - 1];
  for (uint32_t i = 1; i <= n; ++i) Mint[i - 1] = M[i];
  // 2. sequential two-body decays Q_{i-1} -> p_{i-1} + Q_i, i = 2..n
  double Q[4] = {rts, 0, 0, 0};
  for (uint32_t i = 2; i <= n; ++i) {
    double ct = 2.0 * rs[n - 6 + 2 * i] - 1.0;
    double phi = 2.0 * M_PI * rs[n - 5 + 2 * i];
    double st = std::sqrt(1.0 - ct * ct);
    double q = (M[i - 1] * M[i - 1] - M[i] * M[i]) / (2.0 * M[i - 1]);
    double p_rest[4] = {q, q * st * std::cos(phi), q * st * std::sin(phi), q * ct};
    double Q_rest[4] = {std::sqrt(q * q + M[i] * M[i]), -p_rest[1], -p_rest[2], -p_rest[3]};
    double p_cm[4], Q_cm[4];
    if (i == 2) { std::memcpy(p_cm, p_rest, sizeof p_cm); std::memcpy(Q_cm, Q_rest, sizeof Q_cm); }
    else { boost_from_rest(Q, M[i - 1], p_rest, p_cm); boost_from_rest(Q, M[i - 1], Q_rest, Q_cm); }
    std::memcpy(p0 + 4 * (i - 2), p_cm, sizeof p_cm);
    std::memcpy(Q, Q_cm, sizeof Q);
  }
  std::memcpy(p0 + 4 * (n - 1), Q, sizeof Q);
  // 3. massless weight, 4. massive rescaling
  double o2[2];
  int steps = mfo_massive_rescale(n, shat, masses, p0, kk, o2);
  out3[0] = mfo_w0(n, shat); out3[1] = o2[0]; out3[2] = o2[1];
  return steps;
}

// ------------------------------------------------------------------------------------------------
// O5  Parton densities (readings A9, A10): cubic Hermite in (ln x, ln Q^2) on the
// tabulated values xf, node slope = mean of the two secants (one-sided at the ends).
// ------------------------------------------------------------------------------------------------
// Hermite interpolation on uniform knots z_i = z0 + i h through values f[0..n-1] (stride st),
// in cell i (0 <= i <= n-2) at local coordinate t in [0,1].
static double hermite_cell(const double *f, size_t st, uint32_t n, uint32_t i, double h, double t) {
  auto F = [&](uint32_t k) { return f[(size_t)k * st]; };
  auto slope = [&](uint32_t k) {
    if (k == 0) return (F(1) - F(0)) / h;
    if (k == n - 1) return (F(n - 1) - F(n - 2)) / h;
    return 0.5 * ((F(k + 1) - F(k)) / h + (F(k) - F(k - 1)) / h);
  };
  double t2 = t * t, t3 = t2 * t;
  return (2 * t3 - 3 * t2 + 1) * F(i) + (t3 - 2 * t2 + t) * h * slope(i) +
         (-2 * t3 + 3 * t2) * F(i + 1) + (t3 - t2) * h * slope(i + 1);
}

extern "C" double mfo_pdf_interp(const double *xf, uint32_t nx, uint32_t nq, double xmin, double xmax,
                                 double qmin, double qmax, double x, double q2) {
  double lx0 = std::log(xmin), hx = (std::log(xmax) - lx0) / (nx - 1);
  double lq0 = std::log(qmin * qmin), hq = (std::log(qmax * qmax) - lq0) / (nq - 1);
  double lx = std::log(x), lq = std::log(q2);
  double fx = (lx - lx0) / hx, fq = (lq - lq0) / hq;
  int ix = (int)std::floor(fx), iq = (int)std::floor(fq);
  ix = std::min(std::max(ix, 0), (int)nx - 2);
  iq = std::min(std::max(iq, 0), (int)nq - 2);
  double tx = fx - ix, tq = fq - iq;
  tx = std::min(std::max(tx, 0.0), 1.0);       // clamp at run time: no extrapolation (O5)
  tq = std::min(std::max(tq, 0.0), 1.0);
  // interpolate along ln x at every Q^2 row (the two-step rule only reads rows iq-1..iq+2, but
  // computing the whole column of row values and then applying the same 1-D rule is the plainest
  // statement of it)
  std::vector<double> row(nq);
  for (uint32_t q = 0; q < nq; ++q) row[q] = hermite_cell(xf + q, nq, nx, (uint32_t)ix, hx, tx);
  return hermite_cell(row.data(), 1, nq, (uint32_t)iq, hq, tq);
}

// ------------------------------------------------------------------------------------------------
// O7  Cuts ("apply any fiducial cuts"; reading A8): final gluons only, lab frame.
// eta_lab = atanh(kz/|k|) + y_b, y_b = ln(x1/x2)/2; pT invariant; dR from eta and wrapped dphi.
// ------------------------------------------------------------------------------------------------
extern "C" int mfo_cuts(uint32_t ng, const double *kg, double x1, double x2, double ptmin,
                        double etamax, double drmin, double *obs) {
  double yb = 0.5 * std::log(x1 / x2);
  int pass = 1;
  std::vector<double> eta(ng), phi(ng);
  for (uint32_t i = 0; i < ng; ++i) {
    const double *k = kg + 4 * i;
    double pt = std::sqrt(k[1] * k[1] + k[2] * k[2]);
    double kabs = std::sqrt(k[1] * k[1] + k[2] * k[2] + k[3] * k[3]);
    eta[i] = std::atanh(k[3] / kabs) + yb;
    phi[i] = std::atan2(k[2], k[1]);
    if (obs) { obs[2 * i] = pt; obs[2 * i + 1] = eta[i]; }
    if (ptmin > 0 && !(pt > ptmin)) pass = 0;
    if (etamax > 0 && !(std::fabs(eta[i]) < etamax)) pass = 0;
  }
  double drm = 1e300;
  for (uint32_t i = 0; i < ng; ++i)
    for (uint32_t j = i + 1; j < ng; ++j) {
      double dphi = phi[i] - phi[j];
      while (dphi > M_PI) dphi -= 2.0 * M_PI;
      while (dphi <= -M_PI) dphi += 2.0 * M_PI;
      double deta = eta[i] - eta[j];
      double dr = std::sqrt(deta * deta + dphi * dphi);
      drm = std::min(drm, dr);
      if (drmin > 0 && !(dr > drmin)) pass = 0;
    }
  if (obs) obs[2 * ng] = (ng >= 2) ? drm : 0.0;
  return pass;
}
