// mf_device.cuh -- per-event device functions of the LO integrand path, steps S1-S8
// ("generation of random numbers, computation of the phase space kinematics, matrix
// element evaluation and histogram accumulation"; PAPER.md:29 PDF interpolation, phase space with
// fiducial cuts, matrix element).  The paper prints no formulas: each function states the DESIGN.md
// reading (O1-O8) it implements.  One event per thread, everything in registers; the VEGAS edges
// and the PDF table are read from shared memory.
//
// Functions are marked MF_HD so that tests/ can compile this very file for the host with g++ and
// check the per-event arithmetic against the oracle without a GPU (test harness only: the product
// library has no CPU path).
#pragma once
#include <stdint.h>
#include <math.h>

#if defined(__CUDACC__)
#define MF_HD __device__ __forceinline__
#define MF_DEVFN __device__ __forceinline__
#else
#define MF_HD static inline
#define MF_DEVFN static inline
static inline void sincospi(double x, double* s, double* c) { *s = sin(M_PI * x); *c = cos(M_PI * x); }
static inline double rsqrt(double x) { return 1.0 / sqrt(x); }
static inline float rsqrt(float x) { return 1.0f / sqrtf(x); }
#endif

// Barrier points inside the generated helicity-loop bodies (one every 64 statements): with
// MF_SYNC_EVERY = k > 0 every k-th point is a __syncthreads(), which keeps the warps of a block within
// a few hundred instructions of each other so that they share instruction-cache lines (the straight-
// line body is larger than the 32 KB L1.5 I-cache).  Requires the |M|^2 code to be executed by every
// thread of the block (MF_UNIFORM_ME), which costs nothing: a warp runs it whenever one lane passes.
#ifndef MF_SYNC_EVERY
#define MF_SYNC_EVERY 16
#endif
#define MF_GROUP_THREADS 128
#if defined(__CUDA_ARCH__)
// barrier points of the generated |M|^2 code: the warps of one 128-thread GROUP (one warp per SM
// sub-partition) stay on the same instruction-cache lines; the two groups of a 256-thread CTA use
// their own named barrier so that they can run out of phase (mf_me_kernel staggers them: while one
// group is in its per-event prologue the other keeps the FP64 pipe busy).
#define MF_GROUP_SYNC() asm volatile("bar.sync %0, 128;" :: "r"(1 + (int)(threadIdx.x >> 7)) : "memory")
#define MF_SYNC_POINT(i) do { if (MF_SYNC_EVERY > 0 && (i) % (MF_SYNC_EVERY > 0 ? MF_SYNC_EVERY : 1) == 0) MF_GROUP_SYNC(); } while (0)
// whole-CTA barrier points (tuning hook, gen/amplitudes.py SYNC_MACRO): gg -> tt~gg used them while its helicity loop ran over
// three gluons (0.5 MB of SASS per trip: one instruction stream per SM); with all four gluons in the loop the body halves and the
// 128-thread groups of MF_SYNC_POINT are faster (profiles/r1_tuning.md)
#ifndef MF_SYNC_EVERY_WIDE
#define MF_SYNC_EVERY_WIDE 4
#endif
#define MF_SYNC_POINT_W(i) do { if ((i) % MF_SYNC_EVERY_WIDE == 0) __syncthreads(); } while (0)
#else
#define MF_SYNC_POINT(i) do { } while (0)
#define MF_SYNC_POINT_W(i) do { } while (0)
#endif
// opaque identity on a double: stops the compiler from hoisting what is computed from it out of the
// helicity loop (the generator decides what is hoisted: gen/dag.py Dag.plan)
#if defined(__CUDA_ARCH__)
__device__ __forceinline__ void mf_launder(double& x) { asm volatile("" : "+d"(x)); }
__device__ __forceinline__ void mf_launder(float& x) { asm volatile("" : "+f"(x)); }
#define MF_LAUNDER(x) mf_launder(x)
#else
#define MF_LAUNDER(x) do { } while (0)
#endif
#ifndef MF_UNIFORM_ME
#define MF_UNIFORM_ME (MF_SYNC_EVERY > 0)
#endif

#ifndef MF_NEWTON_STEPS
#define MF_NEWTON_STEPS 4   // massive-RAMBO Newton steps (reading A7)
#endif
#define MF_DMAX 18          // VEGAS dimensions of the largest process (gg -> tt~gg) with the classic 4n-random RAMBO
#define MFD_GEN_CLASSIC 1   // generator flags (include/madflow_b200.h MF_GEN_*)
#define MFD_GEN_LINEAR 2
#define MF_NBMAX 64         // bins per dimension
#define MF_PI 3.14159265358979323846

// run constants of one handle (kernel parameter)
struct MfParams {
  int32_t process, d, n_final, nb;
  int32_t gen;                          // MF_GEN_* flags: selectable generators; 0 = the configs' generators
  uint32_t key0, key1;                  // Philox key = (seed lo, seed hi)        (A1)
  double s, ltau0, m_top;               // collider s, ln(shat_min / s)            (O3)
  double tau0;                          // shat_min / s (linear-tau variant O3')
  double me_pref;                       // g_s^(2 ng) / 256 * generator scale, or e^4/4 (O6)
  double me_pref_qq;                    // g_s^4 (2/9) / 4: q q~ -> t t~ (O6q; processes 4 and 5)
  double ptmin, etamax, drmin;          // cuts (O7)
  double tanh_etamax;                   // tanh(etamax): the eta cut is taken on tanh (mf_cuts)
  int32_t n_obs, obs_kind[4], obs_nb[4];  // observable histograms (include/madflow_b200.h mf_set_observables)
  double obs_lo[4], obs_hi[4];
  double wconst;                        // S_f * K / 2  (O8: F = ... S_f W_PS K / (2 shat))
  double pdf_lx0, pdf_ihx, pdf_lq0, pdf_ihq, pdf_lq;   // ln xmin, 1/h_x, ln qmin^2, 1/h_q, ln muF^2
  int32_t pdf_nx, pdf_nq;
  int32_t pdf_smem;                     // doubles of the PDF table staged in shared memory: nx*nq (gluon table), or
                                        // nx*(pdf_nqs*MF_NFL + MF_XPAD) for the flavour grid of the quark channels
  int32_t pdf_iq0, pdf_nqs;             // flavour grid: first Q^2 row and number of rows kept (<= 4): mu_F is a run constant, so
                                        // only the rows its stencil touches are staged (32 KB instead of 400 KB); the
                                        // interpolation in Q^2 is still evaluated per event (A17)
};
#define MF_XPAD 1                       // padding doubles per ln-x row of the staged flavour grid (bank spread)
#define MF_NFL 11                       // tables of the flavour grid, device layout [nx][pdf_nqs * MF_NFL + MF_XPAD], slot =
                                        // PDG id + 5: 5 - q = antiquark, 5 = gluon, 5 + q = quark of flavour q = 1..5 (d u s c b)

// ---- S1: Philox4x32-10 (Salmon et al. SC'11), reading O1/A1 ----------------------------------
MF_HD uint32_t mf_mulhi32(uint32_t a, uint32_t b) {
#if defined(__CUDA_ARCH__)
  return __umulhi(a, b);
#else
  return (uint32_t)(((uint64_t)a * b) >> 32);
#endif
}

MF_HD void mf_philox(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0, uint32_t k1,
                     uint32_t o[4]) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const uint32_t h0 = mf_mulhi32(0xD2511F53u, c0), l0 = 0xD2511F53u * c0;
    const uint32_t h1 = mf_mulhi32(0xCD9E8D57u, c2), l1 = 0xCD9E8D57u * c2;
    c0 = h1 ^ c1 ^ k0; c1 = l1; c2 = h0 ^ c3 ^ k1; c3 = l0;
    k0 += 0x9E3779B9u; k1 += 0xBB67AE85u;
  }
  o[0] = c0; o[1] = c1; o[2] = c2; o[3] = c3;
}

// 52-bit uniform in (0,1): u = ((X >> 12) + 0.5) 2^-52, exact in fp64 (A1)
MF_HD double mf_u52(uint32_t lo, uint32_t hi) {
  const uint64_t X = ((uint64_t)hi << 32) | lo;
  return ((double)(X >> 12) + 0.5) * 0x1p-52;
}

// d uniforms of event `ev`: counter = (ev lo, ev hi, block j, iteration); block j -> dims 2j, 2j+1
template <int D>
MF_HD void mf_uniforms(const MfParams& P, uint32_t iteration, uint64_t ev, double u[D]) {
#pragma unroll
  for (int j = 0; 2 * j < D; ++j) {
    uint32_t o[4];
    mf_philox((uint32_t)ev, (uint32_t)(ev >> 32), (uint32_t)j, iteration, P.key0, P.key1, o);
    u[2 * j] = mf_u52(o[0], o[1]);
    if (2 * j + 1 < D) u[2 * j + 1] = mf_u52(o[2], o[3]);
  }
}

// ---- S2: VEGAS map (O2): k = min(floor(u nb), nb-1); y = e_k + (u nb - k) D_k; J = prod nb D_k --
template <int D>
MF_HD double mf_vegas_map(const double* edges, int nb, const double u[D], double y[D], int bin[D]) {
  double J = 1.0;
  const double dnb = (double)nb;
#pragma unroll
  for (int j = 0; j < D; ++j) {
    const double* e = edges + j * (nb + 1);
    const double t = u[j] * dnb;
    int k = (int)t;
    k = k > nb - 1 ? nb - 1 : k;
    const double e0 = e[k], delta = e[k + 1] - e0;
    y[j] = e0 + (t - (double)k) * delta;
    bin[j] = k;
    J *= dnb * delta;
  }
  return J;
}

// ---- S3: parton fractions (O3): tau = tau0^(1-y0), x1 = tau^y1, x2 = tau/x1 -------------------
// lx1, lx2 = ln x1, ln x2 are exact by construction (no log needed downstream: PDF lookup, boost)
MF_HD void mf_x_map(const MfParams& P, double y0, double y1, double& x1, double& x2, double& shat,
                    double& jx, double& lx1, double& lx2) {
  const double ltau = (1.0 - y0) * P.ltau0;
  const double tau = exp(ltau);
  lx1 = y1 * ltau; lx2 = ltau - lx1;
  x1 = exp(lx1);
  x2 = tau / x1;
  shat = tau * P.s;
  jx = tau * P.ltau0 * ltau;            // tau (-ln tau0)(-ln tau)
}

// O3' (MF_GEN_LINEAR_TAU): tau = tau0 + (1 - tau0) y0, x1 = tau^y1 as in O3, so
// dx1 dx2 = (1 - tau0)(-ln tau) dy0 dy1
MF_HD void mf_x_map_linear(const MfParams& P, double y0, double y1, double& x1, double& x2, double& shat,
                           double& jx, double& lx1, double& lx2) {
  const double tau = fma(1.0 - P.tau0, y0, P.tau0);
  const double ltau = log(tau);
  lx1 = y1 * ltau; lx2 = ltau - lx1;
  x1 = exp(lx1);
  x2 = tau / x1;
  shat = tau * P.s;
  jx = (1.0 - P.tau0) * (-ltau);
}

// ---- S4: phase space (O4): 3n-4-random sequential-decay RAMBO + massive rescaling ---------------
// mass fraction: solve r = (k+1) w^k - k w^(k+1) for w = u^2 in (0,1), k = n - i (closed form, then
// two Newton steps on the polynomial so that the root does not depend on acos/cos rounding)
MF_HD double mf_mass_fraction_sq(int k, double r) {
  double w;
  if (k == 1) {                                   // 2w - w^2 = r
    w = r / (1.0 + sqrt(1.0 - r));
#pragma unroll
    for (int it = 0; it < 2; ++it) w -= (w * (2.0 - w) - r) / (2.0 * (1.0 - w));
  } else {                                        // 3w^2 - 2w^3 = r,  w = 1/2 + cos((2pi - acos(1-2r))/3)
    w = 0.5 + cos((2.0 * MF_PI - acos(1.0 - 2.0 * r)) * (1.0 / 3.0));
#pragma unroll
    for (int it = 0; it < 2; ++it) w -= (w * w * (3.0 - 2.0 * w) - r) / (6.0 * w * (1.0 - w));
  }
  return w;
}

// boost p from the rest frame of Q (mass M known analytically) to the frame in which Q is given
// (iM = 1/M and iQM = 1/(Q0 + M) are passed in: the two boosts of one decay step share them)
MF_HD void mf_boost(const double Q[4], double iM, double iQM, const double p[4], double out[4]) {
  const double Ep = (Q[0] * p[0] + Q[1] * p[1] + Q[2] * p[2] + Q[3] * p[3]) * iM;
  const double f = (p[0] + Ep) * iQM;
  out[0] = Ep; out[1] = p[1] + Q[1] * f; out[2] = p[2] + Q[2] * f; out[3] = p[3] + Q[3] * f;
}

// W0(n, shat) = (pi/2)^(n-1) shat^(n-2) / ((n-1)!(n-2)!) (2pi)^(4-3n)
template <int N>
MF_HD double mf_w0(double shat) {
  if (N == 2) return 1.0 / (8.0 * MF_PI);
  if (N == 3) return shat / (256.0 * MF_PI * MF_PI * MF_PI);
  return shat * shat / (24576.0 * MF_PI * MF_PI * MF_PI * MF_PI * MF_PI);
}

// O4.4: RAMBO's massive rescaling of massless CM momenta k[N][4] (in place); masses m for particles 0,1, 0 for
// the rest (m > 0).  Returns W_m.
template <int N>
MF_HD double mf_massive_rescale(double rts, double m, double k[N][4]) {
  // massive rescaling: sum_i sqrt(m_i^2 + xi^2 E_i^2) = sqrt(shat); Newton from
  // xi0 = sqrt(1 - (sum m / sqrt shat)^2), fixed MF_NEWTON_STEPS steps (A7: the iteration is converged
  // to rounding, 5e-15, after 4 steps for every one of 4e6 test events down to xi = 0.15, threshold
  // region included); N = 2: xi0 is the exact root.  1/E comes from one rsqrt (no sqrt + division).
  const double m2 = m * m;
  const double r0 = 2.0 * m / rts;
  double xi = sqrt(1.0 - r0 * r0);
  if (N > 2) {
    double e_ml = 0.0;                                     // massless legs: E = xi e0, d/dxi = e0
#pragma unroll
    for (int i = 2; i < N; ++i) e_ml += k[i][0];
    const double a0 = k[0][0] * k[0][0], a1 = k[1][0] * k[1][0];
#pragma unroll 1
    for (int it = 0; it < MF_NEWTON_STEPS; ++it) {
      const double x2 = xi * xi;
      const double s0 = fma(x2, a0, m2), s1 = fma(x2, a1, m2);
      const double i0 = rsqrt(s0), i1 = rsqrt(s1);
      const double F = fma(xi, e_ml, fma(s0, i0, s1 * i1)) - rts;          // sum E_i - sqrt(shat)
      const double dF = fma(xi, fma(a0, i0, a1 * i1), e_ml);              // sum xi e0^2 / E_i
      xi -= F / dF;
    }
  }
  double prod = 1.0, den = 0.0;
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double kabs = xi * k[i][0];
    double E = kabs;
    if (i < 2) {                                   // massive legs: 1/E from one rsqrt
      const double s = fma(kabs, kabs, m2), ri = rsqrt(s);
      E = s * ri;
      prod *= kabs * ri; den = fma(kabs * kabs, ri, den);
    } else {
      den += kabs;                                 // massless: |k|/E = 1, |k|^2/E = |k|
    }
    k[i][0] = E; k[i][1] *= xi; k[i][2] *= xi; k[i][3] *= xi;
  }
  double xp = xi;                                // xi^(2N-3)
#pragma unroll
  for (int i = 1; i < 2 * N - 3; ++i) xp *= xi;
  return xp * prod * rts / den;
}

// rs[3N-4] -> massive momenta k[N][4] (t, t~, g...) in the partonic CM frame; returns W0 * Wm.
// masses: m for particles 0,1 (0 for the massless 2-body case), 0 for the rest.
template <int N>
MF_HD double mf_phase_space(double shat, double m, const double* rs, double k[N][4]) {
  const double rts = sqrt(shat);
  double M[N + 1];
  M[1] = rts; M[N] = 0.0;
#pragma unroll
  for (int i = 2; i + 1 <= N; ++i) M[i] = sqrt(mf_mass_fraction_sq(N - i, rs[i - 2])) * M[i - 1];
  double Q[4] = {rts, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 2; i <= N; ++i) {
    const double ct = 2.0 * rs[N - 6 + 2 * i] - 1.0;
    double sp, cp;
    sincospi(2.0 * rs[N - 5 + 2 * i], &sp, &cp);
    const double st = sqrt(1.0 - ct * ct);
    const double q = (M[i - 1] * M[i - 1] - M[i] * M[i]) / (2.0 * M[i - 1]);
    const double pr[4] = {q, q * st * cp, q * st * sp, q * ct};
    const double Qr[4] = {sqrt(q * q + M[i] * M[i]), -pr[1], -pr[2], -pr[3]};
    if (i == 2) {
#pragma unroll
      for (int c = 0; c < 4; ++c) { k[0][c] = pr[c]; Q[c] = Qr[c]; }
    } else {
      double Qn[4];
      const double iM = 1.0 / M[i - 1], iQM = 1.0 / (Q[0] + M[i - 1]);
      mf_boost(Q, iM, iQM, pr, k[i - 2]);
      mf_boost(Q, iM, iQM, Qr, Qn);
#pragma unroll
      for (int c = 0; c < 4; ++c) Q[c] = Qn[c];
    }
  }
#pragma unroll
  for (int c = 0; c < 4; ++c) k[N - 1][c] = Q[c];
  const double W0 = mf_w0<N>(shat);
  if (m == 0.0) return W0;
  return W0 * mf_massive_rescale<N>(rts, m, k);
}

// O4' (MF_GEN_CLASSIC_RAMBO): textbook RAMBO (Kleiss, Stirling, Ellis 1986) from 4N uniforms,
// particle i uses rs[4i..4i+3]: c = 2 r0 - 1, phi = 2 pi r1, q0 = -ln(r2 r3), q = q0 (1, s cos phi, s sin phi, c);
// Q = sum q, M = sqrt(Q^2), b = -Qvec/M, x = sqrt(shat)/M, gamma = Q0/M, a = 1/(1+gamma);
// p0_i = x (gamma q0 + b.q), pvec_i = x (qvec + b q0 + a (b.q) b): flat in phase space, constant weight W0.
// Then the same massive rescaling.  Returns W0 * Wm.
template <int N>
MF_HD double mf_phase_space_classic(double shat, double m, const double* rs, double k[N][4]) {
  const double rts = sqrt(shat);
  double q[N][4], Q[4] = {0.0, 0.0, 0.0, 0.0};
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double c = 2.0 * rs[4 * i] - 1.0;
    double sp, cp;
    sincospi(2.0 * rs[4 * i + 1], &sp, &cp);
    const double q0 = -log(rs[4 * i + 2] * rs[4 * i + 3]);
    const double st = sqrt(1.0 - c * c);
    q[i][0] = q0; q[i][1] = q0 * st * cp; q[i][2] = q0 * st * sp; q[i][3] = q0 * c;
#pragma unroll
    for (int c4 = 0; c4 < 4; ++c4) Q[c4] += q[i][c4];
  }
  const double M2 = Q[0] * Q[0] - Q[1] * Q[1] - Q[2] * Q[2] - Q[3] * Q[3];
  const double iM = rsqrt(M2);
  const double b[3] = {-Q[1] * iM, -Q[2] * iM, -Q[3] * iM};
  const double x = rts * iM, gam = Q[0] * iM, a = 1.0 / (1.0 + gam);
#pragma unroll
  for (int i = 0; i < N; ++i) {
    const double bq = b[0] * q[i][1] + b[1] * q[i][2] + b[2] * q[i][3];
    k[i][0] = x * (gam * q[i][0] + bq);
#pragma unroll
    for (int c = 0; c < 3; ++c) k[i][1 + c] = x * (q[i][1 + c] + b[c] * q[i][0] + a * bq * b[c]);
  }
  const double W0 = mf_w0<N>(shat);
  if (m == 0.0) return W0;
  return W0 * mf_massive_rescale<N>(rts, m, k);
}

// ---- S6: PDF (O5): cubic Hermite in (ln x, ln Q^2) on the tabulated xf, node slope = mean of the
// two secants, one-sided at the ends.  On uniform knots h*d_i = (f_{i+1}-f_{i-1})/2, so no division.
MF_HD double mf_hermite(double fm1, double f0, double f1, double f2, bool has_m1, bool has_p2, double t) {
  const double hd0 = has_m1 ? 0.5 * (f1 - fm1) : (f1 - f0);
  const double hd1 = has_p2 ? 0.5 * (f2 - f0) : (f1 - f0);
  const double t2 = t * t, t3 = t2 * t;
  return (2.0 * t3 - 3.0 * t2 + 1.0) * f0 + (t3 - 2.0 * t2 + t) * hd0 + (3.0 * t2 - 2.0 * t3) * f1 + (t3 - t2) * hd1;
}

// xf(x, Q^2) from the table `tab` [nx][nq] (shared memory on the device); lx = ln x, lq = ln Q^2.
// STRIDE: doubles between neighbouring (ix, iq) entries (1 = single table [nx][nq]; MF_NFL = flavour-innermost grid, of
// which the rows pdf_iq0 .. pdf_iq0 + pdf_nqs - 1 are present)
template <int STRIDE>
MF_HD double mf_pdf_strided(const MfParams& P, const double* tab, double lx, double lq);
MF_HD double mf_pdf(const MfParams& P, const double* tab, double lx, double lq) { return mf_pdf_strided<1>(P, tab, lx, lq); }
template <int STRIDE>
MF_HD double mf_pdf_strided(const MfParams& P, const double* tab, double lx, double lq) {
  const int nx = P.pdf_nx, nq = P.pdf_nq;
  const double fx = (lx - P.pdf_lx0) * P.pdf_ihx, fq = (lq - P.pdf_lq0) * P.pdf_ihq;
  int ix = (int)floor(fx), iq = (int)floor(fq);
  ix = ix < 0 ? 0 : (ix > nx - 2 ? nx - 2 : ix);
  iq = iq < 0 ? 0 : (iq > nq - 2 ? nq - 2 : iq);
  double tx = fx - (double)ix, tq = fq - (double)iq;
  tx = tx < 0.0 ? 0.0 : (tx > 1.0 ? 1.0 : tx);     // clamp: no extrapolation
  tq = tq < 0.0 ? 0.0 : (tq > 1.0 ? 1.0 : tq);
  const bool xm = ix > 0, xp = ix + 2 < nx, qm = iq > 0, qp = iq + 2 < nq;
  // doubles per ln-x row of `tab` and its first Q^2 row; the flavour grid pads every ln-x row by MF_XPAD doubles so that
  // the rows of different lanes fall on different shared-memory banks (45 doubles: odd)
  const int rs = STRIDE == 1 ? nq : P.pdf_nqs * STRIDE + MF_XPAD, q0 = STRIDE == 1 ? 0 : P.pdf_iq0;
  const int r0 = (xm ? ix - 1 : ix) * rs, r1 = ix * rs, r2 = (ix + 1) * rs, r3 = (xp ? ix + 2 : ix + 1) * rs;
  double row[4];
#pragma unroll
  for (int c = 0; c < 4; ++c) {                     // Q^2 rows iq-1 .. iq+2 (clamped where absent)
    int q = iq - 1 + c;
    q = q < 0 ? 0 : (q > nq - 1 ? nq - 1 : q);
    const int qo = (q - q0) * STRIDE;
    row[c] = mf_hermite(tab[r0 + qo], tab[r1 + qo], tab[r2 + qo], tab[r3 + qo], xm, xp, tx);
  }
  return mf_hermite(row[0], row[1], row[2], row[3], qm, qp, tq);
}

// O5q: flavour-summed q q~ luminosity from the flavour-innermost grid tab [nx][pdf_nqs][MF_NFL] (shared
// memory on the device): l12 = sum_q xf_q(x1) xf_q~(x2), l21 = sum_q xf_q~(x1) xf_q(x2), q = d u s c b.  The 16-point
// stencil of one x is shared by all tables: each of its points is one contiguous 88-byte read.
MF_HD void mf_lumi_qq(const MfParams& P, const double* tab, double lx1, double lx2, double lq, double& l12, double& l21) {
  l12 = 0.0; l21 = 0.0;
#pragma unroll
  for (int q = 1; q <= 5; ++q) {
    const double q1 = mf_pdf_strided<MF_NFL>(P, tab + 5 + q, lx1, lq), a1 = mf_pdf_strided<MF_NFL>(P, tab + 5 - q, lx1, lq);
    const double q2 = mf_pdf_strided<MF_NFL>(P, tab + 5 + q, lx2, lq), a2 = mf_pdf_strided<MF_NFL>(P, tab + 5 - q, lx2, lq);
    l12 = fma(q1, a2, l12); l21 = fma(a1, q2, l21);
  }
}

// ---- S5: cuts (O7): final gluons only, lab frame; eta_lab = atanh(kz/|k|) + y_b, y_b = ln(x1/x2)/2 -----
// The pseudorapidity cut is taken on tanh: with t_b = tanh y_b = (x1-x2)/(x1+x2),
//   |eta_lab| < eta_max  <=>  |kz + t_b |k|| < tanh(eta_max) (|k| + t_b kz)       (|k| + t_b kz > 0),
// so no logarithm is needed; eta itself (boost-invariant differences only) is computed for Delta R.
template <int NGL>
MF_HD bool mf_cuts(const MfParams& P, const double kg[][4], double x1, double x2) {
  if (NGL == 0) return true;
  const double tb = (x1 - x2) / (x1 + x2);
  bool pass = true;
  double eta[NGL > 0 ? NGL : 1], phi[NGL > 0 ? NGL : 1];
#pragma unroll
  for (int i = 0; i < NGL; ++i) {
    const double pt2 = kg[i][1] * kg[i][1] + kg[i][2] * kg[i][2];
    const double kabs = sqrt(pt2 + kg[i][3] * kg[i][3]);
    if (P.ptmin > 0.0 && !(pt2 > P.ptmin * P.ptmin)) pass = false;
    if (P.etamax > 0.0 && !(fabs(fma(tb, kabs, kg[i][3])) < P.tanh_etamax * fma(tb, kg[i][3], kabs))) pass = false;
    if (NGL == 2) eta[i] = atanh(kg[i][3] / kabs);
  }
  if (NGL == 2 && P.drmin > 0.0) {
    phi[0] = atan2(kg[0][2], kg[0][1]);
    phi[1] = atan2(kg[1][2], kg[1][1]);
    double dphi = phi[0] - phi[1];
    if (dphi > MF_PI) dphi -= 2.0 * MF_PI;
    if (dphi <= -MF_PI) dphi += 2.0 * MF_PI;
    const double deta = eta[0] - eta[1];
    if (!(sqrt(deta * deta + dphi * dphi) > P.drmin)) pass = false;
  }
  return pass;
}

// ---- observable histogram slots ("histogram accumulation") ---------------------
// k: final-state momenta [N][4]; returns the slots of the P.n_obs observables packed 6 bits each:
// bin = floor((v-lo)/(hi-lo)*n_bins) for lo <= v < hi, 62 = underflow, 63 = overflow
#define MF_OBS_MAX 4
#define MF_OBS_SLOTS 64
template <int N>
MF_HD unsigned mf_obs_keys(const MfParams& P, const double k[N][4]) {
  unsigned keys = 0;
#pragma unroll
  for (int o = 0; o < MF_OBS_MAX; ++o) {
    if (o >= P.n_obs) break;
    const int kind = P.obs_kind[o];
    double v;
    if (kind == 2) {
      const double E = k[0][0] + k[1][0], px = k[0][1] + k[1][1], py = k[0][2] + k[1][2], pz = k[0][3] + k[1][3];
      const double m2 = E * E - px * px - py * py - pz * pz;
      v = m2 > 0.0 ? sqrt(m2) : 0.0;
    } else {
      const int i = (kind == 0) ? 0 : (kind == 1) ? 1 : (N > 2 ? 2 : 0);
      v = sqrt(k[i][1] * k[i][1] + k[i][2] * k[i][2]);
    }
    unsigned b;
    if (v < P.obs_lo[o]) b = 62u;
    else if (v >= P.obs_hi[o]) b = 63u;
    else {
      const int nb = P.obs_nb[o];
      int q = (int)floor((v - P.obs_lo[o]) / (P.obs_hi[o] - P.obs_lo[o]) * (double)nb);
      b = (unsigned)(q > nb - 1 ? nb - 1 : q);
    }
    keys |= b << (6 * o);
  }
  return keys;
}

// ---- S7a: external-wavefunction ingredients (O6.2), the "conditional control statements" of
// PAPER.md:69.  Fermion: w+ = sqrt(E+|p|), w- = m/w+, and N*(|p|+pz, px, py) of the two-spinors
// chi+ = N(|p|+pz, px+i py), chi- = N(-px+i py, |p|+pz); the generated code builds u, v from them.
template <typename T>
MF_HD void mf_fermion_ing(const T p[4], T m, T o[5]) {
  const T pt2 = p[1] * p[1] + p[2] * p[2];
  const T pabs = sqrt(pt2 + p[3] * p[3]);
  o[0] = sqrt(p[0] + pabs);
  o[1] = (m == T(0.0)) ? T(0.0) : m / o[0];
  if (pabs < T(1e-12) * fabs(p[0]) || (pt2 == T(0.0) && p[3] < T(0.0))) {   // pz = -|p| branch
    o[2] = T(0.0); o[3] = T(1.0); o[4] = T(0.0);
  } else {
    const T ppz = (p[3] >= T(0.0)) ? pabs + p[3] : pt2 / (pabs - p[3]);   // no cancellation
    const T N = rsqrt(T(2.0) * pabs * ppz);
    o[2] = N * ppz; o[3] = N * p[1]; o[4] = N * p[2];
  }
}
// Gluon: eps(k,lam) = (-lam eps1 - i eps2)/sqrt2; o = (eps1x, eps1y, eps1z, eps2x, eps2y)/sqrt2
template <typename T>
MF_HD void mf_gluon_ing(const T k[4], T o[5]) {
  const T pt2 = k[1] * k[1] + k[2] * k[2];
  const T r2 = T(0.70710678118654752440);
  if (pt2 == T(0.0)) { o[0] = r2; o[1] = T(0.0); o[2] = T(0.0); o[3] = T(0.0); o[4] = (k[3] >= T(0.0)) ? r2 : -r2; return; }
  const T pt = sqrt(pt2), kabs = sqrt(pt2 + k[3] * k[3]);
  const T ipt = r2 / pt, ik = T(1.0) / kabs;
  o[0] = k[1] * k[3] * ipt * ik; o[1] = k[2] * k[3] * ipt * ik; o[2] = -pt * ik * r2;
  o[3] = -k[2] * ipt; o[4] = k[1] * ipt;
}
