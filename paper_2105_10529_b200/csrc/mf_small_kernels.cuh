// mf_small_kernels.cuh -- the per-iteration O(d*nb) kernels (reduce, finalize/refine, combine) and the
// DFMA peak microbenchmark; included by mf_api.cu only.
#pragma once
#include "mf_kernels.cuh"

// ---- fixed-order sum of per-block partials into the raw sums (adds: sharded accumulation) -----------
__global__ void mf_reduce_kernel(const double* __restrict__ partial, const unsigned long long* __restrict__ pcount,
                                 int nblocks, int na, double* __restrict__ acc, unsigned long long* __restrict__ counts) {
  const int e = blockIdx.x * blockDim.x + threadIdx.x;
  if (e < na) {
    double s = 0.0;
    for (int b = 0; b < nblocks; ++b) s += partial[(size_t)b * na + e];
    acc[e] += s;
  }
  if (e < 2) {
    unsigned long long c = 0;
    for (int b = 0; b < nblocks; ++b) c += pcount[2 * b + e];
    counts[e] += c;
  }
}

// ---- S10 (O10): sigma_I^2 = max(0, (N S2 - I^2)/(N-1)); Lepage refinement of every dimension --------
// one block; thread j < d refines dimension j: smooth (3-point, 2-point at the ends), normalise,
// floor 1e-30, compress r = ((s-1)/ln s)^alpha, re-bin so that each new bin holds sum(r)/nb.
__global__ void mf_finalize_kernel(const MfParams P, double alpha, double n_total, unsigned long long n_events,
                                   const double* __restrict__ acc, const unsigned long long* __restrict__ counts,
                                   double* __restrict__ edges, MfDevState* __restrict__ st) {
  const int j = threadIdx.x, nb = P.nb;
  if (j == 0) {
    const double I = acc[0], S2 = acc[1];
    double var = (n_total * S2 - I * I) / (n_total - 1.0);
    var = var > 0.0 ? var : 0.0;
    const unsigned k = st->n_iter;
    if (k < MF_MAX_ITER) {
      st->it_I[k] = I; st->it_sig[k] = sqrt(var);
      st->it_n[k] = n_events; st->it_pass[k] = counts[0]; st->it_bad[k] = counts[1];
      st->n_iter = k + 1;
    }
  }
  if (j >= P.d) return;
  const double* h = acc + 2 + j * nb;
  double* e = edges + j * (nb + 1);
  double r[MF_NBMAX], eo[MF_NBMAX + 1];
  double tot = 0.0;
  for (int k = 0; k < nb; ++k) {
    double s;
    if (nb == 1) s = h[0];
    else if (k == 0) s = (h[0] + h[1]) * 0.5;
    else if (k == nb - 1) s = (h[nb - 2] + h[nb - 1]) * 0.5;
    else s = (h[k - 1] + h[k] + h[k + 1]) / 3.0;
    r[k] = s; tot += s;
  }
  if (!(tot > 0.0)) return;                               // nothing sampled here: keep this grid
  double rtot = 0.0;
  for (int k = 0; k < nb; ++k) {
    double s = r[k] / tot;
    s = s < 1e-30 ? 1e-30 : s;
    r[k] = (s == 1.0) ? 1.0 : pow((s - 1.0) / log(s), alpha);
    rtot += r[k];
  }
  for (int k = 0; k <= nb; ++k) eo[k] = e[k];
  double cum = 0.0;
  int k = 0;
  for (int m = 1; m < nb; ++m) {
    const double target = rtot * (double)m / (double)nb;
    while (k < nb - 1 && cum + r[k] < target) { cum += r[k]; ++k; }
    double frac = (target - cum) / r[k];
    frac = frac < 0.0 ? 0.0 : (frac > 1.0 ? 1.0 : frac);
    e[m] = eo[k] + frac * (eo[k + 1] - eo[k]);
  }
}

// ---- O11: I = sum(I_j/s_j^2)/sum(1/s_j^2), sigma = (sum 1/s_j^2)^-1/2, chi2/dof ----------------------
__global__ void mf_combine_kernel(MfDevState* __restrict__ st) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const unsigned n = st->n_iter;
  bool any_zero = false;
  for (unsigned j = 0; j < n; ++j) if (!(st->it_sig[j] > 0.0)) any_zero = true;
  double I = 0.0, sig = 0.0, chi2 = 0.0;
  if (n > 0 && any_zero) {                                // fall back to the plain mean
    double m = 0.0, v = 0.0;
    for (unsigned j = 0; j < n; ++j) { m += st->it_I[j]; v += st->it_sig[j] * st->it_sig[j]; }
    I = m / n; sig = sqrt(v) / n;
  } else if (n > 0) {
    double sw = 0.0, swi = 0.0;
    for (unsigned j = 0; j < n; ++j) { const double w = 1.0 / (st->it_sig[j] * st->it_sig[j]); sw += w; swi += w * st->it_I[j]; }
    I = swi / sw; sig = 1.0 / sqrt(sw);
    if (n > 1) {
      for (unsigned j = 0; j < n; ++j) { const double dl = st->it_I[j] - I; chi2 += dl * dl / (st->it_sig[j] * st->it_sig[j]); }
      chi2 /= (double)(n - 1);
    }
  }
  st->res_I = I; st->res_sig = sig; st->res_chi2 = chi2;
}

// ---- fp64 roofline peak: 8 independent DFMA chains per thread, all in registers --------------------
__global__ void __launch_bounds__(256) mf_dfma_kernel(double* out, int iters, double a, double b) {
  double x0 = threadIdx.x * 1e-3, x1 = x0 + 1.0, x2 = x0 + 2.0, x3 = x0 + 3.0, x4 = x0 + 4.0, x5 = x0 + 5.0,
         x6 = x0 + 6.0, x7 = x0 + 7.0;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 16; ++u) {
      x0 = fma(x0, a, b); x1 = fma(x1, a, b); x2 = fma(x2, a, b); x3 = fma(x3, a, b);
      x4 = fma(x4, a, b); x5 = fma(x5, a, b); x6 = fma(x6, a, b); x7 = fma(x7, a, b);
    }
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = ((x0 + x1) + (x2 + x3)) + ((x4 + x5) + (x6 + x7));
}
#define MF_DFMA_PER_ITER (16 * 8)
