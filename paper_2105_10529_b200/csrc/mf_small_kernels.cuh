// mf_small_kernels.cuh -- the per-iteration O(d*nb) kernels (reduce, finalize/refine, combine) and the
// DFMA peak microbenchmark; included by mf_api.cu only.
#pragma once
#include "mf_kernels.cuh"
#ifndef MF_OBS_ACC
#define MF_OBS_ACC (2 * MF_OBS_MAX * MF_OBS_SLOTS)
#endif

// ---- fixed-order sum of per-block partials into the raw sums (adds: sharded accumulation) -----------
// one warp per output element: lane l adds partials l, l+32, ... in order, then a xor-butterfly
// (fixed order: bit-reproducible for a fixed number of partials).  Launch: ceil((na+2)/8) CTAs of 256.
#define MF_REDUCE_THREADS 256
__global__ void __launch_bounds__(MF_REDUCE_THREADS)
mf_reduce_kernel(const double* __restrict__ partial, const unsigned long long* __restrict__ pcount,
                 int nblocks, int na, int row, double* __restrict__ acc, unsigned long long* __restrict__ counts) {
  const int e = blockIdx.x * (MF_REDUCE_THREADS / 32) + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (e < na) {
    double s = 0.0;
    for (int b = lane; b < nblocks; b += 32) s += partial[(size_t)b * row + e];   // rows of `row` doubles, the first na live
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
    if (lane == 0) acc[e] += s;
  } else if (e < na + 2) {
    unsigned long long c = 0;
    for (int b = lane; b < nblocks; b += 32) c += pcount[2 * b + (e - na)];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) c += __shfl_xor_sync(0xffffffffu, c, o);
    if (lane == 0) counts[e - na] += c;
  }
}

// ---- S10 (O10): sigma_I^2 = max(0, (N S2 - I^2)/(N-1)); Lepage refinement of every dimension --------
// one block of d warps; warp j refines dimension j: smooth (3-point, 2-point at the ends), normalise,
// floor 1e-30, compress r = ((s-1)/ln s)^alpha (lanes work on bins lane, lane+32: the pow/log are the
// expensive part), then lane 0 re-bins so that each new bin holds sum(r)/nb.  Sums over bins are
// taken serially by every lane from shared memory (fixed order).
__global__ void mf_finalize_kernel(const MfParams P, double alpha, double n_total, unsigned long long n_events,
                                   const double* __restrict__ acc, const unsigned long long* __restrict__ counts,
                                   double* __restrict__ edges, MfDevState* __restrict__ st, double* __restrict__ obs_total) {
  __shared__ double s_r[MF_DMAX][MF_NBMAX], s_e[MF_DMAX][MF_NBMAX + 1];
  const int j = threadIdx.x >> 5, lane = threadIdx.x & 31, nb = P.nb;
  if (P.n_obs > 0) {                                      // this iteration's observable histograms join the accumulated ones
    const double* oa = acc + 2 + P.d * nb;
    for (int i = threadIdx.x; i < MF_OBS_ACC; i += blockDim.x) obs_total[i] += oa[i];
    if (threadIdx.x == 0) obs_total[MF_OBS_ACC] += 1.0;   // iterations summed
  }
  if (threadIdx.x == 0) {
    const double I = acc[0], S2 = acc[1];
    double var = (n_total * S2 - I * I) / (n_total - 1.0);
    var = var > 0.0 ? var : 0.0;
    const unsigned k = st->n_iter;
    if (k < MF_MAX_ITER) {
      st->it[k].I = I; st->it[k].sig = sqrt(var);
      st->it[k].n = n_events; st->it[k].pass = counts[0]; st->it[k].bad = counts[1];
      st->n_iter = k + 1;
    }
  }
  if (j >= P.d) return;
  const double* h = acc + 2 + j * nb;
  double* e = edges + j * (nb + 1);
  double* r = s_r[j];
  double* eo = s_e[j];
  for (int k = lane; k < nb; k += 32) {
    double s;
    if (nb == 1) s = h[0];
    else if (k == 0) s = (h[0] + h[1]) * 0.5;
    else if (k == nb - 1) s = (h[nb - 2] + h[nb - 1]) * 0.5;
    else s = (h[k - 1] + h[k] + h[k + 1]) / 3.0;
    r[k] = s;
  }
  for (int k = lane; k <= nb; k += 32) eo[k] = e[k];
  __syncwarp();
  double tot = 0.0;
  for (int k = 0; k < nb; ++k) tot += r[k];
  if (!(tot > 0.0)) return;                               // nothing sampled here: keep this grid (warp-uniform)
  __syncwarp();
  for (int k = lane; k < nb; k += 32) {
    double s = r[k] / tot;
    s = s < 1e-30 ? 1e-30 : s;
    r[k] = (s == 1.0) ? 1.0 : pow((s - 1.0) / log(s), alpha);
  }
  __syncwarp();
  if (lane != 0) return;
  double rtot = 0.0;
  for (int k = 0; k < nb; ++k) rtot += r[k];
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

// ---- device-side exchange of the raw sums (multi-GPU without host round trips) -------------------------
// buf = [acc[0..n), (double)counts[0], (double)counts[1]]: one buffer for one all-reduce (counts < 2^53: exact)
__global__ void mf_pack_accum_kernel(const double* __restrict__ acc, const unsigned long long* __restrict__ counts, int n,
                                     double* __restrict__ buf) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) buf[i] = acc[i];
  else if (i < n + 2) buf[i] = (double)counts[i - n];
}
__global__ void mf_unpack_accum_kernel(const double* __restrict__ buf, int n, double* __restrict__ acc,
                                       unsigned long long* __restrict__ counts) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i < n) acc[i] = buf[i];
  else if (i < n + 2) counts[i - n] = (unsigned long long)__double2ll_rn(buf[i]);
}

// ---- O11: I = sum(I_j/s_j^2)/sum(1/s_j^2), sigma = (sum 1/s_j^2)^-1/2, chi2/dof ----------------------
__global__ void mf_combine_kernel(MfDevState* __restrict__ st) {
  if (threadIdx.x != 0 || blockIdx.x != 0) return;
  const unsigned n = st->n_iter;
  bool any_zero = false;
  for (unsigned j = 0; j < n; ++j) if (!(st->it[j].sig > 0.0)) any_zero = true;
  double I = 0.0, sig = 0.0, chi2 = 0.0;
  if (n > 0 && any_zero) {                                // fall back to the plain mean
    double m = 0.0, v = 0.0;
    for (unsigned j = 0; j < n; ++j) { m += st->it[j].I; v += st->it[j].sig * st->it[j].sig; }
    I = m / n; sig = sqrt(v) / n;
  } else if (n > 0) {
    double sw = 0.0, swi = 0.0;
    for (unsigned j = 0; j < n; ++j) { const double w = 1.0 / (st->it[j].sig * st->it[j].sig); sw += w; swi += w * st->it[j].I; }
    I = swi / sw; sig = 1.0 / sqrt(sw);
    if (n > 1) {
      for (unsigned j = 0; j < n; ++j) { const double dl = st->it[j].I - I; chi2 += dl * dl / (st->it[j].sig * st->it[j].sig); }
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
