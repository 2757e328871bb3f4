// mf_proc.cu -- the per-process kernels, compiled once per process with -DMF_PROC=0..5 so that the
// |M|^2 codes build in parallel: the fused iteration (mf_iterate_kernel, mf_iterate_compact_kernel), the
// staged iteration of the heavy processes (mf_front_kernel -> mf_me_kernel -> mf_hist_kernel), and the
// per-event evaluation (mf_eval_kernel); plus their launchers (MfProcOps, mf_proc.h).
#include "mf_kernels.cuh"
#include "mf_proc.h"
#include <type_traits>
#ifndef MF_PROC
#error "compile with -DMF_PROC=0..7"
#endif

__device__ __forceinline__ void mf_stage_tables(const MfParams& P, const double* g_edges, const double* g_pdf,
                                                double* s_edges, double* s_pdf) {
  const int ne = P.d * (P.nb + 1), np = P.pdf_smem;      // gluon table, or the active rows of the flavour grid (mf_params.h)
  for (int i = threadIdx.x; i < ne; i += blockDim.x) s_edges[i] = g_edges[i];
  for (int i = threadIdx.x; i < np; i += blockDim.x) s_pdf[i] = g_pdf[i];
}

// ---- S9: per-warp histogram update in fixed order -------------------------------------------------------
// H[j][bin_j] += t2 for every contributing lane of the warp, lanes that share a bin served in lane order
// (so the sum order is fixed: reading A22).  The peer masks come from six ballots per dimension (one per
// key bit) instead of match.any, whose latency (~800 cycles under load, profiles/r1_tuning.md)
// dominated the reduction stage; the ranks of all dimensions are resolved first so that each round
// issues D independent shared-memory updates.
template <int D>
__device__ __forceinline__ void mf_hist_add(double* __restrict__ hw, int nb, unsigned long long packed, bool contrib,
                                            double t2, unsigned lt_mask) {
  const unsigned full = 0xffffffffu;
  const unsigned cmask = __ballot_sync(full, contrib);
  if (cmask == 0u) return;                               // warp-uniform
  unsigned rank[D], key[D], maxrank = 0;
#pragma unroll
  for (int j = 0; j < D; ++j) {
    key[j] = (unsigned)((packed >> (6 * j)) & 63ull);
    unsigned peers = cmask;
#pragma unroll
    for (int b = 0; b < 6; ++b) {
      const bool bit = (key[j] >> b) & 1u;
      const unsigned bal = __ballot_sync(full, bit);
      peers &= bit ? bal : ~bal;
    }
    rank[j] = __popc(peers & lt_mask);
    maxrank = rank[j] > maxrank ? rank[j] : maxrank;
  }
  for (unsigned r = 0; __any_sync(full, contrib && maxrank >= r); ++r) {      // ranks are < 32
#pragma unroll
    for (int j = 0; j < D; ++j)
      if (contrib && rank[j] == r) hw[j * nb + key[j]] += t2;
    __syncwarp();
  }
}

// D > 10 (classic 4n-random RAMBO): the bins of dimensions 10.. are in a second packed word
template <int D>
__device__ __forceinline__ void mf_hist_add2(double* __restrict__ hw, int nb, unsigned long long lo, unsigned long long hi,
                                             bool contrib, double t2, unsigned lt_mask) {
  mf_hist_add<(D < MF_PACK_DIMS ? D : MF_PACK_DIMS)>(hw, nb, lo, contrib, t2, lt_mask);
  if constexpr (D > MF_PACK_DIMS) mf_hist_add<D - MF_PACK_DIMS>(hw + MF_PACK_DIMS * nb, nb, hi, contrib, t2, lt_mask);
}

// observable histograms of one warp: ho1[o][64] += t, ho2[o][64] += t^2, same fixed-order scheme
__device__ __forceinline__ void mf_obs_add(double* __restrict__ ho1, double* __restrict__ ho2, int n_obs, unsigned keys,
                                           bool contrib, double t, double t2, unsigned lt_mask) {
  const unsigned full = 0xffffffffu;
  const unsigned cmask = __ballot_sync(full, contrib);
  if (cmask == 0u) return;                               // warp-uniform
  unsigned rank[MF_OBS_MAX], key[MF_OBS_MAX], maxrank = 0;
#pragma unroll
  for (int j = 0; j < MF_OBS_MAX; ++j) {
    key[j] = (keys >> (6 * j)) & 63u; rank[j] = 0;
    if (j < n_obs) {                                     // warp-uniform
      unsigned peers = cmask;
#pragma unroll
      for (int b = 0; b < 6; ++b) {
        const bool bit = (key[j] >> b) & 1u;
        const unsigned bal = __ballot_sync(full, bit);
        peers &= bit ? bal : ~bal;
      }
      rank[j] = __popc(peers & lt_mask);
      maxrank = rank[j] > maxrank ? rank[j] : maxrank;
    }
  }
  for (unsigned r = 0; __any_sync(full, contrib && maxrank >= r); ++r) {
#pragma unroll
    for (int j = 0; j < MF_OBS_MAX; ++j)
      if (j < n_obs && contrib && rank[j] == r) { ho1[j * MF_OBS_SLOTS + key[j]] += t; ho2[j * MF_OBS_SLOTS + key[j]] += t2; }
    __syncwarp();
  }
}
#define MF_OBS_ACC (2 * MF_OBS_MAX * MF_OBS_SLOTS)         // doubles per record behind the 2 + d*nb VEGAS sums

// fixed-order end of a reducing CTA: xor-butterfly inside the warp, warps in index order inside the block, one
// partial record (2 + nh doubles, then the observable sums if s_obs != nullptr) and one counter pair per CTA
__device__ __forceinline__ void mf_block_finish(double s1, double s2, unsigned long long n_pass, unsigned long long n_bad,
                                                const double* __restrict__ s_hist, int nh, const double* __restrict__ s_obs,
                                                double* __restrict__ s_red, double* __restrict__ out,
                                                unsigned long long* __restrict__ pc) {
  const int nw = blockDim.x >> 5, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) {
    s1 += __shfl_xor_sync(0xffffffffu, s1, o);
    s2 += __shfl_xor_sync(0xffffffffu, s2, o);
    n_pass += __shfl_xor_sync(0xffffffffu, n_pass, o);
    n_bad += __shfl_xor_sync(0xffffffffu, n_bad, o);
  }
  if (lane == 0) {
    s_red[warp * 4 + 0] = s1; s_red[warp * 4 + 1] = s2;
    s_red[warp * 4 + 2] = __longlong_as_double((long long)n_pass);
    s_red[warp * 4 + 3] = __longlong_as_double((long long)n_bad);
  }
  __syncthreads();
  for (int e = threadIdx.x; e < nh; e += blockDim.x) {
    double s = 0.0;
    for (int w = 0; w < nw; ++w) s += s_hist[w * nh + e];
    out[2 + e] = s;
  }
  if (s_obs) for (int e = threadIdx.x; e < MF_OBS_ACC; e += blockDim.x) {
    double s = 0.0;
    for (int w = 0; w < nw; ++w) s += s_obs[w * MF_OBS_ACC + e];
    out[2 + nh + e] = s;
  }
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0; unsigned long long c = 0, d2 = 0;
    for (int w = 0; w < nw; ++w) {
      a += s_red[w * 4 + 0]; b += s_red[w * 4 + 1];
      c += (unsigned long long)__double_as_longlong(s_red[w * 4 + 2]);
      d2 += (unsigned long long)__double_as_longlong(s_red[w * 4 + 3]);
    }
    out[0] = a; out[1] = b;
    pc[0] = c; pc[1] = d2;
  }
}

// ---- S1-S9 fused ---------------------------------------------------------------------------------
// partial: [gridDim.x][row] doubles (2 + d*nb sums, then the observable sums), pcount: [gridDim.x][2]
// (n_pass, n_nonfinite)
template <int PROC, int CL>
__global__ void __launch_bounds__(MF_THREADS, MfLaunch<PROC>::MINB)
mf_iterate_kernel(const MfParams P, const double* __restrict__ g_edges, const double* __restrict__ g_pdf,
                  uint32_t iteration, unsigned long long first, unsigned long long n, double n_total,
                  double* __restrict__ partial, unsigned long long* __restrict__ pcount, int row) {
  constexpr int D = MfDim<PROC, CL>::D;
  extern __shared__ double smem[];
  const int nb = P.nb, nh = D * nb, nw = blockDim.x >> 5;
  double* s_edges = smem;
  double* s_pdf = s_edges + D * (nb + 1);
  double* s_hist = s_pdf + P.pdf_smem;                   // [nw][D*nb]
  double* s_red = s_hist + nw * nh;                      // [nw][4]
  double* s_obs = s_red + nw * 4;                        // [nw][MF_OBS_ACC] when observables are set
  mf_stage_tables(P, g_edges, g_pdf, s_edges, s_pdf);
  for (int i = threadIdx.x; i < nw * nh; i += blockDim.x) s_hist[i] = 0.0;
  if (P.n_obs > 0) for (int i = threadIdx.x; i < nw * MF_OBS_ACC; i += blockDim.x) s_obs[i] = 0.0;
  __syncthreads();

  const unsigned lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  double* hw = s_hist + warp * nh;
  double s1 = 0.0, s2 = 0.0;
  unsigned long long n_pass = 0, n_bad = 0;
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  const unsigned long long tbase = MF_UNIFORM_ME ? 0u : (threadIdx.x & ~31u);   // block- or warp-uniform trips
  for (unsigned long long base = (unsigned long long)blockIdx.x * blockDim.x + tbase; base < n; base += stride) {
    const unsigned long long i = base + (MF_UNIFORM_ME ? threadIdx.x : lane);
    const bool valid = i < n;
    int bin[D];
    bool pass = false;
    double F = 0.0;
    unsigned okeys = 0;
    if (MF_UNIFORM_ME) {                                 // every thread runs the event (barriers inside);
      F = mf_event<PROC, false, double, CL>(P, s_edges, s_pdf, iteration, first + (valid ? i : n - 1), bin, pass, nullptr, &okeys);
      if (!valid) { F = 0.0; pass = false; }             // lanes past the end recompute event n-1, discarded
    } else if (valid) {
      F = mf_event<PROC, false, double, CL>(P, s_edges, s_pdf, iteration, first + i, bin, pass, nullptr, &okeys);
    }
    if (!isfinite(F)) { F = 0.0; ++n_bad; }              // A20
    if (valid && pass) ++n_pass;
    const double t = F / n_total, t2 = t * t;            // O9: t_i = F_i / N
    s1 += t; s2 += t2;
    // per-warp histogram H[j][k] += t^2, lanes that share a bin are served in lane order
    unsigned long long packed, packed_hi;
    mf_pack_bins<D>(bin, packed, packed_hi);
    mf_hist_add2<D>(hw, nb, packed, packed_hi, valid && t2 != 0.0, t2, lt_mask);
    if (P.n_obs > 0)
      mf_obs_add(s_obs + warp * MF_OBS_ACC, s_obs + warp * MF_OBS_ACC + MF_OBS_ACC / 2, P.n_obs, okeys, valid && F != 0.0, t, t2, lt_mask);
  }
  // fixed-order reductions: xor-butterfly inside the warp, warps in index order inside the block
  mf_block_finish(s1, s2, n_pass, n_bad, s_hist, nh, P.n_obs > 0 ? s_obs : nullptr, s_red, partial + (size_t)blockIdx.x * row, pcount + 2 * blockIdx.x);
}

// ---- S1-S9 fused, with CTA-level compaction of the events that pass the cuts -------------------------
// Phase A: every thread runs the front end (S1-S6) of one event; the passing ones are appended, in
// event order (ballot + prefix over the warps, so the order is deterministic), to a queue in shared
// memory holding {momenta, sqrt(shat), weight prefactor, bins}.  Phase B: once the queue holds a full
// CTA of events (or the input is exhausted) every thread takes one entry and runs S7-S9.  All lanes
// of every warp then carry a passing event through the |M|^2 code (no idle lanes at an 85 % pass
// rate), and all threads reach the barrier points inside it.
template <int PROC>
__global__ void __launch_bounds__(MF_THREADS, MfLaunch<PROC>::MINB)
mf_iterate_compact_kernel(const MfParams P, const double* __restrict__ g_edges, const double* __restrict__ g_pdf,
                          uint32_t iteration, unsigned long long first, unsigned long long n, double n_total,
                          double* __restrict__ partial, unsigned long long* __restrict__ pcount, int row) {
  constexpr int D = MfProc<PROC>::D, N = MfProc<PROC>::N, NF = 4 * N + 3, T = MF_THREADS, CAP = 2 * MF_THREADS;
  extern __shared__ double smem[];
  const int nb = P.nb, nh = D * nb, nw = T >> 5;
  double* s_edges = smem;
  double* s_pdf = s_edges + D * (nb + 1);
  double* s_hist = s_pdf + P.pdf_smem;                   // [nw][D*nb]
  double* s_red = s_hist + nw * nh;                      // [nw][4]
  double* s_q = s_red + nw * 4;                          // [NF][CAP] field-major queue
  int* s_wtot = (int*)(s_q + NF * CAP);                  // [nw]
  mf_stage_tables(P, g_edges, g_pdf, s_edges, s_pdf);
  for (int i = threadIdx.x; i < nw * nh; i += T) s_hist[i] = 0.0;
  __syncthreads();

  const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  double* hw = s_hist + warp * nh;
  double s1 = 0.0, s2 = 0.0;
  unsigned long long n_pass = 0, n_bad = 0;
  const unsigned long long nchunks = (n + T - 1) / T;
  unsigned long long chunk = blockIdx.x;
  int qhead = 0, qcount = 0;                             // block-uniform
  while (true) {
    while (qcount < T && chunk < nchunks) {              // ---- phase A
      const unsigned long long i = chunk * T + tid;
      bool pass = false;
      int bin[D];
      double k[N][4], rts, pref;
      if (i < n) pass = mf_event_front<PROC, false>(P, s_edges, s_pdf, iteration, first + i, bin, k, rts, pref, nullptr);
      const unsigned bal = __ballot_sync(0xffffffffu, pass);
      if (lane == 0) s_wtot[warp] = __popc(bal);
      __syncthreads();
      int base = 0, tot = 0;
      for (int w = 0; w < nw; ++w) { const int c = s_wtot[w]; base += (w < (int)warp) ? c : 0; tot += c; }
      if (pass) {
        ++n_pass;
        const int slot = (qhead + qcount + base + __popc(bal & lt_mask)) % CAP;
#pragma unroll
        for (int p = 0; p < N; ++p)
#pragma unroll
          for (int c = 0; c < 4; ++c) s_q[(4 * p + c) * CAP + slot] = k[p][c];
        s_q[(4 * N) * CAP + slot] = rts;
        s_q[(4 * N + 1) * CAP + slot] = pref;
        unsigned long long packed = 0;                   // D <= 10 bins of 6 bits
#pragma unroll
        for (int j = 0; j < D; ++j) packed |= (unsigned long long)bin[j] << (6 * j);
        s_q[(4 * N + 2) * CAP + slot] = __longlong_as_double((long long)packed);
      }
      __syncthreads();
      qcount += tot;
      chunk += gridDim.x;
    }
    if (qcount == 0) break;
    const int m = qcount < T ? qcount : T;               // ---- phase B
    const bool have = (int)tid < m;
    const int slot = (qhead + (have ? (int)tid : 0)) % CAP;
    double k[N][4];
#pragma unroll
    for (int p = 0; p < N; ++p)
#pragma unroll
      for (int c = 0; c < 4; ++c) k[p][c] = s_q[(4 * p + c) * CAP + slot];
    const double rts = s_q[(4 * N) * CAP + slot], pref = s_q[(4 * N + 1) * CAP + slot];
    const unsigned long long packed = (unsigned long long)__double_as_longlong(s_q[(4 * N + 2) * CAP + slot]);
    __syncthreads();                                     // queue entries are in registers before anyone refills
    double F = pref * mf_me2<PROC>(P, rts, k);           // S7, S8 (every thread: barrier points inside)
    if (!have) F = 0.0;
    if (!isfinite(F)) { F = 0.0; ++n_bad; }
    const double t = F / n_total, t2 = t * t;
    s1 += t; s2 += t2;
    const bool contrib = have && t2 != 0.0;
    mf_hist_add<D>(hw, nb, packed, contrib, t2, lt_mask);
    qhead = (qhead + m) % CAP;
    qcount -= m;
  }
  mf_block_finish(s1, s2, n_pass, n_bad, s_hist, nh, nullptr, s_red, partial + (size_t)blockIdx.x * row, pcount + 2 * blockIdx.x);
}

// ---- staged iteration for the heavy processes: front end -> |M|^2 -> reductions, through HBM --------
// The fused kernels above run the front end (S1-S6) at the occupancy of the |M|^2 code (255 registers,
// 2 warps per scheduler), where it is latency-bound: 21 % of the fused kernel's time for 12 % of its
// FP64 instructions (profiles/r1_tuning.md).  The staged path gives every stage its own
// launch shape and passes 4N+3 doubles per PASSING event through HBM (1.0 GB written + 1.0 GB read per
// 1e7 events, ~0.3 ms at the measured 6.5 TB/s):
//   mf_front_kernel  one CTA per REGION of `cap` consecutive events: S1-S6 and the weight prefactor,
//                    ordered compaction (ballot + prefix over the warps) of the passing events into
//                    the region's record block rec[region][field][cap] (field-major: coalesced)
//   mf_me_kernel     persistent, one 256-thread CTA per SM: an exclusive prefix over the region counts
//                    maps a dense index over ALL passing events to (region, entry), so every lane of
//                    every warp carries a passing event through S7; writes F = pref |M|^2 in place
//   mf_hist_kernel   S9: sum t, sum t^2 and the d x nb histogram in fixed order from (F, packed bins)
// Field order of a record: k[N][4], sqrt(shat), pref (-> F), packed bins (6 bits per dimension), observable slots,
// packed bins of dimensions 10.. (classic 4n-random RAMBO only, CL = 1; otherwise never touched).
#define MF_REC_FIELDS(N) (4 * (N) + 5)
#ifndef MF_FRONT_MINB
#define MF_FRONT_MINB 3              // resident CTAs per SM the front end is compiled for (80 registers; tuned, profiles/r1_tuning.md)
#endif
template <int PROC, int CL>
__global__ void __launch_bounds__(MF_THREADS, MF_FRONT_MINB)
mf_front_kernel(const MfParams P, const double* __restrict__ g_edges, const double* __restrict__ g_pdf,
                uint32_t iteration, unsigned long long first, unsigned long long n, unsigned long long cap,
                double* __restrict__ rec, unsigned int* __restrict__ count) {
  constexpr int D = MfDim<PROC, CL>::D, N = MfProc<PROC>::N, NF = MF_REC_FIELDS(N), T = MF_THREADS;
  extern __shared__ double smem[];
  double* s_edges = smem;
  double* s_pdf = s_edges + D * (P.nb + 1);
  int* s_wtot = (int*)(s_pdf + P.pdf_smem);             // [T/32]
  mf_stage_tables(P, g_edges, g_pdf, s_edges, s_pdf);
  __syncthreads();
  const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  const unsigned long long lo = (unsigned long long)blockIdx.x * cap;
  const unsigned long long hi = lo + cap < n ? lo + cap : n;
  double* R = rec + (size_t)blockIdx.x * NF * cap;
  unsigned filled = 0;                                   // block-uniform
  for (unsigned long long base = lo; base < hi; base += T) {
    const unsigned long long i = base + tid;
    bool pass = false;
    int bin[D];
    double k[N][4], rts, pref;
    unsigned okeys = 0;
    if (i < hi) pass = mf_event_front<PROC, false, CL>(P, s_edges, s_pdf, iteration, first + i, bin, k, rts, pref, nullptr, &okeys);
    const unsigned bal = __ballot_sync(0xffffffffu, pass);
    if (lane == 0) s_wtot[warp] = __popc(bal);
    __syncthreads();
    unsigned before = 0, tot = 0;
#pragma unroll
    for (int w = 0; w < T / 32; ++w) { const unsigned c = s_wtot[w]; before += (w < (int)warp) ? c : 0u; tot += c; }
    if (pass) {
      const size_t slot = filled + before + __popc(bal & lt_mask);
#pragma unroll
      for (int p = 0; p < N; ++p)
#pragma unroll
        for (int c = 0; c < 4; ++c) R[(size_t)(4 * p + c) * cap + slot] = k[p][c];
      R[(size_t)(4 * N) * cap + slot] = rts;
      R[(size_t)(4 * N + 1) * cap + slot] = pref;
      unsigned long long packed, packed_hi;              // bins of 6 bits, 10 per word
      mf_pack_bins<D>(bin, packed, packed_hi);
      R[(size_t)(4 * N + 2) * cap + slot] = __longlong_as_double((long long)packed);
      if (P.n_obs > 0) R[(size_t)(4 * N + 3) * cap + slot] = __longlong_as_double((long long)okeys);
      if (D > MF_PACK_DIMS) R[(size_t)(4 * N + 4) * cap + slot] = __longlong_as_double((long long)packed_hi);
    }
    __syncthreads();
    filled += tot;
  }
  if (tid == 0) count[blockIdx.x] = filled;
}

#ifndef MF_ME_STAGGER
#define MF_ME_STAGGER 0              // cycles by which group g of the |M|^2 CTA starts late (measured: no effect, the groups drift apart by themselves)
#endif
#ifndef MF_ME_THREADS_F32
#define MF_ME_THREADS_F32 384        // CTA size of the fp32 variant (168 registers per thread; tuned, profiles/r1_tuning.md)
#endif
#define MF_TTG_SMEM 1                // gg -> tt~g |M|^2 stage: loop-entering values in shared memory (mf_me2_ttg_smem)
#ifndef MF_ME_THREADS
#define MF_ME_THREADS 256            // CTA size of the |M|^2 stage (one CTA per SM; registers = 65536 / threads)
#endif
// Real = double, or float: the fp32 variant of the |M|^2 stage (records, prefactor and F stay fp64)
template <int PROC, typename Real, int THREADS>
__global__ void __launch_bounds__(THREADS, 1)
mf_me_kernel(const MfParams P, double* __restrict__ rec, const unsigned int* __restrict__ count, int regions,
             unsigned long long cap) {
  constexpr int N = MfProc<PROC>::N, NF = MF_REC_FIELDS(N), T = THREADS;
  constexpr bool LANES = PROC == 3;                      // gg -> tt~gg: one event over four lanes (mf_me2_ttgg_group)
  constexpr bool SMEMOPS = PROC == 2 && MF_TTG_SMEM && std::is_same<Real, double>::value;   // gg -> tt~g: loop-entering values in shared memory
  extern __shared__ unsigned int s_pre[];                // [regions + 1] exclusive prefix, then s_part[T], then the lane tiles
  unsigned int* s_part = s_pre + regions + 1;
  const unsigned tid = threadIdx.x;
  {                                                      // block scan over the region counts
    const int per = (regions + T - 1) / T, a = tid * per, b = (a + per < regions) ? a + per : regions;
    unsigned s = 0;
    for (int r = a; r < b; ++r) s += count[r];
    s_part[tid] = s;
    __syncthreads();
    unsigned off = 0;
    for (unsigned t = 0; t < tid; ++t) off += s_part[t];
    for (int r = a; r < b; ++r) { s_pre[r] = off; off += count[r]; }
    if (tid == T - 1) s_pre[regions] = off;
    __syncthreads();
  }
  const unsigned M = s_pre[regions];
  // chunks of one GROUP (128 threads, own named barrier inside S7): the groups run out of phase, so that one
  // group's per-event prologue (record load, ingredients, reciprocals) overlaps the others' helicity loops
  constexpr unsigned G = MfProc<PROC>::GROUP < T ? MfProc<PROC>::GROUP : T, NG = T / G;
  static_assert(T % G == 0, "the CTA of the |M|^2 stage must be whole groups");
  constexpr unsigned EPC = LANES ? G / 4 : G;            // events per chunk of a group
  const unsigned group = tid / G, gtid = tid % G;
  const unsigned nchunks = (M + EPC - 1) / EPC;
  Real* tile = nullptr;
  if constexpr (LANES) tile = (Real*)(s_pre + ((regions + 1 + T + 1) & ~1)) + (size_t)(tid >> 5) * MF_LANES_TILE;
  if constexpr (SMEMOPS) tile = (Real*)(s_pre + ((regions + 1 + T + 1) & ~1)) + tid;
#if MF_ME_STAGGER > 0
  if (group > 0) { const long long t0 = clock64(); while (clock64() - t0 < (long long)MF_ME_STAGGER * group) { } }
#endif
  for (unsigned q = blockIdx.x * NG + group; q < nchunks; q += gridDim.x * NG) {   // group-uniform trips
    const unsigned lin = q * EPC + (LANES ? gtid >> 2 : gtid);
    const bool have = lin < M;
    const unsigned l = have ? lin : M - 1;               // lanes past the end recompute the last event
    int lo = 0, hi = regions;
    while (hi - lo > 1) { const int mid = (lo + hi) >> 1; if (s_pre[mid] <= l) lo = mid; else hi = mid; }
    double* R = rec + (size_t)lo * NF * cap + (l - s_pre[lo]);
    Real k[N][4];
#pragma unroll
    for (int p = 0; p < N; ++p)
#pragma unroll
      for (int c = 0; c < 4; ++c) k[p][c] = (Real)R[(size_t)(4 * p + c) * cap];
    const double rts = R[(size_t)(4 * N) * cap], pref = R[(size_t)(4 * N + 1) * cap];
    double F;                                            // S7, S8
    if constexpr (LANES) F = pref * (double)mf_me2_ttgg_group<Real>(P, (Real)rts, k, tile);
    else if constexpr (SMEMOPS) F = pref * (double)mf_me2_ttg_smem<Real, T>(P, (Real)rts, k, tile);
    else F = pref * (double)mf_me2<PROC, Real>(P, (Real)rts, k);
    if (have && (!LANES || (tid & 3u) == 0u)) R[(size_t)(4 * N + 1) * cap] = F;
  }
}

template <int PROC, int CL>
__global__ void __launch_bounds__(MF_THREADS)
mf_hist_kernel(const MfParams P, const double* __restrict__ rec, const unsigned int* __restrict__ count, int regions,
               unsigned long long cap, double n_total, double* __restrict__ partial,
               unsigned long long* __restrict__ pcount, int row) {
  constexpr int D = MfDim<PROC, CL>::D, N = MfProc<PROC>::N, NF = MF_REC_FIELDS(N), T = MF_THREADS;
  extern __shared__ double smem[];
  const int nb = P.nb, nh = D * nb, nw = T >> 5;
  double* s_hist = smem;                                 // [nw][D*nb]
  double* s_red = s_hist + nw * nh;                      // [nw][4]
  double* s_obs = s_red + nw * 4;                        // [nw][MF_OBS_ACC] when observables are set
  for (int i = threadIdx.x; i < nw * nh; i += T) s_hist[i] = 0.0;
  if (P.n_obs > 0) for (int i = threadIdx.x; i < nw * MF_OBS_ACC; i += T) s_obs[i] = 0.0;
  __syncthreads();
  const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const unsigned lt_mask = (1u << lane) - 1u;
  double* hw = s_hist + warp * nh;
  double s1 = 0.0, s2 = 0.0;
  unsigned long long n_pass = 0, n_bad = 0;
  for (int r = blockIdx.x; r < regions; r += gridDim.x) {
    const unsigned c = count[r];
    const double* R = rec + (size_t)r * NF * cap;
    for (unsigned e0 = warp * 32u; e0 < c; e0 += T) {    // warp-uniform trips
      const unsigned e = e0 + lane;
      const bool have = e < c;
      double F = have ? R[(size_t)(4 * N + 1) * cap + e] : 0.0;
      const unsigned long long packed = have ? (unsigned long long)__double_as_longlong(R[(size_t)(4 * N + 2) * cap + e]) : 0ull;
      if (have) ++n_pass;
      if (!isfinite(F)) { F = 0.0; ++n_bad; }            // A20
      const double t = F / n_total, t2 = t * t;          // O9
      s1 += t; s2 += t2;
      const bool contrib = have && t2 != 0.0;
      unsigned long long packed_hi = 0ull;
      if (D > MF_PACK_DIMS && have) packed_hi = (unsigned long long)__double_as_longlong(R[(size_t)(4 * N + 4) * cap + e]);
      mf_hist_add2<D>(hw, nb, packed, packed_hi, contrib, t2, lt_mask);
      if (P.n_obs > 0) {
        const unsigned okeys = have ? (unsigned)__double_as_longlong(R[(size_t)(4 * N + 3) * cap + e]) : 0u;
        mf_obs_add(s_obs + warp * MF_OBS_ACC, s_obs + warp * MF_OBS_ACC + MF_OBS_ACC / 2, P.n_obs, okeys, have && F != 0.0, t, t2, lt_mask);
      }
    }
  }
  mf_block_finish(s1, s2, n_pass, n_bad, s_hist, nh, P.n_obs > 0 ? s_obs : nullptr, s_red, partial + (size_t)blockIdx.x * row, pcount + 2 * blockIdx.x);
}

// ---- S1-S8 with per-event outputs -------------------------------------------------------------------
// front end of one event and its per-event records (everything but the weight and |M|^2)
template <int PROC, bool REC, int CL>
__device__ __forceinline__ bool mf_eval_front(const MfParams& P, const double* s_edges, const double* s_pdf, uint32_t iteration,
                                              unsigned long long ev, unsigned long long i, const MfEvalOutDev& o,
                                              double k[MfProc<PROC>::N][4], double& rts, double& pref, double* lum) {
  constexpr int D = MfDim<PROC, CL>::D, NL = 2 + MfProc<PROC>::N;
  int bin[D];
  MfEventRec rec;
  const bool pass = mf_event_front<PROC, REC, CL>(P, s_edges, s_pdf, iteration, ev, bin, k, rts, pref, REC ? &rec : nullptr, nullptr, lum);
  if (o.bins) {
#pragma unroll
    for (int j = 0; j < D; ++j) o.bins[i * D + j] = (uint8_t)bin[j];
  }
  if (o.pass) o.pass[i] = pass ? 1 : 0;
  if (REC) {
    if (o.x) {
#pragma unroll
      for (int j = 0; j < D; ++j) o.x[i * D + j] = rec.y[j];
    }
    if (o.momenta) {
#pragma unroll
      for (int l = 0; l < NL; ++l)
#pragma unroll
        for (int c = 0; c < 4; ++c) o.momenta[(i * NL + l) * 4 + c] = rec.mom[l][c];
    }
    if (o.pdf) { o.pdf[2 * i] = rec.pdf[0]; o.pdf[2 * i + 1] = rec.pdf[1]; }
  }
  return pass;
}

// The generator variants are grid-uniform run-time branches in and around the front end, so that the
// |M|^2 code is instantiated once per kernel.
template <int PROC, bool REC, typename T>
__global__ void __launch_bounds__(MF_THREADS, MfLaunch<PROC>::MINB)
mf_eval_kernel(const MfParams P, const double* __restrict__ g_edges, const double* __restrict__ g_pdf,
               uint32_t iteration, unsigned long long first, unsigned long long n, MfEvalOutDev o) {
  constexpr int N = MfProc<PROC>::N;
  extern __shared__ double smem[];
  double* s_edges = smem;
  double* s_pdf = s_edges + P.d * (P.nb + 1);
  [[maybe_unused]] double* tile = s_pdf + P.pdf_smem + (size_t)(threadIdx.x >> 5) * (PROC == 3 ? MF_LANES_TILE : 0);   // lane tiles of gg -> tt~gg
  mf_stage_tables(P, g_edges, g_pdf, s_edges, s_pdf);
  __syncthreads();
  const unsigned long long stride = (unsigned long long)gridDim.x * blockDim.x;
  for (unsigned long long base = (unsigned long long)blockIdx.x * blockDim.x; base < n; base += stride) {
    unsigned long long i = base + threadIdx.x;           // block-uniform trip count (barriers inside the event)
    if (i >= n) { if (!MF_UNIFORM_ME) break; i = n - 1; }   // tail lanes recompute event n-1 (same values written)
    double k[N][4], rts, pref, lum[MF_NLUM] = {0.0, 0.0, 0.0, 0.0};
    bool pass;
    if (PROC != 0 && (P.gen & MFD_GEN_CLASSIC)) pass = mf_eval_front<PROC, REC, PROC != 0 ? 1 : 0>(P, s_edges, s_pdf, iteration, first + i, i, o, k, rts, pref, lum);
    else pass = mf_eval_front<PROC, REC, PROC != 0 ? 2 : 0>(P, s_edges, s_pdf, iteration, first + i, i, o, k, rts, pref, lum);
    double me2 = 0.0;
    if (MF_UNIFORM_ME || pass) {                         // S7 (in the real type T)
      T kt[N][4];
#pragma unroll
      for (int p = 0; p < N; ++p)
#pragma unroll
        for (int c = 0; c < 4; ++c) kt[p][c] = (T)k[p][c];
      if constexpr (PROC == 3) me2 = (double)mf_me2_ttgg_warp32<T>(P, (T)rts, kt, (T*)tile);   // all 32 lanes (barriers inside)
      else me2 = (double)mf_me2_lum<PROC, T>(P, (T)rts, kt, lum);
    }
    if (!pass) me2 = 0.0;
    double F = pass ? pref * me2 : 0.0;                  // S8
    if (!isfinite(F)) F = 0.0;
    if (o.weight) o.weight[i] = F;
    if (REC && o.me2) o.me2[i] = MfChannels<PROC>::value > 1 ? me2 / (lum[0] + lum[1] + lum[2] + lum[3]) : me2;   // several channels: luminosity-weighted mean
  }
}


#ifndef MF_COMPACT
#define MF_COMPACT 1                 // CTA-level compaction of passing events for the processes with cuts
#endif
static constexpr bool kFused = MF_PROC != 3;         // gg -> tt~gg iterates on the staged path only (four lanes per event in its |M|^2 stage)
static constexpr bool kCompact = MF_COMPACT && MfHeavy<MF_PROC>::value && kFused;
static constexpr size_t kTileBytes = MF_PROC == 3 ? sizeof(double) * (MF_THREADS / 32) * MF_LANES_TILE : 0;   // eval kernel: lane tiles
static constexpr bool kEvalOne = MfHeavy<MF_PROC>::value;
static constexpr bool kF32 = MF_PROC == 2;   // fp32 variant of the |M|^2 stage: gg -> tt~g only (BASELINE configs[4])
// classic 4n-random RAMBO: processes 1-3; the heavy ones on the staged path only
static constexpr int kCL = MF_PROC != 0 ? 1 : 0;    // front-end instance of the classic RAMBO (mf_event.cuh MfDim)
static constexpr int kLT = MF_PROC != 0 ? 2 : 0;    // ... of the configs' RAMBO with the selectable tau map
// f(std::integral_constant<int, G>) with the front-end instance G the run's generator flags select (0 = the configs'
// generators: the instance without any run-time branch), resp. with the instance that fixes the VEGAS dimensions only
// (the reduction stage does not care about the tau map)
template <typename F>
static cudaError_t with_generator(const MfParams& P, F&& f) {
  if (kCL && (P.gen & MFD_GEN_CLASSIC)) return f(std::integral_constant<int, kCL>{});
  if (kLT && (P.gen & MFD_GEN_LINEAR)) return f(std::integral_constant<int, kLT>{});
  return f(std::integral_constant<int, 0>{});
}
template <typename F>
static cudaError_t with_dimensions(const MfParams& P, F&& f) {
  if (kCL && (P.gen & MFD_GEN_CLASSIC)) return f(std::integral_constant<int, kCL>{});
  return f(std::integral_constant<int, 0>{});
}

static cudaError_t proc_setup(const MfParams& P, size_t* smem_iter, size_t* smem_eval, int* occ_iter, int* occ_eval) {
  const size_t tables = (size_t)P.d * (P.nb + 1) + (size_t)P.pdf_smem;
  const size_t nw = MF_THREADS / 32;
  *smem_eval = sizeof(double) * tables + kTileBytes;
  *smem_iter = sizeof(double) * (tables + nw * P.d * P.nb + nw * 4);
  if (kCompact) *smem_iter += sizeof(double) * (4 * MfProc<MF_PROC>::N + 3) * 2 * MF_THREADS + sizeof(int) * nw;
  cudaError_t e;
#if MF_PROC == 3
  *smem_iter = 0; *occ_iter = 1; e = cudaSuccess;        // no fused kernel
#else
  if constexpr (kCompact) {
    e = cudaFuncSetAttribute(mf_iterate_compact_kernel<MF_PROC>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem_iter);
    if (e) return e;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_iter, mf_iterate_compact_kernel<MF_PROC>, MF_THREADS, *smem_iter);
  } else {
    const int smem_obs = (int)(*smem_iter + sizeof(double) * nw * MF_OBS_ACC);            // room for the observable histograms
    e = with_generator(P, [&](auto g) {
      constexpr int G = decltype(g)::value;
      const cudaError_t r = cudaFuncSetAttribute(mf_iterate_kernel<MF_PROC, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_obs);
      return r ? r : cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_iter, mf_iterate_kernel<MF_PROC, G>, MF_THREADS, *smem_iter);
    });
  }
#endif
  if (e) return e;
  if constexpr (!kEvalOne) {
    e = cudaFuncSetAttribute(mf_eval_kernel<MF_PROC, false, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem_eval);
    if (e) return e;
  }
  e = cudaFuncSetAttribute(mf_eval_kernel<MF_PROC, true, double>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem_eval);
  if (e) return e;
  if constexpr (kF32) {
    e = cudaFuncSetAttribute(mf_eval_kernel<MF_PROC, true, float>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)*smem_eval);
    if (e) return e;
  }
  return cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_eval, mf_eval_kernel<MF_PROC, true, double>, MF_THREADS, *smem_eval);
}
static cudaError_t proc_eval(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                             unsigned long long first, unsigned long long n, const MfEvalOutDev& o, bool rec,
                             bool f32, int grid, size_t smem, cudaStream_t st) {
  if (f32) {
    if constexpr (kF32) {
      mf_eval_kernel<MF_PROC, true, float><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, o);
      return cudaGetLastError();
    } else {
      return cudaErrorNotSupported;
    }
  }
  // heavy processes build one eval kernel only (the recording one: each output is written if requested)
  if constexpr (kEvalOne) mf_eval_kernel<MF_PROC, true, double><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, o);
  else if (rec) mf_eval_kernel<MF_PROC, true, double><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, o);
  else mf_eval_kernel<MF_PROC, false, double><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, o);
  return cudaGetLastError();
}

static cudaError_t proc_iterate(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                                unsigned long long first, unsigned long long n, double n_total, double* partial,
                                unsigned long long* pcount, int row, int grid, size_t smem, cudaStream_t st) {
  if (P.n_obs > 0) {
    if (kCompact) return cudaErrorNotSupported;          // observables of the heavy processes: staged path
    smem += sizeof(double) * (MF_THREADS / 32) * MF_OBS_ACC;
  }
#if MF_PROC == 3
  return cudaErrorNotSupported;
#else
  if constexpr (kCompact) {
    if (P.gen != 0) return cudaErrorNotSupported;        // generator variants of the heavy processes: staged path
    mf_iterate_compact_kernel<MF_PROC><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, n_total, partial, pcount, row);
    return cudaGetLastError();
  } else {
    return with_generator(P, [&](auto g) {
      mf_iterate_kernel<MF_PROC, decltype(g)::value><<<grid, MF_THREADS, smem, st>>>(P, edges, pdf, iteration, first, n, n_total, partial, pcount, row);
      return cudaGetLastError();
    });
  }
#endif
}

// ---- staged path: launches ---------------------------------------------------------------------------
#ifndef MF_STAGED
#define MF_STAGED 1                  // heavy processes (with cuts) iterate through the staged path
#endif
static constexpr bool kStaged = MF_STAGED && MfHeavy<MF_PROC>::value;
static constexpr int kRecFields = MF_REC_FIELDS(MfProc<MF_PROC>::N);

static size_t front_smem(const MfParams& P) {
  return sizeof(double) * ((size_t)P.d * (P.nb + 1) + (size_t)P.pdf_smem) + sizeof(int) * (MF_THREADS / 32);
}
static size_t hist_smem(const MfParams& P) {
  return sizeof(double) * (MF_THREADS / 32) * ((size_t)P.d * P.nb + 4 + (P.n_obs > 0 ? MF_OBS_ACC : 0));
}

static size_t me_tile_bytes(int threads) {
  if (MF_PROC == 3) return sizeof(double) * (threads / 32) * MF_LANES_TILE + 8;
  if (MF_PROC == 2 && MF_TTG_SMEM) return sizeof(double) * MF_ME2_GG_TTG_NW * threads + 8;
  return 0;
}
static cudaError_t proc_staged_setup(const MfParams& P, int* rec_fields, int* occ_front, int* occ_hist) {
  *rec_fields = kStaged ? kRecFields : 0;
  *occ_front = *occ_hist = 0;
  if constexpr (!kStaged) return cudaSuccess;
  else {
  cudaError_t e = with_generator(P, [&](auto g) {
    constexpr int G = decltype(g)::value;
    const cudaError_t r = cudaFuncSetAttribute(mf_front_kernel<MF_PROC, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)front_smem(P));
    return r ? r : cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_front, mf_front_kernel<MF_PROC, G>, MF_THREADS, front_smem(P));
  });
  if (e) return e;
  {                                                      // region prefix (<= 32 KB) + tiles, capped at the 227 KB an sm_100 CTA can opt in to
    const int want = 32 * 1024 + (int)me_tile_bytes(MF_ME_THREADS), cap = 227 * 1024;
    e = cudaFuncSetAttribute(mf_me_kernel<MF_PROC, double, MF_ME_THREADS>, cudaFuncAttributeMaxDynamicSharedMemorySize, want < cap ? want : cap);
  }
  if (e) return e;
  if constexpr (kF32) {
    e = cudaFuncSetAttribute(mf_me_kernel<MF_PROC, float, MF_ME_THREADS_F32>, cudaFuncAttributeMaxDynamicSharedMemorySize, 64 * 1024);
    if (e) return e;
  }
  const int smem_hist = (int)(hist_smem(P) + sizeof(double) * (MF_THREADS / 32) * MF_OBS_ACC);
  return with_dimensions(P, [&](auto g) {
    constexpr int G = decltype(g)::value;
    const cudaError_t r = cudaFuncSetAttribute(mf_hist_kernel<MF_PROC, G>, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_hist);
    return r ? r : cudaOccupancyMaxActiveBlocksPerMultiprocessor(occ_hist, mf_hist_kernel<MF_PROC, G>, MF_THREADS, hist_smem(P));
  });
  }
}

// ev (nullable): 4 events recorded at front start / |M|^2 start / |M|^2 end / reductions end
static cudaError_t proc_staged(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                               unsigned long long first, unsigned long long n, double n_total, const MfStageWs& ws,
                               double* partial, unsigned long long* pcount, int row, int grid_me, int grid_hist,
                               bool f32, cudaStream_t st, cudaEvent_t* ev) {
  if constexpr (!kStaged) return cudaErrorNotSupported;
  else {
  cudaError_t e;
  if (ev && (e = cudaEventRecord(ev[0], st))) return e;
  e = with_generator(P, [&](auto g) {
    mf_front_kernel<MF_PROC, decltype(g)::value><<<ws.regions, MF_THREADS, front_smem(P), st>>>(P, edges, pdf, iteration, first, n, ws.cap, ws.rec, ws.count);
    return cudaGetLastError();
  });
  if (e) return e;
  if (ev && (e = cudaEventRecord(ev[1], st))) return e;
  const size_t sm = sizeof(unsigned int) * ((size_t)ws.regions + 1 + (f32 ? MF_ME_THREADS_F32 : MF_ME_THREADS)) + (f32 ? 0 : me_tile_bytes(MF_ME_THREADS));   // (the fp32 variant keeps its operands in registers)
  if (f32) {
    if constexpr (kF32) mf_me_kernel<MF_PROC, float, MF_ME_THREADS_F32><<<grid_me, MF_ME_THREADS_F32, sm, st>>>(P, ws.rec, ws.count, ws.regions, ws.cap);
    else return cudaErrorNotSupported;
  } else {
    mf_me_kernel<MF_PROC, double, MF_ME_THREADS><<<grid_me, MF_ME_THREADS, sm, st>>>(P, ws.rec, ws.count, ws.regions, ws.cap);
  }
  if ((e = cudaGetLastError())) return e;
  if (ev && (e = cudaEventRecord(ev[2], st))) return e;
  e = with_dimensions(P, [&](auto g) {
    mf_hist_kernel<MF_PROC, decltype(g)::value><<<grid_hist, MF_THREADS, hist_smem(P), st>>>(P, ws.rec, ws.count, ws.regions, ws.cap, n_total, partial, pcount, row);
    return cudaGetLastError();
  });
  if (e) return e;
  if (ev && (e = cudaEventRecord(ev[3], st))) return e;
  return cudaSuccess;
  }
}

#define MF_CAT_(a, b) a##b
#define MF_CAT(a, b) MF_CAT_(a, b)
extern const MfProcOps MF_CAT(mf_ops_, MF_PROC) = {proc_setup, proc_eval, proc_iterate, proc_staged_setup, proc_staged};
