// mf_api.cu -- the C-ABI of include/madflow_b200.h: handle management and kernel launches.
// Host code only validates, allocates and enqueues; every step of the path runs in the kernels of
// mf_kernels.cuh.  No CPU fallback: without a device every compute call returns MF_ECUDA.
#include "../../include/madflow_b200.h"
#include "mf_small_kernels.cuh"
#include "mf_proc.h"
#include "mf_params.h"
#include <string>
#include <vector>
#include <new>
#include <cstring>
#include <cstdio>

static thread_local std::string g_err;
extern "C" const char* mf_last_error(void) { return g_err.c_str(); }

static int fail(int code, const std::string& msg) { g_err = msg; return code; }
int mf_fail_(int code, const char* msg) { return fail(code, msg); }      // for the other translation units of the library (mf_noalloc.cu)
#define MF_CUDA(call)                                                                              \
  do {                                                                                             \
    cudaError_t e_ = (call);                                                                       \
    if (e_ != cudaSuccess) return fail(MF_ECUDA, std::string(#call) + ": " + cudaGetErrorString(e_)); \
  } while (0)

// the caller's current device is restored when a call returns
struct MfDeviceGuard {
  int prev = -1; cudaError_t err;
  explicit MfDeviceGuard(int dev) { err = cudaGetDevice(&prev); if (err == cudaSuccess && prev != dev) err = cudaSetDevice(dev); else if (err == cudaSuccess) prev = -1; }
  ~MfDeviceGuard() { if (prev >= 0) cudaSetDevice(prev); }
};
#define MF_ON_DEVICE(h) MfDeviceGuard dev_guard_((h)->device); MF_CUDA(dev_guard_.err)
#define MF_STAGE_RING 256                  // staged launches whose stage times can be summed (mf_stage_ms_sum)

struct mf_vegas {
  mf_config_t cfg;
  MfParams P;
  int device, n_sm;
  int na;                              // 2 + d*nb
  int row;                             // na + MF_OBS_ACC: allocated length of a raw-sum record (observable sums behind)
  double* d_obs;                       // accumulated observable histograms [MF_OBS_ACC] + iterations summed
  size_t smem_iter, smem_eval;
  int occ_iter, occ_eval;              // resident blocks per SM of the two kernels
  uint32_t blocks_per_sm, threads;     // user override (0 = default)
  int max_blocks;
  double *d_edges, *d_pdf, *d_partial, *d_acc;
  unsigned long long *d_pcount, *d_counts;
  MfDevState* d_state;
  const MfProcOps* ops;               // per-process kernels (one translation unit each)
  uint32_t iteration;                  // iterations finalized so far (= Philox counter word 3)
  // stream ordering: state_stream = the stream of the last call that touched the integrator state (raw sums, grid, records),
  // ev_state = recorded behind it; ev_eval = behind the last mf_integrand_eval (which only reads the grid).  Calls on another
  // stream wait for the event they depend on; host reads synchronise on it.
  cudaStream_t state_stream;
  cudaEvent_t ev_state, ev_eval;
  bool have_state_ev, have_eval_ev;
  cudaEvent_t ev0, ev1, evk0, evk1;   // iteration start/end, fused-kernel start/end
  bool have_k, have_it;                // events recorded (fused kernel / whole iteration)
  // staged path (heavy processes): records of the passing events go through HBM between the stages
  int rec_fields, occ_front, occ_hist; // rec_fields = 0: the process has the fused path only
  bool use_staged, have_stage;
  bool f32;                            // cfg.precision == 32: |M|^2 stage in fp32 (staged path and eval only)
  MfStageWs ws;
  size_t ws_doubles, ws_regions;       // allocated sizes
  cudaEvent_t* evs;                    // front start / |M|^2 start / |M|^2 end / reductions end of the LAST staged launch (ring entry)
  cudaEvent_t ring[MF_STAGE_RING][4];  // one entry per staged launch (slices of a large iteration included)
  uint32_t ring_next, ring_count;      // next entry, entries recorded since the last mf_stage_ms_sum
  MfIterRec* h_rec;                    // pinned staging of one iteration record
};

// ---- stream ordering helpers ----------------------------------------------------------------------------
static int state_begin(mf_vegas* h, cudaStream_t st) {       // a call that reads or writes the integrator state on st
  if (h->have_state_ev && st != h->state_stream) MF_CUDA(cudaStreamWaitEvent(st, h->ev_state, 0));
  return MF_OK;
}
static int state_write_begin(mf_vegas* h, cudaStream_t st) { // ... that writes it: evals in flight read the grid
  int rc = state_begin(h, st);
  if (rc) return rc;
  if (h->have_eval_ev) MF_CUDA(cudaStreamWaitEvent(st, h->ev_eval, 0));
  return MF_OK;
}
static int state_end(mf_vegas* h, cudaStream_t st) {
  MF_CUDA(cudaEventRecord(h->ev_state, st));
  h->state_stream = st; h->have_state_ev = true;
  return MF_OK;
}
static int state_sync(mf_vegas* h, bool evals_too) {         // host access to the state
  if (h->have_state_ev) MF_CUDA(cudaEventSynchronize(h->ev_state));
  if (evals_too && h->have_eval_ev) MF_CUDA(cudaEventSynchronize(h->ev_eval));
  return MF_OK;
}
#define MF_STAGE_MAX_EVENTS (1ull << 24)   // events per staged launch (<= 2.1-2.6 GB of records)

extern "C" int mf_vegas_create(const mf_config_t* cfg, mf_vegas_t** out) {
  if (!out) return fail(MF_EINVAL, "out is NULL");
  *out = nullptr;
  MfParams P;
  std::string err;
  int rc = mf_fill_params(cfg, &P, err);
  if (rc) return fail(rc, err);
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0)
    return fail(MF_ECUDA, "no CUDA device (this library has no CPU path)");
  if (cfg->device < 0 || cfg->device >= ndev) return fail(MF_EINVAL, "device ordinal out of range");
  mf_vegas* h = new (std::nothrow) mf_vegas();
  if (!h) return fail(MF_ENOMEM, "host allocation failed");
  std::memset(h, 0, sizeof *h);
  h->cfg = *cfg; h->cfg.pdf_xf = nullptr; h->P = P; h->device = cfg->device;
  h->na = 2 + P.d * P.nb;
  h->row = h->na + MF_OBS_ACC;
#define MF_CREATE_CUDA(call)                                                     \
  do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { std::string m_ = std::string(#call) + ": " + cudaGetErrorString(e_); mf_vegas_destroy(h); return fail(MF_ECUDA, m_); } } while (0)
  MfDeviceGuard dev_guard_(h->device);
  MF_CREATE_CUDA(dev_guard_.err);
  MF_CREATE_CUDA(cudaDeviceGetAttribute(&h->n_sm, cudaDevAttrMultiProcessorCount, h->device));
  h->ops = mf_proc_ops(P.process);
  MF_CREATE_CUDA(h->ops->setup(P, &h->smem_iter, &h->smem_eval, &h->occ_iter, &h->occ_eval));
  if (h->occ_iter < 1 || h->occ_eval < 1) { mf_vegas_destroy(h); return fail(MF_ECUDA, "kernel does not fit on an SM"); }
  MF_CREATE_CUDA(h->ops->staged_setup(P, &h->rec_fields, &h->occ_front, &h->occ_hist));
  if (h->rec_fields && (h->occ_front < 1 || h->occ_hist < 1)) { mf_vegas_destroy(h); return fail(MF_ECUDA, "staged kernel does not fit on an SM"); }
  h->use_staged = h->rec_fields > 0;
  h->f32 = cfg->precision == 32;
  h->max_blocks = h->n_sm * 32;
  const bool flavours = cfg->process >= MF_QQ_TT;        // 11-flavour grid: its active rows (mf_flavour_slice)
  const size_t ne = (size_t)P.d * (P.nb + 1), npdf = (size_t)P.pdf_smem;
  MF_CREATE_CUDA(cudaMalloc(&h->d_edges, ne * sizeof(double)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_pdf, (npdf ? npdf : 1) * sizeof(double)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_partial, (size_t)h->max_blocks * h->row * sizeof(double)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_pcount, (size_t)h->max_blocks * 2 * sizeof(unsigned long long)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_acc, h->row * sizeof(double)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_counts, 2 * sizeof(unsigned long long)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_obs, (MF_OBS_ACC + 1) * sizeof(double)));
  MF_CREATE_CUDA(cudaMemset(h->d_obs, 0, (MF_OBS_ACC + 1) * sizeof(double)));
  MF_CREATE_CUDA(cudaMalloc(&h->d_state, sizeof(MfDevState)));
  MF_CREATE_CUDA(cudaMemset(h->d_state, 0, sizeof(MfDevState)));
  MF_CREATE_CUDA(cudaMemset(h->d_acc, 0, h->row * sizeof(double)));
  MF_CREATE_CUDA(cudaMemset(h->d_counts, 0, 2 * sizeof(unsigned long long)));
  std::vector<double> e(ne);
  for (int j = 0; j < P.d; ++j)
    for (int k = 0; k <= P.nb; ++k) e[(size_t)j * (P.nb + 1) + k] = (double)k / (double)P.nb;
  MF_CREATE_CUDA(cudaMemcpy(h->d_edges, e.data(), ne * sizeof(double), cudaMemcpyHostToDevice));
  if (flavours) {
    std::vector<double> t(npdf);
    mf_flavour_slice(P, cfg->pdf_xf, t.data());
    MF_CREATE_CUDA(cudaMemcpy(h->d_pdf, t.data(), npdf * sizeof(double), cudaMemcpyHostToDevice));
  } else if (npdf) MF_CREATE_CUDA(cudaMemcpy(h->d_pdf, cfg->pdf_xf, npdf * sizeof(double), cudaMemcpyHostToDevice));
  MF_CREATE_CUDA(cudaEventCreate(&h->ev0));
  MF_CREATE_CUDA(cudaEventCreate(&h->ev1));
  MF_CREATE_CUDA(cudaEventCreate(&h->evk0));
  MF_CREATE_CUDA(cudaEventCreate(&h->evk1));
  MF_CREATE_CUDA(cudaEventCreateWithFlags(&h->ev_state, cudaEventDisableTiming));
  MF_CREATE_CUDA(cudaEventCreateWithFlags(&h->ev_eval, cudaEventDisableTiming));
  for (int r = 0; r < MF_STAGE_RING; ++r)
    for (int i = 0; i < 4; ++i) MF_CREATE_CUDA(cudaEventCreate(&h->ring[r][i]));
  h->evs = h->ring[0];
  MF_CREATE_CUDA(cudaMallocHost(&h->h_rec, sizeof(MfIterRec)));
  *out = h;
  return MF_OK;
}

extern "C" int mf_vegas_destroy(mf_vegas_t* h) {
  if (!h) return MF_OK;
  MfDeviceGuard dev_guard_(h->device);
  cudaFree(h->d_edges); cudaFree(h->d_pdf); cudaFree(h->d_partial); cudaFree(h->d_pcount);
  cudaFree(h->d_acc); cudaFree(h->d_counts); cudaFree(h->d_state);
  cudaFree(h->ws.rec); cudaFree(h->ws.count); cudaFree(h->d_obs);
  for (int r = 0; r < MF_STAGE_RING; ++r)
    for (int i = 0; i < 4; ++i) if (h->ring[r][i]) cudaEventDestroy(h->ring[r][i]);
  if (h->ev_state) cudaEventDestroy(h->ev_state);
  if (h->ev_eval) cudaEventDestroy(h->ev_eval);
  if (h->h_rec) cudaFreeHost(h->h_rec);
  if (h->ev0) cudaEventDestroy(h->ev0);
  if (h->ev1) cudaEventDestroy(h->ev1);
  if (h->evk0) cudaEventDestroy(h->evk0);
  if (h->evk1) cudaEventDestroy(h->evk1);
  delete h;
  return MF_OK;
}

extern "C" int mf_ndim(const mf_vegas_t* h, uint32_t* d, uint32_t* n_final) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (d) *d = (uint32_t)h->P.d;
  if (n_final) *n_final = (uint32_t)h->P.n_final;
  return MF_OK;
}

extern "C" int mf_set_launch(mf_vegas_t* h, uint32_t blocks_per_sm, uint32_t threads_per_block) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (threads_per_block != 0 && threads_per_block != MF_THREADS)
    return fail(MF_EINVAL, "threads_per_block must be 0 or the built MF_THREADS (256)");
  if (blocks_per_sm > 32) return fail(MF_EINVAL, "blocks_per_sm must be <= 32");
  h->blocks_per_sm = blocks_per_sm; h->threads = threads_per_block;
  return MF_OK;
}

static inline int live_len(const mf_vegas* h) { return h->P.n_obs > 0 ? h->row : h->na; }   // live entries of a raw-sum record

static int grid_for(const mf_vegas* h, unsigned long long n, int occ) {
  const int per_sm = h->blocks_per_sm ? (int)h->blocks_per_sm : occ;
  unsigned long long want = (n + MF_THREADS - 1) / MF_THREADS;
  unsigned long long cap = (unsigned long long)h->n_sm * per_sm;     // whole waves of resident CTAs
  if (cap > (unsigned long long)h->max_blocks) cap = h->max_blocks;
  unsigned long long g = want < cap ? want : cap;
  return (int)(g ? g : 1);
}

extern "C" int mf_integrand_eval(mf_vegas_t* h, uint32_t iteration, uint64_t first_event, uint64_t n_events,
                                 const mf_eval_out_t* out, void* cuda_stream) {
  if (!h || !out) return fail(MF_EINVAL, "null argument");
  if (n_events == 0) return MF_OK;
  if (!out->weight && !out->x && !out->bins && !out->momenta && !out->me2 && !out->pdf && !out->pass)
    return fail(MF_EINVAL, "no output buffer requested");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  MfEvalOutDev o = {out->weight, out->x, out->bins, out->momenta, out->me2, out->pdf, out->pass};
  const bool rec = out->x || out->momenta || out->me2 || out->pdf;
  int rc = state_begin(h, st);                           // the grid may still be refined on another stream
  if (rc) return rc;
  MF_CUDA(h->ops->eval(h->P, h->d_edges, h->d_pdf, iteration, first_event, n_events, o, rec, h->f32,
                       grid_for(h, n_events, h->occ_eval), h->smem_eval, st));
  MF_CUDA(cudaEventRecord(h->ev_eval, st));
  h->have_eval_ev = true;
  return MF_OK;
}

extern "C" int mf_set_path(mf_vegas_t* h, int32_t staged) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (staged && !h->rec_fields) return fail(MF_EUNSUPPORTED, "this process has the fused path only");
  if (!staged && h->f32) return fail(MF_EUNSUPPORTED, "the fp32 |M|^2 variant runs on the staged path only");
  if (!staged && h->P.process == MF_GG_TTGG)
    return fail(MF_EUNSUPPORTED, "gg -> tt~gg runs on the staged path only (its |M|^2 stage spreads one event over four lanes)");
  if (!staged && h->rec_fields && h->P.gen != 0)
    return fail(MF_EUNSUPPORTED, "the selectable generators of processes 2 and 3 run on the staged path only");
  h->use_staged = staged != 0;
  return MF_OK;
}

// workspace of one staged launch of n events: regions of `cap` consecutive events (a multiple of the
// CTA size), about 4 front-end CTAs per resident slot so that the front-end grid fills whole waves
static int ensure_ws(mf_vegas* h, unsigned long long n) {
  const unsigned long long target = (unsigned long long)h->n_sm * h->occ_front * 4;
  unsigned long long cap = (n + target - 1) / target;
  cap = (cap + MF_THREADS - 1) / MF_THREADS * MF_THREADS;
  const unsigned long long regions = (n + cap - 1) / cap;
  const size_t need = (size_t)regions * h->rec_fields * cap;
  if (need > h->ws_doubles) {
    if (h->ws.rec) { MF_CUDA(cudaFree(h->ws.rec)); h->ws.rec = nullptr; h->ws_doubles = 0; }
    MF_CUDA(cudaMalloc(&h->ws.rec, need * sizeof(double)));
    h->ws_doubles = need;
  }
  if (regions > h->ws_regions) {
    if (h->ws.count) { MF_CUDA(cudaFree(h->ws.count)); h->ws.count = nullptr; h->ws_regions = 0; }
    MF_CUDA(cudaMalloc(&h->ws.count, regions * sizeof(unsigned int)));
    h->ws_regions = regions;
  }
  h->ws.cap = cap; h->ws.regions = (int)regions;
  return MF_OK;
}

extern "C" int mf_vegas_accumulate(mf_vegas_t* h, uint64_t first_event, uint64_t n_events, uint64_t n_total,
                                   void* cuda_stream) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (n_total < 2 || n_events > n_total || first_event > n_total - n_events)
    return fail(MF_EINVAL, "event range outside the iteration");
  if (n_events == 0) return MF_OK;
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  if (int rc0 = state_begin(h, st)) return rc0;
  if (h->use_staged) {
    for (uint64_t done = 0; done < n_events; done += MF_STAGE_MAX_EVENTS) {
      h->evs = h->ring[h->ring_next];                    // one event set per staged launch
      h->ring_next = (h->ring_next + 1) % MF_STAGE_RING;
      if (h->ring_count < MF_STAGE_RING) ++h->ring_count;
      const uint64_t m = n_events - done < MF_STAGE_MAX_EVENTS ? n_events - done : MF_STAGE_MAX_EVENTS;
      int rc = ensure_ws(h, m);
      if (rc) return rc;
      const int grid_me = h->n_sm;                        // one persistent CTA per SM (launch bounds of mf_me_kernel)
      int grid_hist = h->n_sm * h->occ_hist;
      if (grid_hist > h->ws.regions) grid_hist = h->ws.regions;
      if (grid_hist > h->max_blocks) grid_hist = h->max_blocks;
      MF_CUDA(h->ops->staged(h->P, h->d_edges, h->d_pdf, h->iteration, first_event + done, m, (double)n_total, h->ws,
                             h->d_partial, h->d_pcount, h->row, grid_me, grid_hist, h->f32, st, h->evs));
      mf_reduce_kernel<<<(live_len(h) + 2 + 7) / 8, MF_REDUCE_THREADS, 0, st>>>(h->d_partial, h->d_pcount, grid_hist, live_len(h), h->row, h->d_acc, h->d_counts);
      MF_CUDA(cudaGetLastError());
    }
    h->have_stage = true; h->have_k = false;
    return state_end(h, st);
  }
  const int grid = grid_for(h, n_events, h->occ_iter);
  MF_CUDA(cudaEventRecord(h->evk0, st));
  {
    cudaError_t e_ = h->ops->iterate(h->P, h->d_edges, h->d_pdf, h->iteration, first_event, n_events, (double)n_total,
                                     h->d_partial, h->d_pcount, h->row, grid, h->smem_iter, st);
    if (e_ == cudaErrorNotSupported) return fail(MF_EUNSUPPORTED, "observables and the selectable generators of processes 2 and 3 need the staged path");
    MF_CUDA(e_);
  }
  MF_CUDA(cudaEventRecord(h->evk1, st));
  h->have_k = true; h->have_stage = false;
  mf_reduce_kernel<<<(live_len(h) + 2 + 7) / 8, MF_REDUCE_THREADS, 0, st>>>(h->d_partial, h->d_pcount, grid, live_len(h), h->row, h->d_acc, h->d_counts);
  MF_CUDA(cudaGetLastError());
  return state_end(h, st);
}

// duration of the dominant kernel of the last accumulate: the fused kernel, or the |M|^2 stage
static int dominant_ms(mf_vegas* h, float* ms) {
  *ms = 0.0f;
  if (h->have_stage) MF_CUDA(cudaEventElapsedTime(ms, h->evs[1], h->evs[2]));
  else if (h->have_k) MF_CUDA(cudaEventElapsedTime(ms, h->evk0, h->evk1));
  return MF_OK;
}

// one iteration record: a single asynchronous copy on the caller's stream into pinned memory, one synchronisation
static int fetch_iter(mf_vegas* h, uint32_t idx, cudaStream_t st, mf_iter_t* o) {
  MF_CUDA(cudaMemcpyAsync(h->h_rec, &h->d_state->it[idx], sizeof(MfIterRec), cudaMemcpyDeviceToHost, st));
  MF_CUDA(cudaStreamSynchronize(st));
  o->integral = h->h_rec->I; o->sigma = h->h_rec->sig;
  o->n_events = h->h_rec->n; o->n_pass = h->h_rec->pass; o->n_nonfinite = h->h_rec->bad; o->kernel_ms = 0.0f;
  return MF_OK;
}

extern "C" int mf_vegas_finalize(mf_vegas_t* h, uint64_t n_total, void* cuda_stream, mf_iter_t* host_out) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (n_total < 2) return fail(MF_EINVAL, "an iteration needs at least 2 events");
  if (h->iteration >= MF_MAX_ITER) return fail(MF_ESTATE, "too many iterations (1024)");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = state_write_begin(h, st);
  if (rc) return rc;
  mf_finalize_kernel<<<1, 32 * h->P.d, 0, st>>>(h->P, h->cfg.alpha_damp, (double)n_total, n_total, h->d_acc, h->d_counts,
                                        h->d_edges, h->d_state, h->d_obs);
  MF_CUDA(cudaGetLastError());
  // the raw sums stay readable (mf_get_accum) until the next iteration starts
  const uint32_t idx = h->iteration++;
  if ((rc = state_end(h, st))) return rc;
  if (host_out) {
    if ((rc = fetch_iter(h, idx, st, host_out))) return rc;
    if ((rc = dominant_ms(h, &host_out->kernel_ms))) return rc;
  }
  return MF_OK;
}

static int zero_accum(mf_vegas* h, cudaStream_t st) {
  MF_CUDA(cudaMemsetAsync(h->d_acc, 0, live_len(h) * sizeof(double), st));
  MF_CUDA(cudaMemsetAsync(h->d_counts, 0, 2 * sizeof(unsigned long long), st));
  return MF_OK;
}

extern "C" int mf_vegas_iterate(mf_vegas_t* h, uint64_t n_events, void* cuda_stream, mf_iter_t* host_out) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (n_events < 2) return fail(MF_EINVAL, "an iteration needs at least 2 events");
  if (h->iteration >= MF_MAX_ITER) return fail(MF_ESTATE, "too many iterations (1024)");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = state_write_begin(h, st);
  if (rc) return rc;
  MF_CUDA(cudaEventRecord(h->ev0, st));
  if ((rc = zero_accum(h, st))) return rc;
  if ((rc = state_end(h, st))) return rc;
  if ((rc = mf_vegas_accumulate(h, 0, n_events, n_events, cuda_stream))) return rc;
  if ((rc = mf_vegas_finalize(h, n_events, cuda_stream, nullptr))) return rc;
  MF_CUDA(cudaEventRecord(h->ev1, st));
  h->have_it = true;
  if (host_out) {
    if ((rc = fetch_iter(h, h->iteration - 1, st, host_out))) return rc;
    if ((rc = dominant_ms(h, &host_out->kernel_ms))) return rc;
  }
  return MF_OK;
}

extern "C" int mf_last_stage_ms(const mf_vegas_t* h, float* ms3) {
  if (!h || !ms3) return fail(MF_EINVAL, "null argument");
  ms3[0] = ms3[1] = ms3[2] = 0.0f;
  if (!h->have_stage) return fail(MF_ESTATE, "the last accumulate did not run the staged path");
  MF_CUDA(cudaEventSynchronize(h->evs[3]));
  for (int i = 0; i < 3; ++i) MF_CUDA(cudaEventElapsedTime(&ms3[i], h->evs[i], h->evs[i + 1]));
  return MF_OK;
}

extern "C" int mf_stage_ms_sum(mf_vegas_t* h, float* ms3, uint32_t* launches) {
  if (!h || !ms3 || !launches) return fail(MF_EINVAL, "null argument");
  ms3[0] = ms3[1] = ms3[2] = 0.0f; *launches = 0;
  MF_ON_DEVICE(h);
  const uint32_t n = h->ring_count;
  for (uint32_t j = 0; j < n; ++j) {
    cudaEvent_t* e = h->ring[(h->ring_next + MF_STAGE_RING - 1 - j) % MF_STAGE_RING];
    MF_CUDA(cudaEventSynchronize(e[3]));
    for (int i = 0; i < 3; ++i) { float t = 0.0f; MF_CUDA(cudaEventElapsedTime(&t, e[i], e[i + 1])); ms3[i] += t; }
  }
  *launches = n;
  h->ring_count = 0;
  return MF_OK;
}

extern "C" int mf_last_kernel_ms(const mf_vegas_t* h, float* fused_kernel_ms, float* iteration_ms) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (fused_kernel_ms) {
    *fused_kernel_ms = 0.0f;
    if (h->have_stage) { MF_CUDA(cudaEventSynchronize(h->evs[2])); MF_CUDA(cudaEventElapsedTime(fused_kernel_ms, h->evs[1], h->evs[2])); }
    else if (h->have_k) { MF_CUDA(cudaEventSynchronize(h->evk1)); MF_CUDA(cudaEventElapsedTime(fused_kernel_ms, h->evk0, h->evk1)); }
  }
  if (iteration_ms) {
    *iteration_ms = 0.0f;
    if (h->have_it) { MF_CUDA(cudaEventSynchronize(h->ev1)); MF_CUDA(cudaEventElapsedTime(iteration_ms, h->ev0, h->ev1)); }
  }
  return MF_OK;
}

extern "C" int mf_get_accum(mf_vegas_t* h, double* host_acc, uint64_t* host_counts) {
  if (!h || !host_acc) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, false)) return rc;
  MF_CUDA(cudaMemcpy(host_acc, h->d_acc, live_len(h) * sizeof(double), cudaMemcpyDeviceToHost));
  if (host_counts) MF_CUDA(cudaMemcpy(host_counts, h->d_counts, 2 * sizeof(uint64_t), cudaMemcpyDeviceToHost));
  return MF_OK;
}

extern "C" int mf_set_accum(mf_vegas_t* h, const double* host_acc, const uint64_t* host_counts) {
  if (!h || !host_acc) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, false)) return rc;
  MF_CUDA(cudaMemcpy(h->d_acc, host_acc, live_len(h) * sizeof(double), cudaMemcpyHostToDevice));
  if (host_counts) MF_CUDA(cudaMemcpy(h->d_counts, host_counts, 2 * sizeof(uint64_t), cudaMemcpyHostToDevice));
  return MF_OK;
}

extern "C" int mf_zero_accum(mf_vegas_t* h, void* cuda_stream) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  int rc = state_begin(h, st);
  if (rc) return rc;
  if ((rc = zero_accum(h, st))) return rc;
  return state_end(h, st);
}

extern "C" int mf_get_accum_device(mf_vegas_t* h, double* dev_out, void* cuda_stream) {
  if (!h || !dev_out) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int n = live_len(h);
  if (int rc = state_begin(h, st)) return rc;
  mf_pack_accum_kernel<<<(n + 2 + 255) / 256, 256, 0, st>>>(h->d_acc, h->d_counts, n, dev_out);
  MF_CUDA(cudaGetLastError());
  return state_end(h, st);
}

extern "C" int mf_set_accum_device(mf_vegas_t* h, const double* dev_in, void* cuda_stream) {
  if (!h || !dev_in) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int n = live_len(h);
  if (int rc = state_begin(h, st)) return rc;
  mf_unpack_accum_kernel<<<(n + 2 + 255) / 256, 256, 0, st>>>(dev_in, n, h->d_acc, h->d_counts);
  MF_CUDA(cudaGetLastError());
  return state_end(h, st);
}

extern "C" int mf_set_observables(mf_vegas_t* h, const mf_observable_t* obs, uint32_t n_obs) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  if (n_obs > MF_MAX_OBS || (n_obs > 0 && !obs)) return fail(MF_EINVAL, "at most 4 observables");
  for (uint32_t o = 0; o < n_obs; ++o) {
    if (obs[o].kind < 0 || obs[o].kind > 3) return fail(MF_EINVAL, "unknown observable kind");
    if (obs[o].kind == MF_OBS_PT_3 && h->P.n_final < 3) return fail(MF_EINVAL, "this process has no third final particle");
    if (obs[o].n_bins < 1 || obs[o].n_bins > 62) return fail(MF_EINVAL, "observable n_bins must be in 1..62");
    if (!(obs[o].hi > obs[o].lo)) return fail(MF_EINVAL, "observable range is empty");
  }
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, true)) return rc;
  h->P.n_obs = (int32_t)n_obs;
  for (uint32_t o = 0; o < n_obs; ++o) {
    h->P.obs_kind[o] = obs[o].kind; h->P.obs_nb[o] = (int32_t)obs[o].n_bins; h->P.obs_lo[o] = obs[o].lo; h->P.obs_hi[o] = obs[o].hi;
  }
  MF_CUDA(cudaMemset(h->d_obs, 0, (MF_OBS_ACC + 1) * sizeof(double)));
  MF_CUDA(cudaMemset(h->d_acc, 0, h->row * sizeof(double)));
  return MF_OK;
}

extern "C" int mf_get_observables(mf_vegas_t* h, double* host_sum, double* host_sum2, uint32_t* n_iter) {
  if (!h || !host_sum || !host_sum2) return fail(MF_EINVAL, "null argument");
  if (h->P.n_obs == 0) return fail(MF_ESTATE, "no observables set");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, false)) return rc;
  const size_t n = (size_t)h->P.n_obs * MF_OBS_SLOTS;
  MF_CUDA(cudaMemcpy(host_sum, h->d_obs, n * sizeof(double), cudaMemcpyDeviceToHost));
  MF_CUDA(cudaMemcpy(host_sum2, h->d_obs + MF_OBS_ACC / 2, n * sizeof(double), cudaMemcpyDeviceToHost));
  double it = 0.0;
  MF_CUDA(cudaMemcpy(&it, h->d_obs + MF_OBS_ACC, sizeof(double), cudaMemcpyDeviceToHost));
  if (n_iter) *n_iter = (uint32_t)it;
  return MF_OK;
}

extern "C" int mf_accum_len(const mf_vegas_t* h, uint32_t* n) {
  if (!h || !n) return fail(MF_EINVAL, "null argument");
  *n = (uint32_t)live_len(h);
  return MF_OK;
}

extern "C" int mf_result(mf_vegas_t* h, mf_result_t* host_out) {
  if (!h || !host_out) return fail(MF_EINVAL, "null argument");
  if (h->iteration == 0) return fail(MF_ESTATE, "no iteration has been run");
  MF_ON_DEVICE(h);
  mf_combine_kernel<<<1, 32, 0, h->state_stream>>>(h->d_state);      // ordered behind the last finalize on its own stream
  MF_CUDA(cudaGetLastError());
  if (int rc = state_end(h, h->state_stream)) return rc;
  MF_CUDA(cudaStreamSynchronize(h->state_stream));
  double r[3];
  MF_CUDA(cudaMemcpy(r, &h->d_state->res_I, 3 * sizeof(double), cudaMemcpyDeviceToHost));
  host_out->integral = r[0]; host_out->sigma = r[1]; host_out->chi2_dof = r[2]; host_out->n_iter = h->iteration;
  return MF_OK;
}

extern "C" int mf_get_iterations(mf_vegas_t* h, mf_iter_t* host_out, uint32_t max_iter, uint32_t* n_iter) {
  if (!h || !host_out || !n_iter) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, false)) return rc;
  uint32_t n = h->iteration < max_iter ? h->iteration : max_iter;
  std::vector<MfIterRec> recs(n);
  if (n) MF_CUDA(cudaMemcpy(recs.data(), h->d_state->it, n * sizeof(MfIterRec), cudaMemcpyDeviceToHost));
  for (uint32_t i = 0; i < n; ++i) {
    host_out[i].integral = recs[i].I; host_out[i].sigma = recs[i].sig; host_out[i].n_events = recs[i].n;
    host_out[i].n_pass = recs[i].pass; host_out[i].n_nonfinite = recs[i].bad; host_out[i].kernel_ms = 0.0f;
  }
  *n_iter = n;
  return MF_OK;
}

extern "C" int mf_get_grid(mf_vegas_t* h, double* host_edges) {
  if (!h || !host_edges) return fail(MF_EINVAL, "null argument");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, false)) return rc;
  MF_CUDA(cudaMemcpy(host_edges, h->d_edges, (size_t)h->P.d * (h->P.nb + 1) * sizeof(double), cudaMemcpyDeviceToHost));
  return MF_OK;
}

extern "C" int mf_set_grid(mf_vegas_t* h, const double* e) {
  if (!h || !e) return fail(MF_EINVAL, "null argument");
  const int nb = h->P.nb;
  for (int j = 0; j < h->P.d; ++j) {
    const double* r = e + (size_t)j * (nb + 1);
    if (r[0] != 0.0 || r[nb] != 1.0) return fail(MF_EINVAL, "edges must start at 0 and end at 1");
    for (int k = 0; k < nb; ++k) if (!(r[k + 1] > r[k])) return fail(MF_EINVAL, "edges not increasing");
  }
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, true)) return rc;           // refinements and evaluations in flight use the old grid
  MF_CUDA(cudaMemcpy(h->d_edges, e, (size_t)h->P.d * (nb + 1) * sizeof(double), cudaMemcpyHostToDevice));
  return MF_OK;
}

// ---- checkpoint / resume of the integrator state (auxiliary; include/madflow_b200.h) ---------------------
struct MfStateHeader {
  uint32_t magic, version; int32_t process; uint32_t generator, d, n_bins, n_iter, n_obs; uint64_t seed;
};
#define MF_STATE_MAGIC 0x4d465354u      // "MFST"
static size_t state_bytes(const mf_vegas* h, uint32_t n_iter) {
  return sizeof(MfStateHeader) + sizeof(double) * ((size_t)h->P.d * (h->P.nb + 1) + MF_OBS_ACC + 1) + sizeof(MfIterRec) * (size_t)n_iter;
}

extern "C" int mf_state_size(const mf_vegas_t* h, uint64_t* bytes) {
  if (!h || !bytes) return fail(MF_EINVAL, "null argument");
  *bytes = state_bytes(h, h->iteration);
  return MF_OK;
}

extern "C" int mf_get_state(mf_vegas_t* h, void* host_buf, uint64_t bytes) {
  if (!h || !host_buf) return fail(MF_EINVAL, "null argument");
  if (bytes < state_bytes(h, h->iteration)) return fail(MF_EINVAL, "state buffer too small (mf_state_size)");
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, true)) return rc;
  MfStateHeader hd = {MF_STATE_MAGIC, 1u, h->P.process, (uint32_t)h->P.gen, (uint32_t)h->P.d, (uint32_t)h->P.nb, h->iteration, (uint32_t)h->P.n_obs, h->cfg.seed};
  char* p = (char*)host_buf;
  std::memcpy(p, &hd, sizeof hd); p += sizeof hd;
  const size_t ne = sizeof(double) * (size_t)h->P.d * (h->P.nb + 1), nr = sizeof(MfIterRec) * (size_t)h->iteration, no = sizeof(double) * (MF_OBS_ACC + 1);
  MF_CUDA(cudaMemcpy(p, h->d_edges, ne, cudaMemcpyDeviceToHost)); p += ne;
  if (nr) MF_CUDA(cudaMemcpy(p, h->d_state->it, nr, cudaMemcpyDeviceToHost));
  p += nr;
  MF_CUDA(cudaMemcpy(p, h->d_obs, no, cudaMemcpyDeviceToHost));
  return MF_OK;
}

extern "C" int mf_set_state(mf_vegas_t* h, const void* host_buf, uint64_t bytes) {
  if (!h || !host_buf) return fail(MF_EINVAL, "null argument");
  if (bytes < sizeof(MfStateHeader)) return fail(MF_EINVAL, "state buffer too small");
  MfStateHeader hd;
  std::memcpy(&hd, host_buf, sizeof hd);
  if (hd.magic != MF_STATE_MAGIC || hd.version != 1u) return fail(MF_EINVAL, "not a madflow_b200 state (magic / version)");
  if (hd.process != h->P.process || hd.generator != (uint32_t)h->P.gen || hd.d != (uint32_t)h->P.d || hd.n_bins != (uint32_t)h->P.nb || hd.seed != h->cfg.seed)
    return fail(MF_EINVAL, "state belongs to another configuration (process, generator, dimensions, bins or seed differ)");
  if (hd.n_obs != (uint32_t)h->P.n_obs) return fail(MF_EINVAL, "state was saved with another number of observables (call mf_set_observables first)");
  if (hd.n_iter > MF_MAX_ITER) return fail(MF_EINVAL, "corrupt state (iteration count)");
  if (bytes < state_bytes(h, hd.n_iter)) return fail(MF_EINVAL, "state buffer truncated");
  const size_t ne = sizeof(double) * (size_t)h->P.d * (h->P.nb + 1), nr = sizeof(MfIterRec) * (size_t)hd.n_iter, no = sizeof(double) * (MF_OBS_ACC + 1);
  const char* p = (const char*)host_buf + sizeof hd;
  {                                                       // the same validation as mf_set_grid
    std::vector<double> e((size_t)h->P.d * (h->P.nb + 1));
    std::memcpy(e.data(), p, ne);
    for (int j = 0; j < h->P.d; ++j) {
      const double* r = e.data() + (size_t)j * (h->P.nb + 1);
      if (r[0] != 0.0 || r[h->P.nb] != 1.0) return fail(MF_EINVAL, "corrupt state (grid edges)");
      for (int k = 0; k < h->P.nb; ++k) if (!(r[k + 1] > r[k])) return fail(MF_EINVAL, "corrupt state (grid edges)");
    }
  }
  MF_ON_DEVICE(h);
  if (int rc = state_sync(h, true)) return rc;
  MF_CUDA(cudaMemcpy(h->d_edges, p, ne, cudaMemcpyHostToDevice)); p += ne;
  if (nr) MF_CUDA(cudaMemcpy(h->d_state->it, p, nr, cudaMemcpyHostToDevice));
  p += nr;
  MF_CUDA(cudaMemcpy(&h->d_state->n_iter, &hd.n_iter, sizeof(unsigned int), cudaMemcpyHostToDevice));
  MF_CUDA(cudaMemcpy(h->d_obs, p, no, cudaMemcpyHostToDevice));
  h->iteration = hd.n_iter;                              // = the Philox counter word of the next iteration
  h->have_k = h->have_stage = h->have_it = false;
  return MF_OK;
}

extern "C" int mf_me_flops(const mf_vegas_t* h, uint64_t* n_add, uint64_t* n_mul, uint64_t* n_fma) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  static const uint64_t T[8][3] = {{MF_ME2_EE_MUMU_NADD, MF_ME2_EE_MUMU_NMUL, MF_ME2_EE_MUMU_NFMA},
                                   {MF_ME2_GG_TT_NADD, MF_ME2_GG_TT_NMUL, MF_ME2_GG_TT_NFMA},
                                   {MF_ME2_GG_TTG_NADD, MF_ME2_GG_TTG_NMUL, MF_ME2_GG_TTG_NFMA},
                                   {MF_ME2_GG_TTGG_NADD, MF_ME2_GG_TTGG_NMUL, MF_ME2_GG_TTGG_NFMA},
                                   {MF_ME2_EE_MUMU_NADD, MF_ME2_EE_MUMU_NMUL, MF_ME2_EE_MUMU_NFMA},    // q q~ -> t t~: the two-current code
                                   {MF_ME2_GG_TT_NADD + MF_ME2_EE_MUMU_NADD, MF_ME2_GG_TT_NMUL + MF_ME2_EE_MUMU_NMUL + 1,
                                    MF_ME2_GG_TT_NFMA + MF_ME2_EE_MUMU_NFMA + 1},    // p p -> t t~: both subprocesses + the luminosity-weighted sum (mul, fma)
                                   {2 * MF_ME2_QQ_TTG_NADD, 2 * MF_ME2_QQ_TTG_NMUL, 2 * MF_ME2_QQ_TTG_NFMA + 2},     // two channels (q q~, q~ q)
                                   {4 * MF_ME2_QG_TTQ_NADD, 4 * MF_ME2_QG_TTQ_NMUL, 4 * MF_ME2_QG_TTQ_NFMA + 4}};    // four channels
  // gg -> tt~g on the staged fp64 path runs the shared-memory-operand organisation (helicity loop over gluon leg 2 only): its own count
  static const uint64_t S2[3] = {MF_ME2_GG_TTG_S_NADD, MF_ME2_GG_TTG_S_NMUL, MF_ME2_GG_TTG_S_NFMA};
  const uint64_t* t = (h->P.process == MF_GG_TTG && h->use_staged && !h->f32) ? S2 : T[h->P.process];
  if (n_add) *n_add = t[0];
  if (n_mul) *n_mul = t[1];
  if (n_fma) *n_fma = t[2];
  return MF_OK;
}

extern "C" int mf_me_flops_bounds(const mf_vegas_t* h, uint64_t* flops_min, uint64_t* flops_executed) {
  if (!h) return fail(MF_EINVAL, "handle is NULL");
  uint64_t a, m, f;
  int rc = mf_me_flops(h, &a, &m, &f);
  if (rc) return rc;
  uint64_t lo = a + m + 2 * f, ex = lo;
  if (h->P.process == MF_GG_TTG) {
    lo = MF_ME2_GG_TTG_NFLOPS_MIN;
    if (h->use_staged && !h->f32) ex = MF_ME2_GG_TTG_S_NFLOPS_EMITTED;      // with the cheap loop invariants it recomputes per trip
  }
  if (h->P.process == MF_GG_TTGG) {
    lo = MF_ME2_GG_TTGG_NFLOPS_MIN;
    ex = 4ull * (MF_ME2_GG_TTGG_LANES_NADD + MF_ME2_GG_TTGG_LANES_NMUL + 2ull * MF_ME2_GG_TTGG_LANES_NFMA);
  }
  if (flops_min) *flops_min = lo;
  if (flops_executed) *flops_executed = ex;
  return MF_OK;
}

extern "C" int mf_fp64_peak(int32_t device, double seconds, double* host_flops_per_s) {
  if (!host_flops_per_s || !(seconds > 0.0)) return fail(MF_EINVAL, "bad argument");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) return fail(MF_ECUDA, "no such CUDA device");
  MfDeviceGuard dev_guard_(device);
  MF_CUDA(dev_guard_.err);
  int n_sm = 0;
  MF_CUDA(cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, device));
  const int grid = n_sm * 4, threads = 256, iters = 4096;
  struct Res {                                            // released on every return path
    double* d_out = nullptr; cudaEvent_t a = nullptr, b = nullptr;
    ~Res() { if (a) cudaEventDestroy(a); if (b) cudaEventDestroy(b); if (d_out) cudaFree(d_out); }
  } r;
  MF_CUDA(cudaMalloc(&r.d_out, (size_t)grid * threads * sizeof(double)));
  MF_CUDA(cudaEventCreate(&r.a)); MF_CUDA(cudaEventCreate(&r.b));
  mf_dfma_kernel<<<grid, threads>>>(r.d_out, iters, 0.999999, 1e-6);          // warm-up
  MF_CUDA(cudaDeviceSynchronize());
  const double flops_per_launch = 2.0 * MF_DFMA_PER_ITER * (double)iters * grid * threads;
  double best = 0.0, spent = 0.0;
  int reps = 0;
  while (spent < seconds * 1e3 && reps < 10000) {
    MF_CUDA(cudaEventRecord(r.a));
    mf_dfma_kernel<<<grid, threads>>>(r.d_out, iters, 0.999999, 1e-6);
    MF_CUDA(cudaEventRecord(r.b));
    MF_CUDA(cudaEventSynchronize(r.b));
    float ms = 0.0f;
    MF_CUDA(cudaEventElapsedTime(&ms, r.a, r.b));
    spent += ms; ++reps;
    const double f = flops_per_launch / (ms * 1e-3);
    if (f > best) best = f;
  }
  *host_flops_per_s = best;
  return MF_OK;
}
