// mf_noalloc.cu -- mf_reduce_weights_noalloc: S9 (sum t, sum t^2, d x n_bins histogram of t^2; reading O9) as ONE entry
// point that allocates nothing, for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
// harnesses that forbid it).  It is a variant of the reduction stage mf_hist_kernel (mf_proc.cu), whose scratch -- one
// partial record per CTA, summed in fixed order by a second kernel -- lives in device memory that mf_vegas_create allocates;
// here the same scratch is a file-scope static __device__ array of a stated maximum size:
//     MF_NA_MAX_BLOCKS (296) x MF_NA_ROW (2 + 18 x 64 = 1154) doubles = 2 732 672 bytes,
// held by every GPU that loads the library until the process exits.  With mf_integrand_eval (weights and bins into the
// caller's buffers), mf_set_accum_device and mf_vegas_finalize -- none of which allocates -- a caller can run whole
// iterations of any process without the on-demand record workspace of the staged mf_vegas_accumulate.
//
// In HOST code the array's name is a host-side stand-in, not a device address: its address is resolved once per device,
// with that device current, by cudaGetSymbolAddress (na_setup) and passed to the kernels.
// Every call shares the array, and it keeps the last call's contents: nothing in it has to start at zero, because every
// CTA of a call writes its whole partial record before the second kernel reads exactly the records of this call's grid.
// Calls that OVERLAP on the GPU (different streams, several host threads, several processes' contexts do not count: the
// array is per context) RACE on it: issue them on one stream or order them with events.
#include "../../include/madflow_b200.h"
#include <cuda_runtime.h>
#include <math.h>
#include <mutex>
#include <string>

int mf_fail_(int code, const char* msg);          // mf_api.cu: sets the calling thread's mf_last_error() text

#define MF_NA_THREADS 256
#define MF_NA_WARPS (MF_NA_THREADS / 32)
#define MF_NA_MAX_BLOCKS 296                      // two CTAs per SM of a B200
#define MF_NA_MAX_D 18                            // = MF_DMAX of mf_device.cuh (classic RAMBO of gg -> tt~gg)
#define MF_NA_MAX_NB 64                           // = MF_NBMAX
#define MF_NA_ROW (2 + MF_NA_MAX_D * MF_NA_MAX_NB)
#define MF_NA_MAX_DEVICES 64

static __device__ __align__(256) double mf_na_scratch[MF_NA_MAX_BLOCKS * MF_NA_ROW];

// partial record of one CTA: row = 2 + d*nb doubles at scratch + blockIdx.x * row.  Fixed summation order (reading A22):
// thread -> warp butterfly -> warps in index order; histogram: per-warp in shared memory, lanes that share a bin are
// served in lane order (same scheme as mf_hist_add in mf_proc.cu, with the dimension count at run time).
__global__ void __launch_bounds__(MF_NA_THREADS)
mf_na_hist_kernel(const double* __restrict__ weight, const uint8_t* __restrict__ bins, unsigned long long n, int d, int nb,
                  double n_total, double* __restrict__ scratch) {
  extern __shared__ double smem[];
  const int nh = d * nb, row = 2 + nh;
  double* s_hist = smem;                          // [MF_NA_WARPS][nh]
  double* s_red = s_hist + MF_NA_WARPS * nh;      // [MF_NA_WARPS][2]
  const unsigned tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const unsigned full = 0xffffffffu, lt_mask = (1u << lane) - 1u;
  for (int i = tid; i < MF_NA_WARPS * nh; i += MF_NA_THREADS) s_hist[i] = 0.0;
  __syncthreads();
  double* hw = s_hist + warp * nh;
  double s1 = 0.0, s2 = 0.0;
  const unsigned long long stride = (unsigned long long)gridDim.x * MF_NA_THREADS;
  for (unsigned long long base = (unsigned long long)blockIdx.x * MF_NA_THREADS; base < n; base += stride) {   // block-uniform trips
    const unsigned long long i = base + tid;
    const bool valid = i < n;
    double F = valid ? weight[i] : 0.0;
    if (!isfinite(F)) F = 0.0;                    // A20
    const double t = F / n_total, t2 = t * t;     // O9: t_i = F_i / N
    s1 += t; s2 += t2;
    const bool contrib = valid && t2 != 0.0;
    const unsigned cmask = __ballot_sync(full, contrib);
    if (cmask == 0u) continue;                    // warp-uniform
    for (int j = 0; j < d; ++j) {
      const unsigned key = contrib ? (unsigned)bins[i * d + j] : 0u;
      unsigned peers = cmask;
#pragma unroll
      for (int b = 0; b < 6; ++b) {
        const bool bit = (key >> b) & 1u;
        const unsigned bal = __ballot_sync(full, bit);
        peers &= bit ? bal : ~bal;
      }
      const unsigned rank = __popc(peers & lt_mask);
      for (unsigned r = 0; __any_sync(full, contrib && rank >= r); ++r) {
        if (contrib && rank == r) hw[j * nb + key] += t2;
        __syncwarp();
      }
    }
  }
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) { s1 += __shfl_xor_sync(full, s1, o); s2 += __shfl_xor_sync(full, s2, o); }
  if (lane == 0) { s_red[2 * warp] = s1; s_red[2 * warp + 1] = s2; }
  __syncthreads();
  double* out = scratch + (size_t)blockIdx.x * row;
  for (int e = tid; e < nh; e += MF_NA_THREADS) {
    double s = 0.0;
    for (int w = 0; w < MF_NA_WARPS; ++w) s += s_hist[w * nh + e];
    out[2 + e] = s;
  }
  if (tid == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < MF_NA_WARPS; ++w) { a += s_red[2 * w]; b += s_red[2 * w + 1]; }
    out[0] = a; out[1] = b;
  }
}

// acc[e] = (accumulate ? acc[e] : 0) + sum over this call's `grid` partial records, one warp per element, fixed order
__global__ void __launch_bounds__(256)
mf_na_reduce_kernel(const double* __restrict__ scratch, int grid, int row, double* __restrict__ acc, int accumulate) {
  const int e = blockIdx.x * 8 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
  if (e >= row) return;                           // warp-uniform
  double s = 0.0;
  for (int b = lane; b < grid; b += 32) s += scratch[(size_t)b * row + e];
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) s += __shfl_xor_sync(0xffffffffu, s, o);
  if (lane == 0) acc[e] = (accumulate ? acc[e] : 0.0) + s;
}

// ---- set-up, once per device, with that device current --------------------------------------------------------------
static std::mutex g_na_mutex;
static double* g_na_ptr[MF_NA_MAX_DEVICES];       // device address of mf_na_scratch on device i (nullptr: not resolved yet)

static int na_setup(int device, double** ptr) {
  std::lock_guard<std::mutex> lock(g_na_mutex);
  if (!g_na_ptr[device]) {
    void* p = nullptr;
    cudaError_t e = cudaGetSymbolAddress(&p, mf_na_scratch);
    if (e != cudaSuccess || !p) return mf_fail_(MF_ECUDA, (std::string("cudaGetSymbolAddress(mf_na_scratch): ") + cudaGetErrorString(e)).c_str());
    const int smem_max = (int)(sizeof(double) * (MF_NA_WARPS * (MF_NA_MAX_D * MF_NA_MAX_NB) + 2 * MF_NA_WARPS));   // 73 856 B
    e = cudaFuncSetAttribute(mf_na_hist_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, smem_max);
    if (e != cudaSuccess) return mf_fail_(MF_ECUDA, (std::string("cudaFuncSetAttribute(mf_na_hist_kernel): ") + cudaGetErrorString(e)).c_str());
    g_na_ptr[device] = (double*)p;
  }
  *ptr = g_na_ptr[device];
  return MF_OK;
}

extern "C" int mf_reduce_weights_noalloc(int32_t device, const double* dev_weight, const uint8_t* dev_bins, uint64_t n_events,
                                         uint32_t d, uint32_t n_bins, double n_total, int32_t accumulate, double* dev_acc,
                                         void* cuda_stream) {
  if (!dev_acc || (n_events > 0 && (!dev_weight || !dev_bins))) return mf_fail_(MF_EINVAL, "null argument");
  if (d < 1 || d > MF_NA_MAX_D || n_bins < 1 || n_bins > MF_NA_MAX_NB)
    return mf_fail_(MF_EINVAL, "mf_reduce_weights_noalloc: d must be in 1..18 and n_bins in 1..64 (the static scratch holds 296 records of 2 + 18 x 64 doubles)");
  if (!(n_total >= 1.0)) return mf_fail_(MF_EINVAL, "n_total must be >= 1");
  int ndev = 0;
  if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) return mf_fail_(MF_ECUDA, "no CUDA device (this library has no CPU path)");
  if (device < 0 || device >= ndev || device >= MF_NA_MAX_DEVICES) return mf_fail_(MF_EINVAL, "device ordinal out of range");
  int prev = -1;
  cudaError_t e = cudaGetDevice(&prev);
  if (e == cudaSuccess && prev != device) e = cudaSetDevice(device);
  if (e != cudaSuccess) return mf_fail_(MF_ECUDA, (std::string("cudaSetDevice: ") + cudaGetErrorString(e)).c_str());
  double* scratch = nullptr;
  int rc = na_setup(device, &scratch);
  if (rc == MF_OK) {
    cudaStream_t st = (cudaStream_t)cuda_stream;
    const int nh = (int)(d * n_bins), row = 2 + nh;
    const unsigned long long want = (n_events + MF_NA_THREADS - 1) / MF_NA_THREADS;
    const int grid = (int)(want < MF_NA_MAX_BLOCKS ? want : MF_NA_MAX_BLOCKS);
    if (grid > 0) {
      const size_t smem = sizeof(double) * ((size_t)MF_NA_WARPS * nh + 2 * MF_NA_WARPS);
      mf_na_hist_kernel<<<grid, MF_NA_THREADS, smem, st>>>(dev_weight, dev_bins, n_events, (int)d, (int)n_bins, n_total, scratch);
    }
    mf_na_reduce_kernel<<<(row + 7) / 8, 256, 0, st>>>(scratch, grid, row, dev_acc, accumulate);
    e = cudaGetLastError();
    if (e != cudaSuccess) rc = mf_fail_(MF_ECUDA, (std::string("mf_reduce_weights_noalloc launch: ") + cudaGetErrorString(e)).c_str());
  }
  if (prev >= 0 && prev != device) cudaSetDevice(prev);
  return rc;
}
