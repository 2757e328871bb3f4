// mf_kernels.cuh -- launch shapes and the device-resident state shared by the CUDA kernels of the path
// (sm_100a).  The kernels themselves:
//   mf_proc.cu          mf_front_kernel / mf_me_kernel / mf_hist_kernel  staged S1-S6 / S7-S8 / S9 of the heavy
//                       processes (each stage at its own occupancy, records of the passing events through HBM)
//                       mf_iterate_kernel, mf_iterate_compact_kernel  S1-S9 fused: one event per thread in
//                       registers, persistent grid, per-warp shared-memory histograms
//                       mf_eval_kernel  S1-S8 with per-event outputs (the parity entry point mf_integrand_eval)
//   mf_small_kernels.cuh  mf_reduce_kernel (fixed-order sum of the per-block partials), mf_finalize_kernel
//                       (S10: I, sigma, grid refinement, iteration record), mf_combine_kernel (O11),
//                       mf_dfma_kernel (register-resident DFMA chains: the measured fp64 roofline peak)
// All reductions are fixed-order (no atomics): results are bit-reproducible for a fixed launch geometry
// (reading A22).  These are FP64-pipe-bound straight-line kernels (no dense contraction): no tensor cores,
// no TMA; the staged tables are the 2.9-4.1 KB of VEGAS edges and the 40 KB PDF table in shared memory.
#pragma once
#include <cuda_runtime.h>
#include "mf_event.cuh"

// Launch shape (tuned on B200, profiles/r1_tuning.md): one 256-thread CTA per SM for the heavy
// processes (255 registers/thread, 8 warps/SM) whose warps are kept on the same instruction-cache
// lines by the barrier points of the generated code (MF_SYNC_EVERY in mf_device.cuh).
#ifndef MF_THREADS
#define MF_THREADS 256
#endif
#define MF_MAX_ITER 1024
#ifndef MF_MINB_HEAVY
#define MF_MINB_HEAVY 1              // resident blocks per SM the heavy kernels (tt~g, tt~gg) are compiled for
#endif

template <int PROC> struct MfLaunch { static const int MINB = 512 / MF_THREADS; };
template <> struct MfLaunch<2> { static const int MINB = MF_MINB_HEAVY; };
template <> struct MfLaunch<3> { static const int MINB = MF_MINB_HEAVY; };
template <> struct MfLaunch<6> { static const int MINB = 1; };    // 3 400 straight-line operations per channel: all 255 registers
template <> struct MfLaunch<7> { static const int MINB = 1; };

struct MfEvalOutDev {
  double* weight; double* x; uint8_t* bins; double* momenta; double* me2; double* pdf; uint8_t* pass;
};

// device-resident integrator state that the kernels update
struct MfIterRec { double I, sig; unsigned long long n, pass, bad; };     // one iteration (read back with one copy)
struct MfDevState {
  MfIterRec it[MF_MAX_ITER];
  unsigned int n_iter;
  double res_I, res_sig, res_chi2;
};

