// mf_proc.h -- host-side table of the per-process kernel launchers (mf_proc.cu, one object per process)
#pragma once
#include <cuda_runtime.h>
#include "mf_kernels.cuh"

// workspace of the staged path (mf_proc.cu): records of the passing events, [regions][fields][cap] doubles
struct MfStageWs { double* rec; unsigned int* count; unsigned long long cap; int regions; };

struct MfProcOps {
  cudaError_t (*setup)(const MfParams& P, size_t* smem_iter, size_t* smem_eval, int* occ_iter, int* occ_eval);
  cudaError_t (*eval)(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                      unsigned long long first, unsigned long long n, const MfEvalOutDev& o, bool rec, bool f32,
                      int grid, size_t smem, cudaStream_t st);
  cudaError_t (*iterate)(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                         unsigned long long first, unsigned long long n, double n_total, double* partial,
                         unsigned long long* pcount, int row, int grid, size_t smem, cudaStream_t st);
  // staged path; rec_fields = 0 when the process iterates with the fused kernel only
  cudaError_t (*staged_setup)(const MfParams& P, int* rec_fields, int* occ_front, int* occ_hist);
  cudaError_t (*staged)(const MfParams& P, const double* edges, const double* pdf, uint32_t iteration,
                        unsigned long long first, unsigned long long n, double n_total, const MfStageWs& ws,
                        double* partial, unsigned long long* pcount, int row, int grid_me, int grid_hist, bool f32,
                        cudaStream_t st, cudaEvent_t* ev);
};
extern const MfProcOps mf_ops_0, mf_ops_1, mf_ops_2, mf_ops_3, mf_ops_4, mf_ops_5, mf_ops_6, mf_ops_7;
static inline const MfProcOps* mf_proc_ops(int process) {
  static const MfProcOps* const ops[8] = {&mf_ops_0, &mf_ops_1, &mf_ops_2, &mf_ops_3, &mf_ops_4, &mf_ops_5, &mf_ops_6, &mf_ops_7};
  return ops[process];
}
