// mf_proc_stub.cu -- placeholder ops table for a process left out of a tuning build (build.py only=...)
#include "mf_proc.h"
static cudaError_t s_setup(const MfParams&, size_t*, size_t*, int*, int*) { return cudaErrorNotSupported; }
static cudaError_t s_eval(const MfParams&, const double*, const double*, uint32_t, unsigned long long, unsigned long long,
                          const MfEvalOutDev&, bool, bool, int, size_t, cudaStream_t) { return cudaErrorNotSupported; }
static cudaError_t s_iter(const MfParams&, const double*, const double*, uint32_t, unsigned long long, unsigned long long,
                          double, double*, unsigned long long*, int, int, size_t, cudaStream_t) { return cudaErrorNotSupported; }
#define MF_CAT_(a, b) a##b
#define MF_CAT(a, b) MF_CAT_(a, b)
static cudaError_t s_ssetup(const MfParams&, int*, int*, int*) { return cudaErrorNotSupported; }
static cudaError_t s_staged(const MfParams&, const double*, const double*, uint32_t, unsigned long long, unsigned long long,
                            double, const MfStageWs&, double*, unsigned long long*, int, int, int, bool, cudaStream_t, cudaEvent_t*) {
  return cudaErrorNotSupported;
}
extern const MfProcOps MF_CAT(mf_ops_, MF_PROC) = {s_setup, s_eval, s_iter, s_ssetup, s_staged};
