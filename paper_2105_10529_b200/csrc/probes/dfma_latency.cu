// dfma_latency.cu -- DFMA issue/latency probe behind DESIGN.md section 5.2 (fp64 roofline peak).
// nvcc -gencode arch=compute_100a,code=sm_100a -O3 -o dfma_latency dfma_latency.cu && ./dfma_latency
#include <cstdio>
#include <cuda_runtime.h>
template <int C>
__global__ void k(double* out, int iters, double a, double b) {
  double x[C];
  for (int c = 0; c < C; ++c) x[c] = threadIdx.x * 1e-3 + c;
  for (int i = 0; i < iters; ++i) {
#pragma unroll
    for (int u = 0; u < 8; ++u)
#pragma unroll
      for (int c = 0; c < C; ++c) x[c] = fma(x[c], a, b);
  }
  double s = 0; for (int c = 0; c < C; ++c) s += x[c];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}
template <int C> void run(int threads, double* d) {
  int iters = 20000; cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
  k<C><<<148, threads>>>(d, 100, 0.999, 1e-3); cudaDeviceSynchronize();
  cudaEventRecord(a); k<C><<<148, threads>>>(d, iters, 0.999, 1e-3); cudaEventRecord(b); cudaEventSynchronize(b);
  float ms; cudaEventElapsedTime(&ms, a, b);
  int dev; cudaGetDevice(&dev); int khz; cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, dev);
  double cyc = ms * 1e-3 * khz * 1e3;            // at max clock (approx)
  double per_smsp_instr = (double)iters * 8 * C * (threads / 32) / 4.0;   // warp-instrs per SMSP
  printf("chains %d warps/SMSP %.2f : %.2f cycles per DFMA warp-instr per SMSP (%.1f TFLOPs)\n", C, threads / 128.0, cyc / per_smsp_instr,
         2.0 * iters * 8 * C * threads * 148 / (ms * 1e-3) / 1e12);
}
int main() {
  double* d; cudaMalloc(&d, 148 * 1024 * 8);
  run<1>(128, d); run<2>(128, d); run<4>(128, d); run<8>(128, d); run<16>(128, d);
  run<1>(256, d); run<2>(256, d); run<4>(256, d); run<8>(256, d);
  run<1>(512, d); run<2>(512, d); run<4>(512, d);
  return 0;
}
