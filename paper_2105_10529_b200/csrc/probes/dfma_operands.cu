// probe: DFMA throughput with distinct register operands (vs the constant-operand peak kernel)
#include <cstdio>
#include <cuda_runtime.h>
template <int MODE>
__global__ void __launch_bounds__(256) k(double* out, const double* in, int iters) {
  double m[16], a[8];
#pragma unroll
  for (int i = 0; i < 16; ++i) m[i] = in[i * 256 + threadIdx.x];
#pragma unroll
  for (int i = 0; i < 8; ++i) a[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u)
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (MODE == 0) a[i] = fma(a[i], m[0], m[1]);                              // peak-kernel pattern
        if (MODE == 1) a[i] = fma(m[(i + u) & 15], m[(3 * i + u + 5) & 15], a[i]);   // sum-of-products chain
        if (MODE == 2) a[i] = fma(m[(i + u) & 15], a[(i + 3) & 7], a[i]);          // product with another chain
        if (MODE == 3) a[i] = fma(m[u & 15], m[(3 * i + u + 5) & 15], a[i]);        // one multiplicand shared by 8 consecutive DFMAs
        if (MODE == 4) a[i] = fma(m[(u + (i >> 1)) & 15], m[(3 * i + u + 5) & 15], a[i]);   // shared by pairs
      }
  }
  double s = 0; for (int i = 0; i < 8; ++i) s += a[i];
  out[blockIdx.x * 256 + threadIdx.x] = s;
}
template <int MODE> void run(double* o, double* in, int cta_per_sm) {
  int iters = 4000; cudaEvent_t a, b; cudaEventCreate(&a); cudaEventCreate(&b);
  k<MODE><<<148 * cta_per_sm, 256>>>(o, in, 10); cudaDeviceSynchronize();
  cudaEventRecord(a); k<MODE><<<148 * cta_per_sm, 256>>>(o, in, iters); cudaEventRecord(b); cudaEventSynchronize(b);
  float ms; cudaEventElapsedTime(&ms, a, b);
  printf("mode %d  CTAs/SM %d: %.2f TFLOP/s\n", MODE, cta_per_sm, 2.0 * iters * 128.0 * 256 * 148 * cta_per_sm / (ms * 1e-3) / 1e12);
}
int main() {
  double *o, *in; cudaMalloc(&o, 148 * 8 * 256 * 8); cudaMalloc(&in, 16 * 256 * 8); cudaMemset(in, 0, 16 * 256 * 8);
  for (int c : {1, 4}) { run<0>(o, in, c); run<1>(o, in, c); run<2>(o, in, c); run<3>(o, in, c); run<4>(o, in, c); }
  return 0;
}
