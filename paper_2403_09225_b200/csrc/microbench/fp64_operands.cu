// microbench: DFMA throughput when all three source operands are distinct, changing registers (register-file
// bandwidth / bank conflicts) vs. the x = fma(x, a, b) pattern with two loop-invariant operands.
#include <cstdio>
#include <cuda_runtime.h>
template <int KIND>
__global__ void k(double* out, int iters, double a, double b) {
  double x[8], y[8], z[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 1e-3 + i; y[i] = 1.0 + 1e-9 * (threadIdx.x + i); z[i] = 1e-9 * i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 4; ++u)
#pragma unroll
      for (int i = 0; i < 8; ++i) {
        if (KIND == 0) { x[i] = fma(x[i], a, b); }
        else if (KIND == 1) { x[i] = fma(y[(i + u) & 7], z[(i + 2 * u + 1) & 7], x[i]); }        // acc += y*z, 3 distinct
        else if (KIND == 2) { x[i] = fma(y[(i + u) & 7], z[(i + 2 * u + 1) & 7], x[(i + 3) & 7]); } // dest != any src
        else if (KIND == 3) { x[i] = y[(i + u) & 7] * z[(i + 2 * u + 1) & 7] + x[i] ; y[i] = x[(i+5)&7] + z[i]; } // + DADD
        else { x[i] = x[i] * y[(i+u)&7]; }  // DMUL 2 distinct
      }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i] + y[i] + z[i];
  if (s == 12345.678) out[0] = s;
}
template <int KIND>
void run(int warps_per_sm, int sms, double per_iter) {
  int iters = 4096;
  double* d; cudaMalloc(&d, 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int block = warps_per_sm * 32;
  k<KIND><<<sms, block>>>(d, 16, 1.0000001, 1e-9);
  cudaDeviceSynchronize();
  cudaEventRecord(e0);
  k<KIND><<<sms, block>>>(d, iters, 1.0000001, 1e-9);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double inst = (double)sms * warps_per_sm * 32 * iters * per_iter;
  printf("kind=%d warps/SM=%2d: %.3f ms  FP64 instr rate %.1f lanes/clk/SM (64 = peak)\n", KIND, warps_per_sm, ms, inst / (ms * 1e-3) / sms / 1.965e9);
  cudaFree(d);
}
int main() {
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  int sms = p.multiProcessorCount;
  for (int w : {4, 8, 12, 16}) {
    run<0>(w, sms, 32); run<1>(w, sms, 32); run<2>(w, sms, 32); run<3>(w, sms, 64); run<4>(w, sms, 32);
  }
  return 0;
}
