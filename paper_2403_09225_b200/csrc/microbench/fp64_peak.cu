// microbench: DFMA throughput vs warps/SM and ILP; dependent-DFMA latency
#include <cstdio>
#include <cuda_runtime.h>
template <int ILP>
__global__ void k_dfma(double* out, int iters, double a, double b) {
  double x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; ++i) x[i] = threadIdx.x * 1e-3 + i;
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u)
#pragma unroll
      for (int i = 0; i < ILP; ++i) x[i] = fma(x[i], a, b);
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < ILP; ++i) s += x[i];
  if (s == 12345.678) out[0] = s;
}
template <int ILP>
void run(int warps_per_sm, int sms) {
  int iters = 4096;
  double* d; cudaMalloc(&d, 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int block = warps_per_sm * 32 > 1024 ? 1024 : warps_per_sm * 32;
  int bps = warps_per_sm * 32 / block;
  k_dfma<ILP><<<sms * bps, block>>>(d, 16, 1.0000001, 1e-9);
  cudaDeviceSynchronize();
  cudaEventRecord(e0);
  k_dfma<ILP><<<sms * bps, block>>>(d, iters, 1.0000001, 1e-9);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double inst = (double)sms * warps_per_sm * 32 * iters * 16.0 * ILP;
  printf("ILP=%d warps/SM=%2d: %.3f ms  %.2f TFMA/s  (%.1f FMA/clk/SM @1.965GHz)\n", ILP, warps_per_sm, ms, inst / ms / 1e9,
         inst / (ms * 1e-3) / sms / 1.965e9);
  cudaFree(d);
}
int main() {
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  int sms = p.multiProcessorCount;
  printf("%s SMs=%d\n", p.name, sms);
  for (int w : {4, 8, 12, 16, 32, 64}) { run<1>(w, sms); run<2>(w, sms); run<4>(w, sms); run<8>(w, sms); }
  return 0;
}
