// microbench: does a non-FP64 instruction cost an issue cycle next to DFMA (FP64 pipe = 2 cycles/warp-instr)?
#include <cstdio>
#include <cuda_runtime.h>
template <int K, int KIND>
__global__ void k_mix(double* out, int iters, double a, double b, int ia) {
  double x[4];
  float f[4]; int n[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) { x[i] = threadIdx.x * 1e-3 + i; f[i] = threadIdx.x + i; n[i] = threadIdx.x * 3 + i; }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int u = 0; u < 16; ++u)
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        x[i] = fma(x[i], a, b);
#pragma unroll
        for (int k = 0; k < K; ++k) {
          if (KIND == 0) f[(i + k) & 3] = fmaf(f[(i + k) & 3], 1.0001f, 0.5f);
          else if (KIND == 1) n[(i + k) & 3] = n[(i + k) & 3] * ia + 7;
          else if (KIND == 2) n[(i + k) & 3] = (n[(i + k) & 3] ^ ia) + (n[(i+k+1)&3] & 0x55);
          else { float t = f[(i + k) & 3]; f[(i + k) & 3] = (n[(i+k)&3] & 1) ? t : f[(i+k+1)&3]; n[(i+k)&3] += ia; }
        }
      }
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 4; ++i) s += x[i] + f[i] + n[i];
  if (s == 12345.678) out[0] = s;
}
template <int K, int KIND>
void run(int warps_per_sm, int sms) {
  int iters = 2048;
  double* d; cudaMalloc(&d, 8);
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  int block = warps_per_sm * 32;
  k_mix<K, KIND><<<sms, block>>>(d, 16, 1.0000001, 1e-9, 3);
  cudaDeviceSynchronize();
  cudaEventRecord(e0);
  k_mix<K, KIND><<<sms, block>>>(d, iters, 1.0000001, 1e-9, 3);
  cudaEventRecord(e1); cudaEventSynchronize(e1);
  float ms; cudaEventElapsedTime(&ms, e0, e1);
  double inst = (double)sms * warps_per_sm * 32 * iters * 16.0 * 4;
  printf("kind=%d K=%d warps/SM=%2d: %.3f ms  DFMA rate %.1f /clk/SM\n", KIND, K, warps_per_sm, ms, inst / (ms * 1e-3) / sms / 1.965e9);
  cudaFree(d);
}
int main() {
  cudaDeviceProp p; cudaGetDeviceProperties(&p, 0);
  int sms = p.multiProcessorCount;
  for (int w : {8, 16}) {
    run<0, 0>(w, sms);
    run<1, 0>(w, sms); run<2, 0>(w, sms); run<3, 0>(w, sms);
    run<1, 1>(w, sms); run<2, 1>(w, sms);
    run<1, 2>(w, sms); run<2, 2>(w, sms);
    run<1, 3>(w, sms); run<2, 3>(w, sms);
  }
  return 0;
}
