// tt_probe.cuh -- DFMA / FFMA issue-rate probe (diagnostic, not on the hot path).
// Gives the measured vector-ALU peak that DESIGN.md's "alu" roofline is checked against
// (derived peak: 148 SMs x 64 DFMA (128 FFMA) / clk / SM x 2 flop x SM clock).
#pragma once
#include <cuda_runtime.h>

namespace ttp {

template <typename T>
__global__ void __launch_bounds__(256) k_fma_probe(T* __restrict__ out, int iters, T a, T b) {
  T x[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) x[i] = (T)(threadIdx.x + i);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r)
#pragma unroll
      for (int i = 0; i < 8; ++i) x[i] = fma(x[i], a, b);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 8; ++i) s += x[i];
  if (s == (T)123456789) out[0] = s;  // never true in practice; keeps the chain alive
}

// returns TFLOP/s (FMA = 2 flop) or a negative value on error
template <typename T>
inline double fma_tflops(cudaStream_t st) {
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -1.0;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1.0;
  T* d = nullptr;
  if (cudaMalloc(&d, sizeof(T)) != cudaSuccess) return -1.0;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const int iters = 4096, blocks = sms * 8, threads = 256;
  double best = -1.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_fma_probe<T><<<blocks, threads, 0, st>>>(d, iters, (T)1.0000001, (T)1e-9);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flop = 2.0 * 64.0 * iters * (double)blocks * threads;
    const double tf = flop / (ms * 1e-3) / 1e12;
    if (rep > 0 && tf > best) best = tf;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) return -1.0;
  return best;
}

}  // namespace ttp
