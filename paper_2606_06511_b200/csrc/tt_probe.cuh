// tt_probe.cuh -- DFMA / FFMA issue-rate probe and random-gather bandwidth probe (diagnostics, not on the hot path).
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

// ---- random-gather probe: what the memory system delivers for the access pattern of K1 / K6 -----------------------
// n_items random items of `item_doubles` consecutive doubles (3 = one vertex, 9 = the three vertices of a soup
// triangle) read from an array of `array_bytes` (larger than the L2), each thread one item, ids by a counter hash.
// Reports the USEFUL bytes per second (item size x items / time): the ceiling a gather kernel that touched nothing
// else and computed nothing would see -- sector granularity (a 24-byte vertex straddles two 32-byte sectors half of
// the time) and DRAM row locality included.
__device__ __forceinline__ unsigned long long probe_hash(unsigned long long z) {
  z = (z ^ (z >> 30)) * 0xbf58476d1ce4e5b9ull;
  z = (z ^ (z >> 27)) * 0x94d049bb133111ebull;
  return z ^ (z >> 31);
}
template <int ITEM>
__global__ void __launch_bounds__(256) k_gather_probe(const double* __restrict__ a, unsigned long long n_slots,
                                                      long long n_items, double* __restrict__ out) {
  const long long i = (long long)blockIdx.x * 256 + threadIdx.x;
  if (i >= n_items) return;
  const double* p = a + (size_t)ITEM * (size_t)(probe_hash((unsigned long long)i) % n_slots);
  double s = 0.0;
#pragma unroll
  for (int k = 0; k < ITEM; ++k) s += __ldg(p + k);
  if (s == 123456789.0) out[0] = s;  // never true: keeps the loads alive
}
// returns useful GB/s, or a negative value on error
template <int ITEM>
inline double gather_gbs(size_t array_bytes, long long n_items, cudaStream_t st) {
  double* a = nullptr;
  double* o = nullptr;
  if (cudaMalloc(&a, array_bytes) != cudaSuccess) { (void)cudaGetLastError(); return -1.0; }
  if (cudaMalloc(&o, sizeof(double)) != cudaSuccess) { cudaFree(a); (void)cudaGetLastError(); return -1.0; }
  cudaMemsetAsync(a, 0, array_bytes, st);
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0);
  cudaEventCreate(&e1);
  const unsigned long long n_slots = array_bytes / (sizeof(double) * ITEM);
  double best = -1.0;
  for (int rep = 0; rep < 4; ++rep) {
    cudaEventRecord(e0, st);
    k_gather_probe<ITEM><<<(unsigned)((n_items + 255) / 256), 256, 0, st>>>(a, n_slots, n_items, o);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) break;
    float ms = 0.f;
    cudaEventElapsedTime(&ms, e0, e1);
    const double gbs = (double)n_items * ITEM * sizeof(double) / (ms * 1e-3) / 1e9;
    if (rep > 0 && gbs > best) best = gbs;
  }
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  cudaFree(a);
  cudaFree(o);
  if (cudaGetLastError() != cudaSuccess) return -1.0;
  return best;
}

}  // namespace ttp
