// =====================================================================================
// gfcc_probe.cuh -- FP64 tensor-pipe (DMMA) issue-rate probe: the roofline denominator of the sigma GEMMs.
//
// MEASURED_PEAKS.json has no FP64 entry, so the library measures the ceiling of the instruction its GEMM
// engine is built on: every warp runs a register-only loop of independent mma.sync.m8n8k4.f64 chains
// (no memory traffic), all SMs busy, timed with CUDA events on the caller's stream.
// 2*8*8*4 = 512 flop per warp-wide DMMA.
// =====================================================================================
#pragma once
#include <cuda_runtime.h>

namespace gfcc {

template <int CHAINS>
__global__ void __launch_bounds__(256) k_dmma_probe(double* __restrict__ sink, int iters, double a0, double b0) {
  double c[CHAINS][2];
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) { c[k][0] = (double)threadIdx.x; c[k][1] = (double)k; }
  const double a = a0 + 1e-9 * (threadIdx.x & 3), b = b0 - 1e-9 * (threadIdx.x >> 2);
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int k = 0; k < CHAINS; ++k)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                   : "+d"(c[k][0]), "+d"(c[k][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int k = 0; k < CHAINS; ++k) s += c[k][0] + c[k][1];
  if (s == 123.456) sink[blockIdx.x * blockDim.x + threadIdx.x] = s;   // never true in practice; keeps the chain alive
}

// returns TFLOP/s (best of `reps` launches of ~`iters` DMMAs per chain), or a negative value on a CUDA error
inline double dmma_peak_probe(cudaStream_t st, int iters, int reps) {
  constexpr int CHAINS = 16;
  int dev = 0, sms = 0;
  if (cudaGetDevice(&dev) != cudaSuccess) return -1;
  if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return -1;
  double* sink = nullptr;
  if (cudaMalloc(&sink, sizeof(double)) != cudaSuccess) return -1;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int blocks = sms * 2, threads = 256;
  double best = -1;
  for (int r = 0; r < reps + 1; ++r) {   // first launch is the warm-up
    cudaEventRecord(e0, st);
    k_dmma_probe<CHAINS><<<blocks, threads, 0, st>>>(sink, iters, 1.0000001, 0.9999999);
    cudaEventRecord(e1, st);
    if (cudaEventSynchronize(e1) != cudaSuccess) { best = -1; break; }
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    const double flops = 512.0 * CHAINS * (double)iters * (threads / 32) * blocks;
    if (r > 0 && ms > 0) best = fmax(best, flops / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(sink);
  return best;
}

}  // namespace gfcc
