// microbench.cuh — register-resident FMA-chain kernels that measure the plain-ALU peaks the roofline of
// bench.py is quoted against (MEASURED_PEAKS.json has no FP64/FP32 FMA peak).
#pragma once
#include <cuda_runtime.h>

namespace rwgt {

template <typename T, int ILP>
__global__ void __launch_bounds__(256) fma_chain_kernel(T* out, T a, T b, int iters) {
  T x[ILP];
#pragma unroll
  for (int i = 0; i < ILP; i++) x[i] = T(threadIdx.x + i);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < ILP; i++) x[i] = fma(x[i], a, b);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < ILP; i++) s += x[i];
  if (s == T(12345.678)) out[0] = s;          // keeps the chain alive, practically never taken
}

__global__ void __launch_bounds__(256) dmma_chain_kernel(double* out, double a, double b, int iters) {
  double c[8][2];
#pragma unroll
  for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int i = 0; i < 8; i++)
      asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
  }
  double s = 0;
#pragma unroll
  for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
  if (s == 12345.678) out[0] = s;
}

// kind 0: FP64 FMA, 1: FP32 FMA, 2: FP64 DMMA m8n8k4.  Returns TFLOP/s (2 flop per FMA), best of 5.
static int measure_peak(int kind, double* tflops) {
  int dev = 0; cudaGetDevice(&dev); cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
  double* d = nullptr; if (cudaMalloc((void**)&d, 64) != cudaSuccess) return -1;
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096, ILP = 8, threads = 256; int blocks = prop.multiProcessorCount * 8;
  double best = 0;
  for (int rep = 0; rep < 6; rep++) {
    cudaEventRecord(e0);
    if (kind == 0) fma_chain_kernel<double, ILP><<<blocks, threads>>>(d, 1.0000001, 1e-9, iters);
    else if (kind == 1) fma_chain_kernel<float, ILP><<<blocks, threads>>>((float*)d, 1.0000001f, 1e-9f, iters);
    else dmma_chain_kernel<<<blocks, threads>>>(d, 1.0000001, 1e-9, iters);
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    double fl = (kind == 2) ? (double)blocks * (threads / 32) * iters * 8.0 * (8 * 8 * 4 * 2.0) : (double)blocks * threads * iters * ILP * 2.0;
    if (rep > 0) best = fmax(best, fl / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) return -1;
  *tflops = best; return 0;
}

}  // namespace rwgt
