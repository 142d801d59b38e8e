// microbench.cu — register-resident FMA-chain kernels that measure the plain-ALU peaks the roofline of
// bench.py is quoted against (MEASURED_PEAKS.json has no FP64/FP32 FMA peak).
// A measurement aid: built into its own library (librwgt_microbench.so, include/rwgt_microbench.h), NOT into librwgt.so.
#include <cuda_runtime.h>
#include <cmath>

#include "../../include/rwgt_microbench.h"

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

// acc[i] = fma(y[.], z[.], acc[i]) with register-resident operands, the operand pattern of real complex arithmetic.
// REUSE = 0: three distinct source registers per FMA; REUSE = 1: one source shared by 16 consecutive FMAs (the
// operand-reuse cache can serve it).  Measured on B200: a DFMA with three distinct 64-bit sources issues every
// ~3.0 cycles per sub-partition, with one reused source every ~2.4, against 2.0 for the x = fma(x, a, b) chain.
template <typename T, int REUSE>
__global__ void __launch_bounds__(256) fma_operand_kernel(T* out, const T* in, int iters) {
  T y[8], z[8], acc[16];
#pragma unroll
  for (int i = 0; i < 8; i++) { y[i] = in[threadIdx.x + i]; z[i] = in[threadIdx.x + 8 + i]; }
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = T(i);
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 4; r++)
#pragma unroll
      for (int i = 0; i < 16; i++) acc[i] = REUSE ? fma(y[r], z[i & 7], acc[i]) : fma(y[(i + r) & 7], z[(i * 3 + r) & 7], acc[i]);
  }
  T s = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) s += acc[i];
  if (s == T(12345.678)) out[0] = s;
}

// packed FP32: fma.rn.f32x2 (SASS FFMA2), the same two operand patterns and the chain
__device__ __forceinline__ unsigned long long mb_pk(float a, float b) { unsigned long long r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(a), "f"(b)); return r; }
__device__ __forceinline__ unsigned long long mb_fma2(unsigned long long a, unsigned long long b, unsigned long long c) { unsigned long long d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
template <int MODE>      // 0: chains x = fma2(x, a, b);  1: three distinct sources;  2: one source shared by 16 consecutive FMAs
__global__ void __launch_bounds__(256) ffma2_kernel(float* out, const float* in, int iters) {
  unsigned long long y[8], z[8], acc[16];
#pragma unroll
  for (int i = 0; i < 8; i++) { y[i] = mb_pk(in[threadIdx.x + i] + 1.0000001f, in[threadIdx.x + i + 32] + 1.0000001f); z[i] = mb_pk(in[threadIdx.x + 8 + i] + 1e-9f, in[threadIdx.x + 40 + i] + 1e-9f); }
#pragma unroll
  for (int i = 0; i < 16; i++) acc[i] = mb_pk((float)i, (float)(i + 1));
  for (int it = 0; it < iters; it++) {
#pragma unroll
    for (int r = 0; r < 4; r++)
#pragma unroll
      for (int i = 0; i < 16; i++)
        acc[i] = MODE == 0 ? mb_fma2(acc[i], y[0], z[0]) : MODE == 2 ? mb_fma2(y[r], z[i & 7], acc[i]) : mb_fma2(y[(i + r) & 7], z[(i * 3 + r) & 7], acc[i]);
  }
  unsigned long long sacc = 0;
#pragma unroll
  for (int i = 0; i < 16; i++) sacc ^= acc[i];
  if (sacc == 12345678ull) out[0] = 1.0f;
}

// 8 warps of FP64 FMA chains and 4 warps of DMMA chains in one CTA per SM: do the two share a pipe?
__global__ void __launch_bounds__(384, 1) dfma_dmma_kernel(double* out, double a, double b, int it_fma, int it_mma) {
  if ((threadIdx.x >> 5) < 8) {
    double x[8];
#pragma unroll
    for (int i = 0; i < 8; i++) x[i] = threadIdx.x + i;
    for (int it = 0; it < it_fma; it++) {
#pragma unroll
      for (int i = 0; i < 8; i++) x[i] = fma(x[i], a, b);
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += x[i];
    if (s == 12345.678) out[0] = s;
  } else {
    double c[8][2];
#pragma unroll
    for (int i = 0; i < 8; i++) { c[i][0] = threadIdx.x; c[i][1] = i; }
    for (int it = 0; it < it_mma; it++) {
#pragma unroll
      for (int i = 0; i < 8; i++)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};" : "+d"(c[i][0]), "+d"(c[i][1]) : "d"(a), "d"(b));
    }
    double s = 0;
#pragma unroll
    for (int i = 0; i < 8; i++) s += c[i][0] + c[i][1];
    if (s == 12345.678) out[0] = s;
  }
}

// kind 0: FP64 FMA chain x = fma(x,a,b);  1: FP32 FMA chain;  2: FP64 DMMA m8n8k4 chain;
//      3: FP64 FMA with three distinct register sources;  4: FP64 FMA with one reused source;
//      5: FP32 FMA with three distinct register sources;  6: FP32 FMA with one reused source;
//      7: FP64 FMA chains (8 warps) and DMMA chains (4 warps) running CONCURRENTLY on every SM, summed rate
//         (equal to kind 0 / kind 2 alone if the two share one pipe, their sum if not).
//      8 / 9 / 10: packed FP32 fma.rn.f32x2 (FFMA2): chains / three distinct sources / one reused source.
// Returns TFLOP/s (2 flop per FMA), best of 5.
static int measure_peak(int kind, double* tflops) {
  int dev = 0; cudaGetDevice(&dev); cudaDeviceProp prop; cudaGetDeviceProperties(&prop, dev);
  double* d = nullptr; if (cudaMalloc((void**)&d, 4096 * sizeof(double)) != cudaSuccess) return -1;
  cudaMemset(d, 0, 4096 * sizeof(double));
  cudaEvent_t e0, e1; cudaEventCreate(&e0); cudaEventCreate(&e1);
  const int iters = 4096, ILP = 8, threads = 256; int blocks = prop.multiProcessorCount * 8;
  double best = 0;
  for (int rep = 0; rep < 6; rep++) {
    double fl = (double)blocks * threads * iters * ILP * 2.0;
    cudaEventRecord(e0);
    switch (kind) {
      case 0: fma_chain_kernel<double, ILP><<<blocks, threads>>>(d, 1.0000001, 1e-9, iters); break;
      case 1: fma_chain_kernel<float, ILP><<<blocks, threads>>>((float*)d, 1.0000001f, 1e-9f, iters); break;
      case 2: dmma_chain_kernel<<<blocks, threads>>>(d, 1.0000001, 1e-9, iters); fl = (double)blocks * (threads / 32) * iters * 8.0 * (8 * 8 * 4 * 2.0); break;
      case 3: fma_operand_kernel<double, 0><<<blocks, threads>>>(d, d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 2.0; break;
      case 4: fma_operand_kernel<double, 1><<<blocks, threads>>>(d, d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 2.0; break;
      case 5: fma_operand_kernel<float, 0><<<blocks, threads>>>((float*)d, (float*)d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 2.0; break;
      case 6: fma_operand_kernel<float, 1><<<blocks, threads>>>((float*)d, (float*)d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 2.0; break;
      case 8: ffma2_kernel<0><<<blocks, threads>>>((float*)d, (float*)d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 4.0; break;
      case 9: ffma2_kernel<1><<<blocks, threads>>>((float*)d, (float*)d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 4.0; break;
      case 10: ffma2_kernel<2><<<blocks, threads>>>((float*)d, (float*)d, iters / 8); fl = (double)blocks * threads * (iters / 8) * 64 * 4.0; break;
      default: {
        const int itf = 16384, itm = 4096;      // equal pipe time for the two groups if they share the pipe at the same rate
        dfma_dmma_kernel<<<prop.multiProcessorCount, 384>>>(d, 1.0000001, 1e-9, itf, itm);
        fl = (double)prop.multiProcessorCount * (256.0 * itf * 8 * 2.0 + 4.0 * itm * 8 * (8 * 8 * 4 * 2.0));
      }
    }
    cudaEventRecord(e1); cudaEventSynchronize(e1);
    float ms = 0; cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0) best = fmax(best, fl / (ms * 1e-3) / 1e12);
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1); cudaFree(d);
  if (cudaGetLastError() != cudaSuccess) return -1;
  *tflops = best; return 0;
}

}  // namespace rwgt

extern "C" int rwgt_microbench_peak(int kind, double* out_tflops) {
  if (kind < 0 || kind > 10 || !out_tflops) return -1;
  return rwgt::measure_peak(kind, out_tflops);
}
