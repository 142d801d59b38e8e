// event_file.cuh — the host side of the reweighting procedure (PAPER.md:87 steps 2 "Parse events" and 8 "Return new weights";
// initialisation, I/O and host<->device transfer dominate small event sets; the paper's library
// parses LHE event files).  LHE files do not exist here, so a binary structure-of-arrays event file stands in:
//
//   event file  (include/rwgt.h: rwgt_event_file_header, 64 bytes, little endian)
//       magic "RWGTEVT1", uint32 version = 1, uint32 n_ext, uint64 n_events, char process[32], 8 bytes reserved
//       double momenta[n_ext][4][n_events]      (E,px,py,pz planes: the SoA layout of rwgt_run)
//       double weights[n_events]
//   result file (rwgt_result_file_header, 64 bytes)
//       magic "RWGTRES1", uint32 version = 1, uint32 n_sets K, uint64 n_events, char process[32], uint64 first_event
//       double me_old[n_events], me_new[K][n_events], w_new[K][n_events]
//       double sum_w_old, sum_w_new[K]           (eq. 2: sigma ~ sum_k W_k, per parameter set)
//
// rwgt_run_file streams a contiguous event range through the device in chunks: a reader thread fills pinned buffer (c+1) % 2 from the
// file while chunk c goes through the chunked H2D / kernel / D2H pipeline of rwgt_run_multi_host and a writer thread puts the results
// of chunk c-1 into the result file.
#pragma once
#include <cuda_runtime.h>
#include <fcntl.h>
#include <sys/stat.h>
#include <unistd.h>
#include <condition_variable>
#include <cstdint>
#include <cstring>
#include <mutex>
#include <string>
#include <thread>

#include "../../include/rwgt.h"

namespace rwgt {

// ---------------------------------------------------------------------------- eq. 2: deterministic sums of weight rows
// sum_k W_k for each of n_rows rows of length n (row stride = rstride).  No atomics: a fixed grid of SUM_BLOCKS blocks per row, each
// block owns a fixed contiguous slice (boundaries depend on n only), threads accumulate strided partials in index order, a fixed
// shared-memory tree combines them, and the last block of a row (ticket counter) adds the SUM_BLOCKS partials in block order.
// The result is a function of (values, n) only: bitwise reproducible, independent of scheduling.
constexpr int SUM_BLOCKS = 64, SUM_THREADS = 256;
__global__ void __launch_bounds__(SUM_THREADS) sum_rows_kernel(const double* __restrict__ w, long long n, long long rstride, double* __restrict__ partial,
                                                             unsigned* __restrict__ ticket, double* __restrict__ out) {
  __shared__ double sh[SUM_THREADS];
  __shared__ bool last;
  const int row = blockIdx.y, b = blockIdx.x;
  const long long per = (n + SUM_BLOCKS - 1) / SUM_BLOCKS, lo = b * per, hi = (lo + per < n) ? lo + per : n;
  const double* r = w + (size_t)row * rstride;
  double acc = 0.0;
  for (long long i = lo + threadIdx.x; i < hi; i += SUM_THREADS) acc += __ldg(r + i);
  sh[threadIdx.x] = acc;
  __syncthreads();
  for (int d = SUM_THREADS / 2; d >= 1; d >>= 1) { if ((int)threadIdx.x < d) sh[threadIdx.x] += sh[threadIdx.x + d]; __syncthreads(); }
  if (threadIdx.x == 0) {
    partial[row * SUM_BLOCKS + b] = sh[0];
    __threadfence();
    last = (atomicAdd(ticket + row, 1u) == SUM_BLOCKS - 1);
  }
  __syncthreads();
  if (last && threadIdx.x == 0) {
    __threadfence();
    double s = 0.0;
    for (int j = 0; j < SUM_BLOCKS; j++) s += *((volatile double*)(partial + row * SUM_BLOCKS + j));
    out[row] = s;
    ticket[row] = 0u;                      // ready for the next call on this stream
  }
}

// ---------------------------------------------------------------------------- file headers
static_assert(sizeof(rwgt_event_file_header) == 64 && sizeof(rwgt_result_file_header) == 64, "file headers are 64 bytes");

static bool pread_all(int fd, void* buf, size_t bytes, off_t off) {
  char* p = (char*)buf;
  while (bytes > 0) { ssize_t r = ::pread(fd, p, bytes, off); if (r <= 0) return false; p += r; off += r; bytes -= (size_t)r; }
  return true;
}
static bool pwrite_all(int fd, const void* buf, size_t bytes, off_t off) {
  const char* p = (const char*)buf;
  while (bytes > 0) { ssize_t r = ::pwrite(fd, p, bytes, off); if (r <= 0) return false; p += r; off += r; bytes -= (size_t)r; }
  return true;
}

// one pinned double buffer set of the file pipeline: inputs [planes + 1][chunk], outputs [1 + 2K][chunk]
struct FileBuffers {
  double* in[2] = {nullptr, nullptr}; double* out[2] = {nullptr, nullptr}; long long chunk = 0; int planes = 0, K = 0;
  void release() { for (int i = 0; i < 2; i++) { if (in[i]) cudaFreeHost(in[i]); if (out[i]) cudaFreeHost(out[i]); in[i] = out[i] = nullptr; } chunk = 0; }
  cudaError_t ensure(long long c, int pl, int k) {
    if (c <= chunk && pl == planes && k == K) return cudaSuccess;
    release();
    for (int i = 0; i < 2; i++) {
      cudaError_t e = cudaHostAlloc((void**)&in[i], sizeof(double) * (size_t)(pl + 1) * c, cudaHostAllocDefault);
      if (e == cudaSuccess) e = cudaHostAlloc((void**)&out[i], sizeof(double) * (size_t)(1 + 2 * k) * c, cudaHostAllocDefault);
      if (e != cudaSuccess) { release(); return e; }
    }
    chunk = c; planes = pl; K = k; return cudaSuccess;
  }
};

}  // namespace rwgt
