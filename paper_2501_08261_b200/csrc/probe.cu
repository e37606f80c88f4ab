// probe.cu -- fp64 throughput probes used by bench.py only (lisa_td_probe.h); built into
// liblisa_td_probe.so, separate from the product library.
#include <cuda_runtime.h>

#include "lisa_td_probe.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "written for sm_100a (B200) only"
#endif

#define PROBE_CUDA(call)                  \
  do {                                    \
    if ((call) != cudaSuccess) return -4; \
  } while (0)

extern "C" {

// ---------------------------------------------------------------------- DFMA probe
__global__ void k_probe_dfma(long long iters, double* sink) {
  double a0 = 1.0 + threadIdx.x * 1e-9, a1 = a0 + 1e-3, a2 = a0 + 2e-3, a3 = a0 + 3e-3;
  double a4 = a0 + 4e-3, a5 = a0 + 5e-3, a6 = a0 + 6e-3, a7 = a0 + 7e-3;
  const double m = 0.999999, c = 1e-7;
  for (long long i = 0; i < iters; ++i) {
    a0 = fma(a0, m, c); a1 = fma(a1, m, c); a2 = fma(a2, m, c); a3 = fma(a3, m, c);
    a4 = fma(a4, m, c); a5 = fma(a5, m, c); a6 = fma(a6, m, c); a7 = fma(a7, m, c);
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
}

// Warps 0..dfma_warps-1 of every block run 8 independent DFMA chains per thread, the next dmma_warps
// warps run 4 independent DMMA (mma.sync m8n8k4 f64) accumulator pairs: do the two paths share a pipe?
__global__ void __launch_bounds__(1024) k_probe_fp64_pipes(long long iters, int dfma_warps, int dmma_warps, double* sink) {
  const int wid = threadIdx.x >> 5;
  const double x = 1.0 + threadIdx.x * 1e-9, y = 0.999999;
  double r = 0.0;
  if (wid < dfma_warps) {
    double a0 = x, a1 = x + 1e-3, a2 = x + 2e-3, a3 = x + 3e-3, a4 = x + 4e-3, a5 = x + 5e-3, a6 = x + 6e-3, a7 = x + 7e-3;
    for (long long i = 0; i < iters; ++i) {
      a0 = fma(a0, y, x); a1 = fma(a1, y, x); a2 = fma(a2, y, x); a3 = fma(a3, y, x);
      a4 = fma(a4, y, x); a5 = fma(a5, y, x); a6 = fma(a6, y, x); a7 = fma(a7, y, x);
    }
    r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
  } else {
    double d[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (long long i = 0; i < iters; ++i) {
#pragma unroll
      for (int q = 0; q < 4; ++q)
        asm volatile("mma.sync.aligned.m8n8k4.row.col.f64.f64.f64.f64 {%0,%1}, {%2}, {%3}, {%0,%1};\n"
                     : "+d"(d[2 * q]), "+d"(d[2 * q + 1])
                     : "d"(x), "d"(y));
    }
    r = ((d[0] + d[1]) + (d[2] + d[3])) + ((d[4] + d[5]) + (d[6] + d[7]));
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = r;
}

int lisa_td_probe_fp64_pipes(long long iters, int blocks, int dfma_warps, int dmma_warps, double* sink, float* ms_host,
                             void* stream) {
  if (iters <= 0 || blocks <= 0 || dfma_warps < 0 || dmma_warps < 0 || dfma_warps + dmma_warps < 1 ||
      dfma_warps + dmma_warps > 32 || !sink || !ms_host)
    return -1;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  PROBE_CUDA(cudaEventCreate(&e0));
  PROBE_CUDA(cudaEventCreate(&e1));
  PROBE_CUDA(cudaEventRecord(e0, st));
  k_probe_fp64_pipes<<<blocks, 32 * (dfma_warps + dmma_warps), 0, st>>>(iters, dfma_warps, dmma_warps, sink);
  PROBE_CUDA(cudaPeekAtLastError());
  PROBE_CUDA(cudaEventRecord(e1, st));
  PROBE_CUDA(cudaEventSynchronize(e1));
  PROBE_CUDA(cudaEventElapsedTime(ms_host, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return 0;
}

int lisa_td_probe_dfma(long long iters, int blocks, int threads, double* sink, float* ms_host, void* stream) {
  if (iters <= 0 || blocks <= 0 || threads <= 0 || threads > 1024 || !sink || !ms_host)
    return -1;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  PROBE_CUDA(cudaEventCreate(&e0));
  PROBE_CUDA(cudaEventCreate(&e1));
  PROBE_CUDA(cudaEventRecord(e0, st));
  k_probe_dfma<<<blocks, threads, 0, st>>>(iters, sink);
  PROBE_CUDA(cudaPeekAtLastError());
  PROBE_CUDA(cudaEventRecord(e1, st));
  PROBE_CUDA(cudaEventSynchronize(e1));
  PROBE_CUDA(cudaEventElapsedTime(ms_host, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return 0;
}

}  // extern "C"
