// probe.cu -- fp64 throughput probes used by bench.py only (lisa_td_probe.h); built into
// liblisa_td_probe.so, separate from the product library.
#include <cuda_runtime.h>

#include "common.cuh"
#include "lisa_td_probe.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "written for sm_100a (B200) only"
#endif

#define PROBE_CUDA(call)                  \
  do {                                    \
    if ((call) != cudaSuccess) return -4; \
  } while (0)

// ---------------------------------------------------------------------- register-operand probe
// How many DISTINCT 64-bit register operands an fp64 instruction reads decides its issue interval on
// B200: one or two (DMUL, or DFMA with a constant / immediate / repeated operand) -> every 2 cycles,
// three fresh ones -> every 3 cycles.
template <int PAT>
__global__ void __launch_bounds__(128, 4) k_probe_fp64_operands(long long iters, double* sink) {
  double a[8], b[8], c[8];
#pragma unroll
  for (int i = 0; i < 8; ++i) {
    a[i] = 1.0 + threadIdx.x * 1e-9 + i * 1e-3;
    b[i] = 0.999999 + 1e-9 * i + 1e-12 * threadIdx.x;
    c[i] = 1e-9 * (i + 1) + 1e-15 * threadIdx.x;
  }
  for (long long it = 0; it < iters; ++it) {
#pragma unroll
    for (int i = 0; i < 8; ++i) {
      if (PAT == 0) a[i] = fma(a[i], 0.999999, 1e-7);
      if (PAT == 1) a[i] = a[i] * b[i];
      if (PAT == 2) a[i] = fma(a[i], b[i], c[0]);
      if (PAT == 3) a[i] = fma(a[i], b[i], c[i]);
    }
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = ((a[0] + a[1]) + (a[2] + a[3])) + ((a[4] + a[5]) + (a[6] + a[7]));
}

// K2's order-31 sweep and nothing else: lagrange_dot2h_x2<16> of common.cuh (the function K2 calls nine
// times per walker and sample pair) in a loop on a shared-memory tile, in K2's block shape (128 threads,
// four blocks per SM, LagS in the constant bank).  352 fp64 instructions per call; four of the eleven
// per node pair read three fresh registers.  What this kernel reaches is the ceiling of K2's instruction mix.
constexpr int PROBE_LE = 160;
__global__ void __launch_bounds__(128, 4) k_probe_k2_sweep(long long iters, const lisa::LagS ls, double* sink) {
  __shared__ double2 tile[2 * PROBE_LE];
  for (int i = threadIdx.x; i < 2 * PROBE_LE; i += 128) tile[i] = make_double2(1.0 + 1e-3 * i, 2.0 - 1e-3 * i);
  __syncthreads();
  double epsa = 0.3 + 1e-3 * threadIdx.x, epsb = epsa + 1e-4, acc = 0.0;
  const int e = 2 * threadIdx.x + 16;
#pragma unroll 1
  for (long long it = 0; it < iters; ++it) {
    double vp[2], vc[2];
    lisa::lagrange_dot2h_x2<16>(epsa, epsb, 16, ls, tile, tile + PROBE_LE, e + (int)(it & 3), vp, vc);
    acc += (vp[0] + vc[0]) + (vp[1] + vc[1]);
    epsa += 1e-5;
    epsb += 1e-5;
  }
  sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

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

int lisa_td_probe_fp64_operands(int pattern, long long iters, int blocks, double* sink, float* ms_host, void* stream) {
  if (pattern < 0 || pattern > 4 || iters <= 0 || blocks <= 0 || !sink || !ms_host) return -1;
  cudaStream_t st = (cudaStream_t)stream;
  cudaEvent_t e0, e1;
  PROBE_CUDA(cudaEventCreate(&e0));
  PROBE_CUDA(cudaEventCreate(&e1));
  PROBE_CUDA(cudaEventRecord(e0, st));
  switch (pattern) {
    case 0: k_probe_fp64_operands<0><<<blocks, 128, 0, st>>>(iters, sink); break;
    case 1: k_probe_fp64_operands<1><<<blocks, 128, 0, st>>>(iters, sink); break;
    case 2: k_probe_fp64_operands<2><<<blocks, 128, 0, st>>>(iters, sink); break;
    case 3: k_probe_fp64_operands<3><<<blocks, 128, 0, st>>>(iters, sink); break;
    default: {
      lisa::LagS ls;  // values that keep every partial product finite; the timing does not depend on them
      for (int k = 0; k < lisa::MAX_HALF; ++k) {
        ls.rho[k] = 0.1 + 1e-3 * k;
        ls.rc[k] = 0.99 + 1e-3 * k;
      }
      ls.g = 1.0;
      k_probe_k2_sweep<<<blocks, 128, 0, st>>>(iters, ls, sink);
    }
  }
  PROBE_CUDA(cudaPeekAtLastError());
  PROBE_CUDA(cudaEventRecord(e1, st));
  PROBE_CUDA(cudaEventSynchronize(e1));
  PROBE_CUDA(cudaEventElapsedTime(ms_host, e0, e1));
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return 0;
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
