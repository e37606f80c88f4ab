/*
 * lisa_td_probe.h -- measurement support for bench.py, NOT part of the product ABI (include/lisa_td.h).
 * Built into its own shared library, liblisa_td_probe.so (paper_2501_08261_b200/build.py).
 *
 * The fp64 roofline denominator is not in MEASURED_PEAKS.json, so bench.py measures it in the same
 * run as the kernels.  Return value 0 or a negative number; both
 * calls synchronise.
 */
#ifndef LISA_TD_PROBE_H
#define LISA_TD_PROBE_H
#ifdef __cplusplus
extern "C" {
#endif

/* A register-resident chain of `iters` x 8 dependent-free DFMA per thread on `blocks` x `threads`;
 * returns the elapsed milliseconds (CUDA events) in *ms_host and writes one double per thread to
 * sink (device, blocks*threads doubles) so the work is not optimised away.
 * FLOP count = 2 * 8 * iters * blocks * threads. */
__attribute__((visibility("default"))) int lisa_td_probe_dfma(long long iters, int blocks, int threads, double* sink,
                                                              float* ms_host, void* stream);

/* In every block, dfma_warps warps run 8 independent DFMA chains per thread and dmma_warps warps
 * run 4 independent mma.sync.m8n8k4.f64 accumulator pairs, `iters` rounds each (dfma_warps +
 * dmma_warps <= 32).  FLOP count = 2 * iters * blocks * (256 * dfma_warps + 1024 * dmma_warps).
 * Answers whether the fp64 tensor path (K3) and the DFMA pipe (K1, K2) are separate units: on B200
 * the times add, i.e. they are one resource.  sink: blocks * 32 * (dfma_warps + dmma_warps) doubles. */
__attribute__((visibility("default"))) int lisa_td_probe_fp64_pipes(long long iters, int blocks, int dfma_warps,
                                                                    int dmma_warps, double* sink, float* ms_host,
                                                                    void* stream);

/* Issue rate of fp64 instructions by the number of distinct register operands they read, on
 * `blocks` x 128 threads (4 blocks per SM resident), `iters` rounds:
 *   pattern 0: a = fma(a, const, const)      8 per round, one register operand
 *   pattern 1: a = a * b                     8 per round, two register operands
 *   pattern 2: a = fma(a, b, c0)             8 per round, two fresh + one repeated operand
 *   pattern 3: a = fma(a, b, c)              8 per round, three distinct register operands
 *   pattern 4: K2's order-31 Lagrange sweep (lagrange_dot2h_x2<16> of common.cuh) on a shared-memory
 *              tile in K2's block shape, 352 per round: the ceiling of K2's instruction mix
 * Instruction count per thread = (pattern < 4 ? 8 : 352) * iters.  sink: blocks * 128 doubles. */
__attribute__((visibility("default"))) int lisa_td_probe_fp64_operands(int pattern, long long iters, int blocks,
                                                                       double* sink, float* ms_host, void* stream);
#ifdef __cplusplus
}
#endif
#endif
