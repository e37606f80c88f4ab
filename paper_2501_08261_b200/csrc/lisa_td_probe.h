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
#ifdef __cplusplus
}
#endif
#endif
