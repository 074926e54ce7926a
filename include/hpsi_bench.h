/*
 * hpsi_bench.h - C ABI of libhpsi_bench.so: FP64 pipe probes that bench.py loads for its calibration block.  Not part of
 * the product library (libhpsi.so exports nothing of this): a register-resident issue-rate microbenchmark says what the
 * FP64 pipes of this B200 can do, next to the cuBLAS DGEMM figure BASELINE.json names as the denominator.
 */
#ifndef HPSI_BENCH_H_
#define HPSI_BENCH_H_

#ifdef __cplusplus
extern "C" {
#endif

/* Run `iters` dependent-chain rounds of register-resident DMMA.8x8x4 (kind 0), DFMA (kind 1) or both interleaved
 * (kind 2) on every SM (4 CTAs of 8 warps per SM); kind 100+w runs the DMMA probe with w one-warp CTAs (1..32) per SM.
 * ms_out / flops_out: HOST, elapsed milliseconds (CUDA events) and flops executed.  Returns 0, -1 on a bad argument,
 * -3 on a CUDA error (hpsi_bench_last_error() has the text). */
int hpsi_bench_fp64_pipe(int kind, int iters, double* ms_out, double* flops_out);
const char* hpsi_bench_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* HPSI_BENCH_H_ */
