/*
 * sfft_bench.h -- measurement support for bench.py ONLY (libsfft_bench.so; not part of the product ABI in
 * include/sfft.h and never linked into libsfft_b200.so).
 */
#ifndef SFFT_BENCH_H_
#define SFFT_BENCH_H_
#ifdef __cplusplus
extern "C" {
#endif

struct sfft_plan;

/* Achieved FP64 throughput of the current device in TFLOP/s from a register-resident probe kernel,
 * kind 0 = plain FMA pipe (DFMA), kind 1 = FP64 tensor cores (mma.sync.m8n8k4.f64).  These are the
 * denominators of the "alu" rooflines in DESIGN.md / bench.py.  Synchronous; best of 3 timed runs.
 * Returns 0 on success. */
int sfft_bench_fp64_peak(int kind, double *tflops);

/* FP64 work of the x-direction lag correlation (steps a3+a4) of one sfft_build_system per batch entry, counted
 * from the plan's own launch configuration: *executed = flops the kernel issues (FFT butterflies at 5 N log2 N
 * per 64-point transform plus 512 per mma.sync.m8n8k4.f64), *tensor = the part of it issued as DMMA. */
int sfft_bench_corr_flops(const struct sfft_plan *plan, double *executed, double *tensor);

#ifdef __cplusplus
}
#endif
#endif
