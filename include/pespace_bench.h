/* pespace_bench.h -- measurement scaffolding of libpespace.so, kept apart from the product boundary
 * (include/pespace.h): an FP64 micro-benchmark for the roofline denominator, event timing of the
 * dominant kernels, and a launch counter.  bench.py and the tests use them; a sampler never needs them.
 * These calls hold process-wide state (one switch, one bounded event list, one counter), all of it atomic or
 * mutex-protected; the calls of pespace.h themselves keep none. */
#ifndef PESPACE_BENCH_H
#define PESPACE_BENCH_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* FP64 FMA micro-benchmark used as the roofline denominator: runs `iters` blocks of 64
 * DFMAs (8 independent chains) per thread on every SM and returns the sustained rate in
 * TFLOP/s (FMA = 2 flop) and the kernel time in ms.  Synchronous.
 *   mode 0: a = a*m + c with m, c shared by the chains (two register operands per DFMA):
 *           the FP64 pipe peak, 1 warp-instruction / 2 cycles / SM sub-partition;
 *   mode 1: a = a*b + c with three distinct register operands per DFMA: the register-file
 *           read bandwidth then limits the pipe to 1 / 3 cycles (profiles/r01_fp64_operand_bandwidth.md);
 *   modes 2-5: FP64 tensor-core probe, `iters` blocks of 8 x NACC mma.sync.m8n8k4.f64 (DMMA, 256 FMAs per warp
 *           instruction) per warp: 2: NACC = 8 independent accumulators; 3: NACC = 2; 4: NACC = 8 with one
 *           independent DFMA per DMMA interleaved; 5: with four (profiles/r02_dmma.md);
 *   modes 6-10: register-operand probes (profiles/r02_operand_reuse.md): 6: DFMA a_j = a_j m + c_j, one operand
 *           shared with the preceding instruction; 7: DFMA a_j = a_j b_{j&1} + c_j, shared with the one before
 *           that; 8: FP32 FFMA with three distinct registers (128 FMAs per thread and block of rounds; the rate
 *           is returned in FP32 TFLOP/s); 9: packed FFMA2 with three distinct register pairs; 10: FFMA with
 *           multiplier and addend shared (the FP32 pipe peak). */
int pespace_fp64_peak(int mode, int iters, double* h_out_tflops, double* h_out_ms);

/* Kernel timing for roofline reports.  While enabled, every launch of the dominant kernel
 * (the fused per-bin likelihood kernel, or the Fisher kernel) is bracketed by CUDA events on the
 * launching stream.
 * pespace_profile_read synchronises those events and returns the summed kernel time in ms and
 * the number of launches since the last read (either pointer may be NULL), then resets.  At most 65536 launches are
 * kept between two reads; later ones are not timed. */
int pespace_profile_enable(int on);
int pespace_profile_read(double* h_main_ms, int64_t* h_launches);

/* Number of kernels this library has launched since load (all calls, all streams). */
int64_t pespace_launch_count(void);

#ifdef __cplusplus
}
#endif
#endif
