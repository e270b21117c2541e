/* qmll_aux.h -- measurement aids of libqmll.so (bench.py, paper_2206_01580_b200/peaks.py).  Not part of the
 * method's boundary (include/qmll.h): nothing here computes a step of the path.  Process-wide host-side state,
 * guarded by a mutex where it is shared with the compute calls. */
#ifndef QMLL_AUX_H_
#define QMLL_AUX_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* Counters for benchmarks: number of kernel launches issued by this library since the last reset
 * (process-wide, host-side counter). */
int64_t qmll_launch_count(void);
void qmll_reset_launch_count(void);

/* Measurement aid (bench.py roofline): when enabled, every launch of the tensor-core kernel inside
 * qmll_normal_equations is bracketed by CUDA events on the caller's stream.  The collect call waits for them,
 * returns the summed kernel time in ms and the number of launches since the last collect, and frees them
 * (at most 4096 launches are recorded between collects).  Not thread-safe. */
void qmll_time_normal_equations_kernel(int enable);
int qmll_collect_normal_equations_kernel_ms(double* total_ms, int* launches);

/* Roofline denominators MEASURED_PEAKS.json lacks: a register-only loop of one
 * instruction mix on every SM (kinds listed in paper_2206_01580_b200/peaks.py and csrc/microbench.cu).  Launches
 * one kernel on `cuda_stream`; the caller times it with CUDA events.  workspace (device): first n_blocks int64 =
 * clock64 ticks per block.  ops_per_launch = lane-operations (bytes for the shared-memory kind) the launch does. */
int qmll_microbench(int kind, int iters, int blocks_per_sm, void* workspace, size_t workspace_bytes,
                    double* ops_per_launch, int* n_blocks, void* cuda_stream);

/* Timing of tcgen05.mma itself: M = 128, kind::f16, both operands in shared memory, one CTA per SM; `iters` x 4 x
 * `accumulators` MMAs of width n (64, 96, 128 or 256) rotating over `accumulators` (1, 2 or 4; 1 or 2 for n = 256) TMEM
 * accumulators, issued back to back by one elected lane.  workspace (device, >= 8 bytes): int64 clock64 ticks of block 0
 * from the first issue to completion.  Behind the "max(n/2, 32 + n/4) clocks per MMA" law of DESIGN.md section 5.2. */
int qmll_microbench_mma(int n, int accumulators, int iters, void* workspace, size_t workspace_bytes, void* cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* QMLL_AUX_H_ */
