/*
 * mdwf_bench.h -- measurement entry points of libmdwf_b200.so.  NOT part of the solver boundary (include/mdwf.h, the calls
 * SURVEY.md section 8(b) lists): these exist so that bench.py and the profiling command (timeop.py) can time the kernels of
 * the hot path in isolation and measure the roofline denominators on the device the run uses (DESIGN.md sections 6, 7).
 * They live in their own translation units (csrc/mdwf_bench.cu, csrc/peak_kernels.cu).
 */
#ifndef MDWF_BENCH_H
#define MDWF_BENCH_H
#include "mdwf.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Measurement: run op (MDWF_OP_MPC or MDWF_OP_MPCDAG) `reps` times after `warmup`
 * untimed runs, in precision "fp64" | "fp32" | "half", on library-owned hash-filled vectors, timed with
 * CUDA events on the context's stream.  out4[0] = ms per application (both kernels), out4[1] / out4[2] =
 * ms per launch of its first / second kernel timed alone, out4[3] = kernels launched by this call.  For the 16-bit
 * Mpc the first kernel is the one mdwf_solve launches (K1 reading the B p stream of the fused CG update), unless the
 * option "bp_stream" is "0". */
int mdwf_time_op(mdwf_ctx *ctx, int op, const char *precision, int reps, int warmup, double *out4);

/* Measurement of the ALU roofline denominators: the device's fp32 fused-multiply-add
 * rate with scalar FFMA (tfma2[0]) and with the packed f32x2 FFMA2 the fp32-arithmetic kernels use (tfma2[1]),
 * in 1e12 FMA per second (two flops each), 16 independent chains per thread on every SM. */
int mdwf_fma_rates(mdwf_ctx *ctx, double *tfma2);

/* L2 -> SM delivery rates and DRAM streaming rates of this device, GB/s (best of 3): out4[0] 16-byte LDG bypassing L1
 * (ld.global.cg) over a 64 MB L2-resident buffer read 40 times by all SMs; out4[1] the same buffer through bulk-asynchronous
 * copies (cp.async.bulk, 2 CTAs per SM x 6 stages x 16 KB in flight); out4[2] / out4[3] the two kernels streaming 4 GB
 * from DRAM.  These are the ceilings the hop kernels' L2 traffic is judged against (profiles/r02_l2_sm_ceiling.md). */
int mdwf_l2_rates(mdwf_ctx *ctx, double *out4);

/* The batched operator of mdwf_apply_batch on nrhs right-hand sides held in library buffers, timed with
 * CUDA events: out2[0] = ms per batched application (K1 + K2, two launches for the whole batch), out2[1] = kernels launched.
 * precision "fp32" | "half"; op MDWF_OP_MPC or MDWF_OP_MPCDAG; 1 <= nrhs <= 64. */
int mdwf_time_op_batch(mdwf_ctx *ctx, int op, const char *precision, int nrhs, int reps, int warmup, double *out2);

#ifdef __cplusplus
}
#endif
#endif /* MDWF_BENCH_H */
