/*
 * twq_testing.h -- hooks for the test-suite and the bench harness.  NOT part of the product ABI (include/twq.h):
 * nothing here changes what a call computes, only which launch plan the planner picks, so that small test shapes
 * can reach the code paths that production shapes take (CTA pairs, unsplit tiles, forced cluster sizes), and a way
 * to read the plan back.  The planner never reads the environment.
 */
#ifndef TWQ_TESTING_H_
#define TWQ_TESTING_H_

#include <stddef.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Bits of the process-wide planner override word (0 = production behaviour). */
#define TWQ_PLAN_NO_SPLIT      1u    /* tcgen05 kernel: no K split for shapes with few output tiles */
#define TWQ_PLAN_NO_PAIR       2u    /* tcgen05 kernel: no CTA pairs (cta_group::2) */
#define TWQ_PLAN_NO_YSTAGE     4u    /* tcgen05 kernel: finished tiles are stored from registers, no staged TMA store */
#define TWQ_PLAN_NO_ALIAS2     8u    /* tcgen05 kernel: the stage-1 ring may not overlay the L2T tile */
#define TWQ_PLAN_NO_DECODE     16u   /* small batches go to the tcgen05 kernel as well */
#define TWQ_PLAN_FUSED_CS(c)   (((unsigned)(c) & 15u) << 8)    /* forced cluster size of the tcgen05 kernel */
#define TWQ_PLAN_DECODE_CS(c)  (((unsigned)(c) & 31u) << 12)   /* forced cluster size of the small-batch kernel */
#define TWQ_PLAN_FUSED_TN_CAP(c) (((unsigned)(c) & 3u) << 17)   /* tcgen05 kernel token tile: 1 = at most 64, 2 = at most 32 */

void twq_testing_set_plan_flags(unsigned flags);
unsigned twq_testing_get_plan_flags(void);

/* Fields written by twq_testing_describe_plan (ints). */
enum {
    TWQ_PLAN_KERNEL = 0,       /* 0 = small-batch (decode) kernel, 1 = tcgen05 kernel */
    TWQ_PLAN_CLUSTER,          /* CTAs per cluster */
    TWQ_PLAN_GRID,             /* CTAs */
    TWQ_PLAN_TILE_TOKENS,      /* tokens per tile (padded tokens for the small-batch kernel) */
    TWQ_PLAN_SPLITS,           /* K splits */
    TWQ_PLAN_PAIR,             /* 1 = CTA pairs */
    TWQ_PLAN_SMEM,             /* dynamic shared memory, bytes */
    TWQ_PLAN_RING,             /* ring depth of the packed-operand pipeline */
    TWQ_PLAN_CHUNKS,           /* small-batch kernel: ring chunks per call; tcgen05 kernel: work units */
    TWQ_PLAN_S1RING,           /* depth of the stage-1 (X, L1) ring */
    TWQ_PLAN_ALIAS,            /* tcgen05 kernel: 1 / 2 = the stage-1 ring overlays the residual rings (/ and the L2T tile) */
    TWQ_PLAN_FIELDS
};
/* The launch plan twq_dual_linear would use for this shape on the current device (or the no-device defaults).
 * Writes up to n_out ints; returns the number of fields, or -1 for an invalid shape. */
int twq_testing_describe_plan(int M, int N, int K, int r, int G, int* out, int n_out);

/* Measured dense int8 tensor rate in TOP/s: an MMA-only loop of tcgen05.mma kind::i8 (128 x 128 x 32) on every SM
 * (csrc/peak_i8.cu), best of `reps` launches of iters x 8 MMAs per SM.  SYNCHRONISES the stream.  Negative on failure.
 * bench.py prints it next to the 2 x BF16 figure that the prefill roofline uses. */
float twq_testing_measure_i8_tops(int iters, int reps, void* stream);

/* Cold-fill probe (csrc/cold_fill.cu): ONE launch of `ctas` CTAs (one per SM), each bringing `bytes` (a multiple of 64, at most
 * 200 KiB) from src + cta * stride into its shared memory -- mode 0: four bulk copies completing on an mbarrier (the small-batch
 * kernel's mechanism), mode 1: plain 16-byte loads, eight in flight per thread.  out_ns[cta] (device, ctas x u64) receives the
 * %globaltimer nanoseconds from the CTA's first instruction to its last byte.  Asynchronous on `stream`.  The caller provides
 * the buffer (ctas * stride bytes per region) and rotates regions so that nothing is L2-resident: the result is the floor under
 * any decode-shaped call that streams its weights once, which the bytes / bandwidth roofline ignores.  Returns 0, -1 (bad
 * argument / no sm_100 device) or -2 (launch failure). */
int twq_testing_cold_fill(const void* src, size_t stride, int bytes, int mode, int ctas, unsigned long long* out_ns, void* stream);

/* In-kernel timeline (csrc/trace.cuh).  Hands a device buffer of at least 16384 unsigned 64-bit words to the library;
 * NULL switches the timeline off.  Returns 1 if this library was built with the timeline compiled in
 * (`python -m paper_2606_01556_b200._build --trace` -> libtwq_trace.so), 0 if not (the product library: the call has
 * no effect). */
int twq_testing_set_trace_buffer(void* dev_buf);

#ifdef __cplusplus
}
#endif
#endif /* TWQ_TESTING_H_ */
