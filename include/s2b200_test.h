/*
 * s2b200_test.h -- test hooks, tuning overrides and microbenchmarks of libs2b200.so.
 *
 * NOT part of the product ABI of include/s2b200.h: these entry points exist so that the parity tests can force
 * every launch shape, so that bench.py can measure roofline denominators in the same process, and so that the
 * double-single arithmetic can be pinned operand by operand.  A production caller needs none of them.
 */
#ifndef S2B200_TEST_H
#define S2B200_TEST_H

#include "s2b200.h"

#ifdef __cplusplus
extern "C" {
#endif

/* Launch-shape overrides for tests and tuning sweeps; value 0 restores the automatic choice.
 *   key 0: number of j-slices S      key 1: lanes per i-particle (1,2,4,..,32)
 *   key 2: warp columns over j (1,2,4,8; only with lanes == 32)
 *   key 3: CTAs per SM assumed by the balancer      key 4: j-tile length (multiple of 32)
 *   key 5: 1 = combine j-slices with the separate reduce kernel even when the fused combine applies,
 *          2 = combine them with fp64 atomics on the final records instead (the paper's Sapporo2 scheme, L88): one
 *          launch, but the last bits then vary run to run; ignored when NN / neighbour lists are requested,
 *          3 = use the fused combine (last CTA of each i-group) whenever the shape allows it
 *   key 6: CTAs per thread-block cluster along the slice axis in the fused combine (1 = none, 2, 4, 8)
 *   key 7: 1 = never use the register-tiled sweep (several i per thread), 2 = always use it
 *   key 8: 1 = never use the uniform-operand sweep (j-particles read chunk by chunk from the constant bank, one
 *          launch per chunk; fp64 only), 2 = always use it when the context computes in fp64
 *   key 9: 1 = never use the zero-copy path of small host calls (n_i <= 128 with host arrays: the kernels read the
 *          i-list from, and write the final records to, pinned host memory, so no copy is enqueued),
 *          4 = S2_FP32 contexts: no fp64 re-evaluation of ill-conditioned i-particles (A/B of reading R-F32),
 *          5 = S2_FP32 contexts: re-evaluate EVERY i-particle in fp64 (tests of the fix-up kernels: the sums are then fp64-accurate),
 *          6 = block-step integrator: the small-step kernel is not used (every step through the ordinary force call, one
 *              synchronisation per step; A/B of s2_bts_run)
 *   key 10: block-step integrator: largest active set the small-step kernel takes (1 .. 1024; 0 = the default, 512) */
int s2_set_tuning(s2_ctx *ctx, int key, int value);
/* Shape of the last force launch: out[0]=S, [1]=lanes per i, [2]=warp columns, [3]=grid size,
 * [4]=threads per CTA, [5]=dynamic shared memory bytes, [6]=0 no combine needed / 1 reduce kernel ran /
 * 2 combine fused into the sweep launch (last CTA of each i-group reduces, fixed order) / 3 uniform-operand
 * sweep: out[0] is then the number of chunk launches (sums carried in address order, nothing to combine) /
 * 4 combined by atomics (key 5 = 2),
 * [7]=resident CTAs per SM (occupancy query), [8]=i-particles per thread (register-tiled sweep when > 1),
 * [9]=CTAs per cluster. */
int s2_last_launch_info(const s2_ctx *ctx, int out[10]);
/* Host wall time, in microseconds per call, of s2_calc_ilist + s2_get_results (all outputs but neighbour lists)
 * repeated `reps` times after 3 warm-up calls, measured inside the library with the steady clock: the latency of
 * a small force call as a C caller sees it (BASELINE config 2; PAPER.md L114, L124 on small-n_i overheads), without
 * any binding layer.  i_address: host array of ni addresses.  S2_WANT_NGB is not accepted.  SYNC. */
int s2_time_host_roundtrip(s2_ctx *ctx, int ni, const int *i_address, double eps2, unsigned flags, int reps,
                           double *us_per_call);

/* Peak microbenchmarks used as roofline denominators and for the FP64 operand-path model:
 * a grid that fills the device runs `iters` rounds of 8 independent chains per thread.
 *   kind 0 = DFMA with constant operands (nominal fp64 rate)      1 = FFMA (fp32)
 *   kind 2 = DFMA with three distinct 64-bit register operands    3 = DFMA with one operand shared by
 *   consecutive instructions (operand-reuse cache)                 4 = DADD with two distinct register operands
 *   kind 5-8 = packed FP32 (two lane-operations per instruction, both counted): 5 = FFMA2 with constant operands,
 *   6 = FFMA2 with three distinct register pairs, 7 = FFMA2 with a 32-bit register broadcast to both halves,
 *   8 = FADD2 with two distinct register pairs
 * Returns achieved lane-instructions per second in *fma_per_s.  SYNC. */
int s2_peak_fma(s2_ctx *ctx, int kind, int iters, double *fma_per_s);

/* Latency of an exchange between SMs through L2, the floor under the integrator's small-step kernel: CTA 0 stores a
 * word, each of the other ctas - 1 CTAs (one per SM, 2 <= ctas <= SM count) polls it and answers in a word of its own,
 * CTA 0 polls all answers; relaxed gpu-scope accesses, no fences.  Returns SM cycles (clock64) per round trip = two
 * hops, averaged over iters.  SYNC. */
int s2_hop_latency(s2_ctx *ctx, int ctas, int iters, double *cycles_per_round_trip);

/* Test hook for the double-single arithmetic of the S2_DS path (reading P11): for k < n (host arrays) the operands
 * a[k], b[k] are split into (hi, lo) float pairs on the device and out[8k .. 8k+7] receives, as fp64,
 *   [0] the round trip of a   [1] a + b   [2] a - b (cancellation-safe form)   [3] a b   [4] a^2   [5] -3 a
 *   [6] |a|^(-1/2)   [7] a b + a.   SYNC. */
int s2_test_ds_ops(s2_ctx *ctx, int n, const double *a, const double *b, double *out);

/* Device time in milliseconds of the last neighbour-list compaction (scan kernels + fill kernel, s2_ngb.cu), when
 * s2_enable_timing is on; the bytes it moved are 20 B per i-particle + 8 B per list member.  SYNC. */
int s2_get_csr_timing(s2_ctx *ctx, float *scan_ms, float *fill_ms);

/* S2_FP32 contexts: number of i-particles of the last force call whose jerk sum was found ill-conditioned and that were
 * re-evaluated in fp64 (reading R-F32); 0 for other precisions.  SYNC. */
int s2_fp32_fixup_count(s2_ctx *ctx, int *n);

/* Block-step integrator (s2_bts_*, include/s2b200.h): how much of the run went through the small-step kernel -- its
 * launches, the block steps they ran, and (runs with time_device != 0) their summed device time in milliseconds. */
struct s2_bts;
int s2_bts_small_stats(const struct s2_bts *b, long long *launches, long long *steps, double *device_ms);
/* Where a step of the small-step kernel spends its time, as seen by one CTA: with on = 1 + the CTA's index (CTA 0 combines
 * and corrects the first active particle of every step, so it is on the critical path; CTAs beyond the active count only
 * sweep and wait) the kernel adds up the SM cycles (clock64) between its marks into ten sums that out (may be NULL)
 * receives -- [0] waiting for and scanning the owners' headers, [1] polling the records, [2] sweep, [3] adding the
 * j-splits and writing the rows, [4] polling and adding the rows of all owners, [5] corrector, [6] the grid barrier,
 * [7] histogram, reload, prediction, [8] publishing the next active set, [9] the number of steps.  Turning it on
 * zeroes the sums; on = 0 turns it off; s2_bts_init leaves it off.  SYNC. */
int s2_bts_small_profile(struct s2_bts *b, int on, long long out[10]);

#ifdef __cplusplus
}
#endif
#endif /* S2B200_TEST_H */
