/*
 * s2b200.h -- C ABI of the B200-native direct N-body force library
 * (the data-parallel hot path of "Sapporo2: a versatile direct N-body library",
 *  arXiv:1510.04068; citations below are lines of PAPER.md).
 *
 * The paper states the problem in GRAPE terms -- "support for the GRAPE API" (L32),
 * GRAPE-5 / GRAPE-6 style calls (L34), "how the GRAPE hardware operates" (L92) -- and
 * prints no function signature.  The call set follows that statement of the problem:
 * open/close, set j-particle, predict-to-time, compute forces for an i-list, read
 * results and neighbour lists (sec 2.2.4: copy kernel, predict kernel, gravity
 * kernel; sec 3: acc, jerk, nearest neighbour, neighbour list; sec 2.2.2:
 * storage always fp64, precision chosen at run time; sec 2.1: i = sinks,
 * j = sources, j-split for few sinks).
 *
 * General rules
 *   - Plain C: pointers and sizes only.  "host" pointers are ordinary (pageable or
 *     pinned) CPU memory; "device" pointers are CUDA device memory on the context's
 *     device.  The caller owns every array it passes, before and after the call; the
 *     library copies in and out and keeps no reference after the call returns.
 *   - The context owns all device buffers.  They come from the s2_allocator callbacks
 *     given to s2_open (PyTorch's caching allocator in the Python binding) or, when the
 *     allocator is NULL, from cudaMalloc.  s2_close releases them.
 *   - All kernels and copies are enqueued on the CUDA stream given to s2_open (a
 *     cudaStream_t passed as void*; NULL = legacy default stream).  Calls marked ASYNC
 *     return after enqueueing; calls marked SYNC synchronise that stream.
 *   - Every call returns S2_OK (0) or a negative code; no exception crosses the ABI.
 *     Asynchronous CUDA errors surface at the next SYNC call as S2_ECUDA.
 *   - Ordering: s2_predict needs committed j-particles; s2_calc_* uses the state of the
 *     last s2_predict; s2_get_* refer to the last s2_calc_*.  Violations give S2_ESTATE.
 *   - A context is not thread-safe; distinct contexts are independent.
 *   - There is no CPU fallback: without a usable CUDA device s2_open fails with S2_ECUDA.
 *
 * Conventions (the paper is silent on all of them; DESIGN.md lists the readings)
 *   - G = 1; results are accelerations, not forces.  Plummer softening eps2 enters
 *     acc, jerk, snap and pot, not the neighbour distances.
 *   - pot_i = - sum_j m_j / sqrt(r_ij^2 + eps2)   (negative).
 *   - self-interaction is skipped by identity: id_j == id_i, for every output.
 *   - nearest neighbour: the j with the smallest unsoftened r_ij^2, j != i; ties go to
 *     the lowest j address; returned as that particle's id and r_ij^2 (squared).  No
 *     candidate: id = -1, r2 = +inf.
 *   - neighbour of i: r_ij^2 < h2_i (strict), j != i.  ngb_count is the true count; a
 *     list holds at most ngb_cap members, the lowest j addresses, ascending.
 *   - the two integer decisions use d2 = fma(dz,dz, fma(dy,dy, dx*dx)) evaluated in
 *     IEEE fp64 on the fp64 predicted positions, in every precision mode.
 */
#ifndef S2B200_H
#define S2B200_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct s2_ctx s2_ctx; /* opaque */

/* pair-arithmetic precision ("converted to either float or double-single";
 * native fp64 L128).  Storage is fp64 in all modes. */
enum { S2_FP64 = 0, S2_DS = 1, S2_FP32 = 2 };

/* per-call output flags (nearest neighbour and neighbour list "can be
 * disabled by changing a template parameter") */
enum { S2_WANT_NN = 1, S2_WANT_NGB = 2 };

/* return codes */
enum {
    S2_OK = 0,
    S2_EINVAL = -1,    /* bad argument (NULL where required, n < 0, unknown order/precision/flag) */
    S2_ERANGE = -2,    /* address outside [0, nj_capacity), n larger than a capacity */
    S2_ENOMEM = -3,    /* allocator returned NULL */
    S2_ECUDA = -4,     /* CUDA runtime error (see s2_last_cuda_error) or no device */
    S2_ESTATE = -5,    /* call order violated */
    S2_EOVERFLOW = -6  /* some neighbour list exceeded ngb_cap; all other results are valid,
                          counts are true counts, lists are truncated to the lowest addresses */
};

/* Device-memory callbacks.  alloc returns a device pointer aligned to >= 256 bytes or NULL. */
typedef struct {
    void *(*alloc)(size_t bytes, void *user);
    void (*free)(void *ptr, void *user);
    void *user;
} s2_allocator;

/* --- life cycle ----------------------------------------------------------------------- */

/* Creates a context on CUDA device `device`.
 *   order        2 (GRAPE-5 style, L34: acc and pot only), 4 (GRAPE-6 style: acc, jerk) or
 *                6 (also snap; j carries snap and crackle) [L34, L76]
 *   precision    S2_FP64 | S2_DS | S2_FP32
 *   nj_capacity  maximum number of j-particles (addresses 0 .. nj_capacity-1)
 *   ngb_cap      maximum neighbour-list length kept per i (e.g. 256); 0 disables lists
 *   a            allocator callbacks or NULL (cudaMalloc/cudaFree)
 *   cuda_stream  cudaStream_t as void*
 * SYNC (allocation). */
int s2_open(s2_ctx **out, int device, int order, int precision, int nj_capacity, int ngb_cap,
            const s2_allocator *a, void *cuda_stream);
int s2_close(s2_ctx *ctx);
int s2_set_stream(s2_ctx *ctx, void *cuda_stream);
/* Waits for everything enqueued so far.  SYNC. */
int s2_synchronize(s2_ctx *ctx);

/* --- a1: set / commit j-particles ("copy kernel"; L76 fp64 storage) -------- */

/* Stages n j-particles in pinned host memory (host pointers; pos..crackle are (n,3) row-major;
 * snap and crackle may be NULL when order <= 4, in which case they are ignored; acc and jerk may be NULL when
 * order == 2 and are then stored as zero, so that the predictor reduces to x + v dt).
 * address[k] is the slot in the j-store, id[k] >= 0 the identity used for the self test.
 * May be called several times before one s2_commit_j.  Host-only, no GPU work. */
int s2_set_j(s2_ctx *ctx, int n, const int *address, const int *id, const double *t,
             const double *mass, const double *pos, const double *vel, const double *acc,
             const double *jerk, const double *snap, const double *crackle);
/* Copies the staged particles to the device and scatters them into the SoA j-store. ASYNC. */
int s2_commit_j(s2_ctx *ctx);
/* Same scatter, from arrays that already live in device memory (same layouts as s2_set_j).
 * Address range is the caller's responsibility here (checked on the device: out-of-range
 * entries are dropped and reported as S2_ERANGE at the next SYNC call).  ASYNC. */
int s2_commit_j_device(s2_ctx *ctx, int n, const int *d_address, const int *d_id, const double *d_t,
                       const double *d_mass, const double *d_pos, const double *d_vel,
                       const double *d_acc, const double *d_jerk, const double *d_snap,
                       const double *d_crackle);

/* --- a2: predict ("one kernel to predict the particles to the new time-step") */

/* Taylor-predicts j-particles 0 .. nj-1 to time t (dt = t - t_j, any sign):
 *   2nd and 4th order: x_p through jerk, v_p through jerk;  6th order: x_p, v_p, a_p through crackle.
 * Subsequent s2_calc_* calls sum over exactly these nj particles.  ASYNC. */
int s2_predict(s2_ctx *ctx, double t, int nj);

/* --- a3-a8: forces on an i-list ---------------------------------- */

/* i-particles given as addresses into the predicted j-store (their state is the device-
 * predicted one).  h2: squared neighbour radii, one per i, required iff S2_WANT_NGB.
 * host-pointer form: ASYNC after an internal pinned copy. */
int s2_calc_ilist(s2_ctx *ctx, int ni, const int *i_address, const double *h2, double eps2,
                  unsigned flags);
/* device-pointer form of the same call (arrays must stay valid until the next SYNC). ASYNC. */
int s2_calc_ilist_device(s2_ctx *ctx, int ni, const int *d_i_address, const double *d_h2,
                         double eps2, unsigned flags);
/* i-particles given explicitly (sinks need not be sources, L46).  id[k] < 0 matches no j.
 * acc is read only when order == 6 (relative acceleration for snap); vel may be NULL when order == 2.
 * host pointers. ASYNC. */
int s2_calc_explicit(s2_ctx *ctx, int ni, const int *id, const double *pos, const double *vel,
                     const double *acc, const double *h2, double eps2, unsigned flags);

/* --- a9: read results ("transfer of the force computation results") -------- */

/* Results of the last s2_calc_* for i = 0 .. ni-1 (position in the i-list).  Any output
 * pointer may be NULL.  acc/jerk/snap are (ni,3); snap is written only when order == 6; jerk is zero when
 * order == 2.
 * nn_id/nn_r2 are meaningful only if S2_WANT_NN was set, ngb_count only if S2_WANT_NGB.
 * Returns S2_EOVERFLOW (results still written) if any list was truncated.  SYNC. */
int s2_get_results(s2_ctx *ctx, int ni, double *acc, double *jerk, double *snap, double *pot,
                   int *nn_id, double *nn_r2, int *ngb_count);
/* Neighbour list of the i-th entry of the i-list: j addresses, ascending, at most
 * min(cap, ngb_cap) entries; *n_out = number written.  SYNC. */
int s2_get_neighbours(s2_ctx *ctx, int i, int cap, int *n_out, int *list);
/* All lists in CSR form: offsets has ni+1 entries, list has offsets[ni] <= list_cap entries
 * (S2_ERANGE if list_cap is too small; offsets are still written so the caller can resize). SYNC. */
int s2_get_neighbours_csr(s2_ctx *ctx, int ni, long long *offsets, int *list, long long list_cap);

/* --- test hooks and diagnostics ---------------------------------------------------------- */

/* fp64 predicted state of j-particles first .. first+n-1 ((n,3) arrays, any may be NULL;
 * acc = predicted acceleration for order 6, undefined for order 4).  SYNC. */
int s2_get_predicted_j(s2_ctx *ctx, int first, int n, double *pos, double *vel, double *acc);
/* stored (unpredicted) state: id, t, mass (n) and pos (n,3); any may be NULL.  SYNC. */
int s2_get_j(s2_ctx *ctx, int first, int n, int *id, double *t, double *mass, double *pos);

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
 *          i-list from, and write the final records to, pinned host memory, so no copy is enqueued) */
int s2_set_tuning(s2_ctx *ctx, int key, int value);
/* Shape of the last force launch: out[0]=S, [1]=lanes per i, [2]=warp columns, [3]=grid size,
 * [4]=threads per CTA, [5]=dynamic shared memory bytes, [6]=0 no combine needed / 1 reduce kernel ran /
 * 2 combine fused into the sweep launch (last CTA of each i-group reduces, fixed order) / 3 uniform-operand
 * sweep: out[0] is then the number of chunk launches (sums carried in address order, nothing to combine) /
 * 4 combined by atomics (key 5 = 2),
 * [7]=resident CTAs per SM (occupancy query), [8]=i-particles per thread (register-tiled sweep when > 1),
 * [9]=CTAs per cluster. */
int s2_last_launch_info(const s2_ctx *ctx, int out[10]);
/* Number of kernels this context has launched since s2_open. */
long long s2_kernel_launches(const s2_ctx *ctx);
/* When enabled, CUDA events bracket each kernel of predict / calc on the context's stream. */
int s2_enable_timing(s2_ctx *ctx, int on);
/* Device time in milliseconds of the kernels of the last s2_predict and the last s2_calc_*
 * (force sweep, reduce/compaction); 0 for kernels that did not run.  SYNC. */
int s2_get_timing(s2_ctx *ctx, float *predict_ms, float *force_ms, float *reduce_ms);

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

/* Test hook for the double-single arithmetic of the S2_DS path (reading P11): for k < n (host arrays) the operands
 * a[k], b[k] are split into (hi, lo) float pairs on the device and out[8k .. 8k+7] receives, as fp64,
 *   [0] the round trip of a   [1] a + b   [2] a - b (cancellation-safe form)   [3] a b   [4] a^2   [5] -3 a
 *   [6] |a|^(-1/2)   [7] a b + a.   SYNC. */
int s2_test_ds_ops(s2_ctx *ctx, int n, const double *a, const double *b, double *out);

const char *s2_strerror(int code);
/* cudaGetErrorString of the last CUDA failure seen by this context ("" if none). */
const char *s2_last_cuda_error(const s2_ctx *ctx);
/* Library version string, e.g. "s2b200 0.1 (sm_100a)". */
const char *s2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* S2B200_H */
