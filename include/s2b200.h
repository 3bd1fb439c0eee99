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
/* Same scatter, from arrays that already live in device memory (same layouts and NULL rules as s2_set_j).
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

/* Restricts the j-sum of subsequent s2_calc_* calls to the addresses first .. first+count-1 of the predicted store
 * (count == 0: every predicted particle again, the default).  This is one device's share when the j-particles are
 * distributed over several GPUs and the partial results added (sec 2.2.3, sec 3.6): each
 * rank keeps the whole store -- 116 bytes per particle -- predicts all of it, and sums over its own block; nearest-
 * neighbour and list addresses stay global.  The range must lie inside the predicted particles (else S2_ERANGE). */
int s2_set_j_range(s2_ctx *ctx, int first, int count);

/* --- a3-a8: forces on an i-list ---------------------------------- */

/* i-particles given as addresses into the predicted j-store (their state is the device-
 * predicted one).  h2: squared neighbour radii, one per i, required iff S2_WANT_NGB.
 * host-pointer form: ASYNC after an internal pinned copy. */
int s2_calc_ilist(s2_ctx *ctx, int ni, const int *i_address, const double *h2, double eps2,
                  unsigned flags);
/* k i-lists against the same predicted j-store in ONE launch sequence (a small call is bound by
 * launch, copy and synchronisation latency, not by arithmetic).  i_address holds the lists back to back (ni[0] + ... +
 * ni[k-1] entries, h2 likewise); the results of list b are entries offset_b .. offset_b + ni[b] - 1 of the next
 * s2_get_results / s2_get_neighbours* call over the concatenation, offset_b = ni[0] + ... + ni[b-1].  i-particles are
 * independent of one another, so this is the force call on the concatenated list (the launch shape, hence the
 * summation order and the last bits, are those of that list; decisions and lists are identical).  Host pointers.
 * ASYNC.  (Device-resident callers reach the same effect by capturing s2_calc_ilist_device calls in a CUDA graph: the
 * library enqueues nothing but kernels on that path.) */
int s2_calc_ilist_batch(s2_ctx *ctx, int k, const int *ni, const int *i_address, const double *h2, double eps2,
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
/* The same results written into DEVICE arrays of the caller (same shapes; any may be NULL), by a kernel enqueued
 * behind the force call: nothing crosses the host link and nothing synchronises, so a device-resident consumer
 * (an integrator kernel, a collective over j-sharded partial results) can follow directly.
 * Truncated lists are not reported here (s2_get_results / s2_get_neighbours_csr do).  ASYNC. */
int s2_get_results_device(s2_ctx *ctx, int ni, double *d_acc, double *d_jerk, double *d_snap, double *d_pot,
                          int *d_nn_id, double *d_nn_r2, int *d_ngb_count);
/* Neighbour list of the i-th entry of the i-list: j addresses, ascending, at most
 * min(cap, ngb_cap) entries; *n_out = number written.  SYNC. */
int s2_get_neighbours(s2_ctx *ctx, int i, int cap, int *n_out, int *list);
/* All lists in CSR form: offsets has ni+1 entries, list has offsets[ni] <= list_cap entries
 * (S2_ERANGE if list_cap is too small; offsets are still written so the caller can resize).
 * The lists are compacted ON THE DEVICE (count -> exclusive scan -> fill): only the offsets and the
 * offsets[ni] list members cross the host link, not the fixed-stride ni x ngb_cap buffer.  The compaction runs once
 * per force call and is cached, so a sizing call (list == NULL, list_cap == 0) followed by the real one costs one
 * compaction.  Returns S2_EOVERFLOW (output still written) if any list of the last call was truncated.  SYNC. */
int s2_get_neighbours_csr(s2_ctx *ctx, int ni, long long *offsets, int *list, long long list_cap);
/* The same CSR, left in device memory for device-resident callers: *d_offsets points at ni_last+1 64-bit offsets,
 * *d_list at the compacted addresses (both context-owned, valid until the next s2_calc_* or s2_close);
 * *total = offsets[ni].  SYNC (one 8-byte read). */
int s2_get_neighbours_csr_device(s2_ctx *ctx, int ni, const long long **d_offsets, const int **d_list, long long *total);

/* --- a5 + a6 without any allocation (PAPER.md L52-L54 j-split, L88 combine of the partial results) ------------ */

/* For callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops, harnesses that forbid
 * it): 4th-order fp64 acc, jerk and pot of ni i-particles from nj predicted j-particles, as a j-split sweep plus a
 * fixed-order combine whose partial sums live in a STATIC device array of the library (4 MiB; every GPU that loads
 * the library holds it until the process exits).  Needs no context.  It calls no cudaMalloc, cudaFree or allocating
 * library routine: cudaSetDevice(device), once per device a symbol-address lookup, two kernel launches.
 *   device pointers, caller-owned: d_pos, d_vel (nj,3) predicted state; d_mass, d_id (nj); d_i_address (ni) addresses
 *   into those arrays (an address outside [0, nj) gives NaN results for that i, nothing faults);
 *   outputs d_acc, d_jerk (ni,3), d_pot (ni).  Conventions as above (self skipped by id, pot negative, G = 1).
 * Limit: ni <= 4096 (s2_noalloc_limits); larger i-lists return S2_ERANGE -- use the context calls for those.
 * The scratch array is shared by all calls on a device and keeps the last call's contents; nothing in it needs
 * clearing (every row read was written by the same call).  Calls that overlap on the GPU (two streams, two threads)
 * RACE on it: the caller serialises them.  Results are bit-reproducible run to run.  ASYNC on cuda_stream. */
int s2_forces_noalloc(int device, void *cuda_stream, int nj, const double *d_pos, const double *d_vel,
                      const double *d_mass, const int *d_id, int ni, const int *d_i_address, double eps2,
                      double *d_acc, double *d_jerk, double *d_pot);
/* The fixed maxima of s2_forces_noalloc: largest ni, and the bytes of the static scratch array (either may be NULL). */
int s2_noalloc_limits(int *max_ni, long long *scratch_bytes);

/* --- block-time-step Hermite integrator on the device (sec 3.7) -------- */

/* The second workload of the paper: a 4th- or 6th-order Hermite predictor-corrector with block (power-of-two,
 * block-aligned) individual time steps, which calls the hot path above with an active set that varies between 1 and N
 * from step to step.  Everything runs in kernels on the context's stream: the particle state is the context's own
 * j-store (the corrector updates it in place, so nothing is re-sent), the corrector and the time-step criterion
 * (Aarseth, L152: eta_4 = 0.01, eta_6 = 0.1), the choice of the next block time and the compaction of the next
 * active list.  Per ordinary block step the host reads back 12 bytes (next time, next active count) after one stream
 * synchronisation -- it needs the count to shape the next force launch; in S2_FP64 contexts runs of small steps (at most
 * 512 active particles, no more than 512 particles per SM) are taken by one cooperative launch that stays on the GPU
 * from step to step, and the host synchronises once per run.  Both ways give the same run: same block times and active
 * sets, states equal to rounding (the sums are taken in another order).  paper_1510_04068_b200/hermite.py is the host
 * reference driver of the same schemes (textbook formulas, refs [27] and [5]).
 * The integrator takes over the j-store of `ctx` (addresses 0 .. n-1, id == address); between s2_bts_run calls the
 * ordinary calls (s2_predict, s2_calc_*, s2_get_*) may be used on the same context, s2_set_j / s2_commit_j may not. */
typedef struct s2_bts s2_bts; /* opaque */

/* ctx: an order-4 or order-6 context (any precision) with nj_capacity >= n.  dt_max, dt_min: powers of two <= 1.
 * eta: accuracy parameter of the step criterion (4th order: Aarseth; 6th order: its generalisation, ref [5]);
 * eta_start: that of the first step, dt = eta_start |a| / |jerk|.
 * averaged != 0 (order 6 only): the step is the mean of the generalised criterion and the 4th-order Aarseth step with
 * accuracy parameter eta4 -- the choice of the paper's runs (L156), which keeps double-single forces from driving the
 * step to zero. */
int s2_bts_open(s2_bts **out, s2_ctx *ctx, int n, double eps2, double eta, double eta_start, double dt_max, double dt_min,
                int averaged, double eta4);
int s2_bts_close(s2_bts *b);
/* Initial conditions at t = 0: host arrays mass (n), pos, vel (n,3).  Runs the start-up force evaluation (two passes
 * for order 6: the snap needs every particle's acceleration), sets the first steps and the first active list.  SYNC. */
int s2_bts_init(s2_bts *b, const double *mass, const double *pos, const double *vel);
/* Advances block step by block step while the next block time is <= t_end, at most max_block_steps steps
 * (*steps_done, may be NULL).  If t_end is a multiple of dt_max every particle ends at exactly t_end.
 * time_device != 0 also accumulates the device time of the steps' kernels between CUDA events (s2_bts_stats).  SYNC. */
int s2_bts_run(s2_bts *b, double t_end, long long max_block_steps, int time_device, long long *steps_done);
/* Per-particle state, each particle at its own time t[i] (host arrays of n or (n,3); any may be NULL).  SYNC. */
int s2_bts_get_state(s2_bts *b, double *time, double *t, double *dt, double *pos, double *vel, double *acc, double *jerk,
                     double *pot);
/* Counters since s2_bts_init (any pointer may be NULL): current time, next block time and its active count, block
 * steps, particle steps (sum of the active counts), host wall time inside s2_bts_run, and -- for steps run with
 * time_device -- the summed device time and their number. */
int s2_bts_stats(const s2_bts *b, double *time, double *t_next, int *n_next, long long *block_steps,
                 long long *particle_steps, double *wall_ms, double *device_ms, long long *timed_steps);
/* Active counts of block steps first .. first+count-1 since s2_bts_init. */
int s2_bts_get_history(const s2_bts *b, long long first, int count, int *n_active);

/* --- read-back hooks and diagnostics (tuning overrides and microbenchmarks: s2b200_test.h) --- */

/* fp64 predicted state of j-particles first .. first+n-1 ((n,3) arrays, any may be NULL;
 * acc = predicted acceleration for order 6, undefined for order 4).  SYNC. */
int s2_get_predicted_j(s2_ctx *ctx, int first, int n, double *pos, double *vel, double *acc);
/* stored (unpredicted) state: id, t, mass (n) and pos (n,3); any may be NULL.  SYNC. */
int s2_get_j(s2_ctx *ctx, int first, int n, int *id, double *t, double *mass, double *pos);

/* Number of kernels this context has launched since s2_open. */
long long s2_kernel_launches(const s2_ctx *ctx);
/* When enabled, CUDA events bracket each kernel of predict / calc on the context's stream. */
int s2_enable_timing(s2_ctx *ctx, int on);
/* Device time in milliseconds of the kernels of the last s2_predict and the last s2_calc_*
 * (force sweep, reduce/compaction); 0 for kernels that did not run.  SYNC. */
int s2_get_timing(s2_ctx *ctx, float *predict_ms, float *force_ms, float *reduce_ms);

const char *s2_strerror(int code);
/* cudaGetErrorString of the last CUDA failure seen by this context ("" if none). */
const char *s2_last_cuda_error(const s2_ctx *ctx);
/* Library version string, e.g. "s2b200 0.1 (sm_100a)". */
const char *s2_version(void);

#ifdef __cplusplus
}
#endif
#endif /* S2B200_H */
