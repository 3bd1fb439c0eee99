// s2_bts.cu -- device-resident block-time-step Hermite integrator (sec 3.7
// L152-L168: "sixth order Hermite integrator with block time-steps", Plummer spheres, energy errors 1e-12 / 1e-10).
//
// The paper's point in L156-L164 is that in a block-step run the time goes into everything AROUND the force kernel:
// picking the active set, the corrector, the time-step rule, and the traffic between host and device.  Here all of it
// stays on the GPU.  The particle state IS the library's base j-store (t_j, m, x, v, a, jerk [, snap, crackle] at each
// particle's own time): the corrector reads a particle's old state there and writes the new one in place, so there is
// no commit copy at all.  One block step is
//     force sweep (+ reduce) for the active list                              -- s2_api.cu run_force, shape by n_active
//     corrector            corrector + time-step rule + write-back, level histogram by integer atomics: inside reduce_kernel
//                          when the force call combines with it, else bts_correct_kernel (s2_bts_correct.cuh)
//     bts_select_predict_kernel   next block time from the histogram, ordered compaction of the next active list,
//                          prediction of every j to that time, {t_next, n_next} written to pinned host memory
// and the host reads 12 bytes after one stream synchronisation (it needs n_next to shape the next sweep).
// That is the ordinary step.  Most block steps, though, move a handful of particles, and three dependent launches plus a
// synchronisation cost 30 us for a microsecond of arithmetic: in fp64 contexts, runs of steps with at most 512 active
// particles are handed to ONE cooperative launch of bts_small_steps_kernel (s2_force_fp64.cu), which keeps every
// particle's state in the shared memory of the SM that owns it and runs step after step without leaving the GPU; it
// returns at the first step that does not qualify, with the control block, the list and the j-store as an ordinary step
// expects them.  The host then synchronises once per run of small steps.
//
// Block time steps are powers of two and block-aligned (t_i is a multiple of dt_i), hence
//     t_next = t_now + min_i dt_i        and        i is active at t_next  <=>  t_next is a multiple of dt_i,
// so neither a t_i + dt_i array nor a global min-reduction over particles is needed: the smallest step follows from a
// 64-bin histogram of step levels that the corrector keeps up to date.
//
// Corrector and time-step rule are the textbook ones of the schemes the paper names (4th order ref [27], 6th order
// ref [5]); they are written out in paper_1510_04068_b200/hermite.py (the host reference driver, which the tests run
// against the oracle in lock-step with this one) and repeated at the kernels below.
#include <math_constants.h>

#include <string.h>

#include <algorithm>
#include <chrono>

#include "s2_ctx.h"
#include "../../include/s2b200_test.h"
#include "s2_predict.cuh"
#include "s2_bts_correct.cuh"

using namespace s2;

namespace {

constexpr int kLevels = 64;          // dt = 2^-level, level 0 .. 63
constexpr int kSelThreads = 256;
constexpr int kSelPerBlock = kSelThreads;   // particles per block of the select kernel (one per thread)

// ---- start-up: first steps from acc and jerk alone, dt = eta_s |a| / |j| (hermite.py __init__) -------------------
__global__ void __launch_bounds__(256) bts_init_kernel(BtsArgs a, int final_pass)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.n) return;
    const double *r = a.rec + (size_t)i * REC;             // the start-up i-list is 0 .. n-1
    double ac[3] = {r[0], r[1], r[2]}, jk[3] = {r[3], r[4], r[5]};
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a.f[8 + c][i] = ac[c];
        a.f[11 + c][i] = jk[c];
        if (a.order == 6 && final_pass) a.f[14 + c][i] = r[9 + c];   // snap needs every particle's acceleration: second pass
    }
    a.pot[i] = r[6];
    if (!final_pass) return;
    const double raw = a.eta_start * norm3(ac) / fmax(norm3(jk), 1e-300);
    const double dt = fmin(fmax(pow2_floor(fmax(raw, a.dt_min)), a.dt_min), a.dt_max);
    a.dt[i] = dt;
    atomicAdd(&a.hist[level_of(dt)], 1);
}

// ---- corrector + time-step rule on the active particles: bts_correct_one (s2_bts_correct.cuh), one thread per particle.
// When the force call combines its j-slices with reduce_kernel, that kernel applies it itself (one launch less per block step).
__global__ void __launch_bounds__(128) bts_correct_kernel(BtsArgs a)
{
    // programmatic dependent launch along the chain sweep -> (reduce) -> correct -> select -> predict: every kernel lets
    // its successor be staged at once and waits for its predecessor's results itself
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= a.n_act) return;
    bts_correct_one(a, k, a.rec + (size_t)k * REC);
}

// ---- next block time, next active list, and the prediction of the j-store to that time: one launch -------------
// Every block (256 particles, one per thread) derives dt_min from the level histogram (64 parallel loads and two
// ballots), hence t_next = t_now + dt_min; predicts its particles to t_next (predict_one: the same arithmetic as
// predict_kernel); compacts its active particles (ascending) into its staging segment by ballot + popc and publishes
// its count.  The last block to arrive concatenates the segments in block order -- the list is ascending by address
// whatever the arrival order -- and writes {t_next, n_next} to the device control block and to pinned host memory.
template <int ORDER>
__global__ void __launch_bounds__(kSelThreads) bts_select_predict_kernel(BtsArgs a, PredictArgs pa, double t_now_host, int use_host_time)
{
    __shared__ int s_w[kSelThreads / 32];
    __shared__ unsigned s_hist[2];
    __shared__ int s_last;
    __shared__ int s_off[kSelThreads + 1];
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (threadIdx.x < kLevels) {
        const unsigned b = __ballot_sync(0xffffffffu, a.hist[threadIdx.x] > 0);
        if (lane == 0) s_hist[warp] = b;
    }
    __syncthreads();
    const int lev = s_hist[1] ? 63 - __clz(s_hist[1]) : 31 - __clz(s_hist[0] | 1u);   // highest occupied level = smallest step
    const double t_next = (use_host_time ? t_now_host : a.ctl->t_next) + scalbn(1.0, -lev);
    const int i = blockIdx.x * kSelThreads + threadIdx.x;
    bool act = false;
    if (i < a.n) {
        const double x = t_next / a.dt[i];               // exact: dt is a power of two
        act = x == floor(x);
        predict_one<ORDER>(pa, i, t_next);
    }
    const unsigned bal = __ballot_sync(0xffffffffu, act);
    if (lane == 0) s_w[warp] = __popc(bal);
    __syncthreads();
    int base = __popc(bal & ((1u << lane) - 1u));
    int total = 0;
#pragma unroll
    for (int w = 0; w < kSelThreads / 32; ++w) {
        if (w < warp) base += s_w[w];
        total += s_w[w];
    }
    if (act) a.stage[(size_t)blockIdx.x * kSelThreads + base] = i;
    if (threadIdx.x == 0) a.bcnt[blockIdx.x] = total;
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0) {
        const unsigned prev = atomicAdd(a.arrive, 1u);
        s_last = prev == gridDim.x - 1;
    }
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // last block: exclusive scan of the block counts, kSelThreads at a time, then a flat copy of each chunk's members
    int off = 0;
    for (int b0 = 0; b0 < (int)gridDim.x; b0 += kSelThreads) {
        const int b = b0 + threadIdx.x;
        const int c = b < (int)gridDim.x ? __ldcg(a.bcnt + b) : 0;
        int incl = c;
#pragma unroll
        for (int m = 1; m < 32; m <<= 1) {
            const int o = __shfl_up_sync(0xffffffffu, incl, m);
            if (lane >= m) incl += o;
        }
        __syncthreads();
        if (lane == 31) s_w[warp] = incl;
        __syncthreads();
        int wb = 0;
        for (int w = 0; w < warp; ++w) wb += s_w[w];
        s_off[threadIdx.x] = wb + incl - c;
        if (threadIdx.x == kSelThreads - 1) s_off[kSelThreads] = wb + incl;
        __syncthreads();
        const int chunk_total = s_off[kSelThreads];
        for (int k = threadIdx.x; k < chunk_total; k += kSelThreads) {
            int lo = 0, hi = kSelThreads - 1;            // block of member k: last lb with s_off[lb] <= k
            while (lo < hi) {
                const int mid = (lo + hi + 1) >> 1;
                if (s_off[mid] <= k) lo = mid; else hi = mid - 1;
            }
            a.ilist[off + k] = __ldcg(a.stage + (size_t)(b0 + lo) * kSelThreads + (k - s_off[lo]));
        }
        off += chunk_total;
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        *a.arrive = 0u;
        a.ctl->t_next = t_next;
        a.ctl->n_next = off;
        a.h_ctl->t_next = t_next;
        a.h_ctl->n_next = off;
    }
}

__global__ void bts_iota_kernel(int *p, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = i;
}

}  // namespace

namespace s2 {
cudaError_t launch_predict(const PredictArgs &a, cudaStream_t st);
cudaError_t launch_bts_small_steps(const ForceArgs &a, const BtsArgs &b, const PredictArgs &pa, int device, int sm_count, cudaStream_t st);
}

// Small block steps (fp64 contexts): runs of steps with at most kSmallCap active particles are taken by ONE launch of
// bts_small_steps_kernel (s2_force_fp64.cu), which sweeps, combines, corrects, selects and predicts step after step behind
// grid barriers and returns at the first step that does not qualify; the host then runs that step the ordinary way.
constexpr int kSmallCapDefault = 512;

template <class K, class A, class... R>
static cudaError_t launch_pdl(K kern, dim3 grid, dim3 block, cudaStream_t st, const A &a, R... rest)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a, rest...);
}

struct s2_bts {
    s2_ctx *ctx = nullptr;
    int n = 0;
    double eps2 = 0, eta = 0, eta_start = 0, dt_max = 0, dt_min = 0, eta4 = 0;
    int averaged = 0;
    Buf xrows, xrec, xhdr;                    // exchange buffers of the small-step kernel (BtsArgs), zero before its first launch
    bool x_clean = false;
    bool profile = false;                     // s2_bts_small_profile
    int profile_cta = 0;
    Buf dt, pot, ilist, stage, bcnt, misc;    // misc: {BtsCtl ctl (256 B); unsigned arrive (64 B); int hist[64]; unsigned bar[2] (64 B)}
    BtsCtl *h_ctl = nullptr;                  // pinned
    int *h_log = nullptr;                     // pinned, kBtsLog entries: active counts of the steps of one small-step launch
    bool ready = false;
    double time = 0.0;
    long long block_steps = 0, particle_steps = 0;
    double device_ms = 0.0, wall_ms = 0.0;
    long long timed_steps = 0;
    long long small_launches = 0, small_steps = 0;   // through bts_small_steps_kernel
    double small_device_ms = 0.0;
    std::vector<int> hist_ni;
    cudaEvent_t ev[2] = {nullptr, nullptr};
};

static BtsArgs bts_args(s2_bts *b)
{
    s2_ctx *ctx = b->ctx;
    BtsArgs a{};
    for (int k = 0; k < nfields(ctx->order); ++k) a.f[k] = base_field(ctx, k);
    a.dt = (double *)b->dt.p;
    a.pot = (double *)b->pot.p;
    a.rec = (const double *)ctx->result.p;
    a.ilist = (int *)b->ilist.p;
    a.stage = (int *)b->stage.p;
    a.bcnt = (int *)b->bcnt.p;
    a.ctl = (BtsCtl *)b->misc.p;
    static_assert(sizeof(BtsCtl) <= 256, "control block outgrew its slot");
    a.arrive = (unsigned *)((char *)b->misc.p + 256);     // misc: {BtsCtl (256 B slot); unsigned arrive (64 B slot); int hist[64]}
    a.hist = (int *)((char *)b->misc.p + 320);
    a.bar = (unsigned *)((char *)b->misc.p + 576);
    a.h_log = b->h_log;
    a.prof = b->profile ? (long long *)((char *)b->misc.p + 640) : nullptr;
    a.prof_cta = b->profile_cta;
    a.h_ctl = b->h_ctl;
    a.n = b->n;
    a.order = ctx->order;
    a.eta = b->eta; a.eta_start = b->eta_start; a.dt_max = b->dt_max; a.dt_min = b->dt_min;
    a.eta4 = b->eta4; a.averaged = b->averaged;
    return a;
}

static PredictArgs bts_predict_args(s2_bts *b)
{
    s2_ctx *ctx = b->ctx;
    PredictArgs p{};
    const int nf = nfields(ctx->order), np = nplanes(ctx->order), nq = n_qplanes(ctx->precision, ctx->order);
    for (int k = 0; k < nf; ++k) p.f[k] = base_field(ctx, k);
    p.id = base_id(ctx);
    for (int k = 0; k < np; ++k) p.p[k] = plane(ctx, k);
    for (int k = 0; k < nq; ++k) p.q[k] = qplane(ctx, k);
    p.t = 0.0;
    p.t_dev = &((BtsCtl *)b->misc.p)->t_next;
    p.nj = b->n;
    p.order = ctx->order;
    p.precision = ctx->precision;
    p.pdl = 1;
    return p;
}

static int bts_predict_dev_time(s2_bts *b)   // predict every j to the device-resident t_next (stand-alone launch)
{
    s2_ctx *ctx = b->ctx;
    CU(launch_predict(bts_predict_args(b), ctx->stream));
    ctx->launches++;
    ctx->predicted = true;
    ctx->nj_pred = b->n;
    ctx->calc_done = false;
    return S2_OK;
}

// next block time + next active list + prediction to that time, one launch
static int bts_select_predict(s2_bts *b, double t_now, bool host_time)
{
    s2_ctx *ctx = b->ctx;
    const int nb = (b->n + kSelPerBlock - 1) / kSelPerBlock;
    BtsArgs a = bts_args(b);
    if (ctx->order == 6)
        CU(launch_pdl(bts_select_predict_kernel<6>, dim3(nb), dim3(kSelThreads), ctx->stream, a, bts_predict_args(b), t_now, host_time ? 1 : 0));
    else
        CU(launch_pdl(bts_select_predict_kernel<4>, dim3(nb), dim3(kSelThreads), ctx->stream, a, bts_predict_args(b), t_now, host_time ? 1 : 0));
    ctx->launches++;
    ctx->predicted = true;
    ctx->nj_pred = b->n;
    ctx->calc_done = false;
    return S2_OK;
}

// ---- the ABI (include/s2b200.h, "block-time-step integrator") ------------------------------------------------------

extern "C" int s2_bts_open(s2_bts **out, s2_ctx *ctx, int n, double eps2, double eta, double eta_start, double dt_max,
                           double dt_min, int averaged, double eta4)
{
    if (!out) return S2_EINVAL;
    *out = nullptr;
    if (!ctx || n <= 0 || n > ctx->nj_cap || (ctx->order != 4 && ctx->order != 6)) return S2_EINVAL;
    int e1, e2;
    if (!(eta > 0) || !(eta_start > 0) || !(dt_min > 0) || !(dt_max >= dt_min) || dt_max > 1.0 || eps2 < 0) return S2_EINVAL;
    if (averaged && (ctx->order != 6 || !(eta4 > 0))) return S2_EINVAL;
    if (frexp(dt_max, &e1) != 0.5 || frexp(dt_min, &e2) != 0.5 || e2 < -62) return S2_EINVAL;   // powers of two, level <= 63
    CU(cudaSetDevice(ctx->device));
    s2_bts *b = new s2_bts();
    b->ctx = ctx; b->n = n; b->eps2 = eps2; b->eta = eta; b->eta_start = eta_start; b->dt_max = dt_max; b->dt_min = dt_min;
    b->averaged = averaged ? 1 : 0; b->eta4 = eta4;
    const int nb = (n + kSelPerBlock - 1) / kSelPerBlock;
    int rc = dev_reserve(ctx, b->dt, (size_t)n * sizeof(double));
    if (rc == S2_OK) rc = dev_reserve(ctx, b->pot, (size_t)n * sizeof(double));
    if (rc == S2_OK) rc = dev_reserve(ctx, b->ilist, (size_t)n * sizeof(int));
    if (rc == S2_OK) rc = dev_reserve(ctx, b->stage, (size_t)nb * kSelPerBlock * sizeof(int));
    if (rc == S2_OK) rc = dev_reserve(ctx, b->bcnt, (size_t)std::max(nb, 1024) * sizeof(int));   // (the small-step kernel: one count per CTA)
    if (rc == S2_OK) rc = dev_reserve(ctx, b->misc, 640 + 128);                  // (+ 10 profile sums at 640)
    if (rc == S2_OK) {
        cudaError_t e = cudaHostAlloc((void **)&b->h_ctl, sizeof(BtsCtl), cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaHostAlloc((void **)&b->h_log, kBtsLog * sizeof(int), cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaEventCreate(&b->ev[0]);
        if (e == cudaSuccess) e = cudaEventCreate(&b->ev[1]);
        if (e != cudaSuccess) rc = fail_cuda(ctx, e);
    }
    if (rc != S2_OK) {
        s2_bts_close(b);
        return rc;
    }
    *out = b;
    return S2_OK;
}

extern "C" int s2_bts_close(s2_bts *b)
{
    if (!b) return S2_EINVAL;
    s2_ctx *ctx = b->ctx;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (Buf *q : {&b->dt, &b->pot, &b->ilist, &b->stage, &b->bcnt, &b->misc, &b->xrows, &b->xrec, &b->xhdr}) dev_release(ctx, *q);
    if (b->h_ctl) cudaFreeHost(b->h_ctl);
    if (b->h_log) cudaFreeHost(b->h_log);
    for (auto &e : b->ev)
        if (e) cudaEventDestroy(e);
    delete b;
    return S2_OK;
}

// Initial conditions at t = 0 (host arrays), start-up force evaluation(s), first steps, first active list.
extern "C" int s2_bts_init(s2_bts *b, const double *mass, const double *pos, const double *vel)
{
    if (!b || !mass || !pos || !vel) return S2_EINVAL;
    s2_ctx *ctx = b->ctx;
    const int n = b->n;
    CU(cudaSetDevice(ctx->device));
    std::vector<int> addr(n);
    std::vector<double> zero((size_t)3 * n, 0.0), tz(n, 0.0);
    for (int i = 0; i < n; ++i) addr[i] = i;
    int rc = s2_set_j(ctx, n, addr.data(), addr.data(), tz.data(), mass, pos, vel, zero.data(), zero.data(),
                      ctx->order == 6 ? zero.data() : nullptr, ctx->order == 6 ? zero.data() : nullptr);
    if (rc == S2_OK) rc = s2_commit_j(ctx);
    if (rc != S2_OK) return rc;
    CU(cudaMemsetAsync(b->misc.p, 0, b->misc.bytes, ctx->stream));
    bts_iota_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>((int *)b->ilist.p, n);
    CU(cudaGetLastError());
    const int passes = ctx->order == 6 ? 2 : 1;
    for (int p = 0; p < passes; ++p) {
        rc = s2_predict(ctx, 0.0, n);
        if (rc == S2_OK) rc = run_force(ctx, n, (const int *)b->ilist.p, nullptr, false, b->eps2, 0, false);
        if (rc != S2_OK) return rc;
        BtsArgs a = bts_args(b);
        bts_init_kernel<<<(n + 255) / 256, 256, 0, ctx->stream>>>(a, p == passes - 1);
        CU(cudaGetLastError());
        ctx->launches += 1;
    }
    memset(b->h_ctl, 0, sizeof(BtsCtl));
    b->profile = false;
    b->x_clean = false;                      // the sequence tags start again: stale words must not match them
    b->time = 0.0;
    b->block_steps = b->particle_steps = 0;
    b->small_launches = b->small_steps = 0;
    b->small_device_ms = 0.0;
    b->hist_ni.clear();
    rc = bts_select_predict(b, 0.0, true);
    if (rc != S2_OK) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaGetLastError());
    b->ready = true;
    return S2_OK;
}

// Advances block step by block step until the next block time would exceed t_end or max_block_steps are done.
// time_device != 0: CUDA events bracket the kernels of every step and their elapsed times are accumulated
// (s2_bts_stats), at the price of two event records per step.
extern "C" int s2_bts_run(s2_bts *b, double t_end, long long max_block_steps, int time_device, long long *steps_done)
{
    if (!b || max_block_steps < 0) return S2_EINVAL;
    if (!b->ready) return S2_ESTATE;
    s2_ctx *ctx = b->ctx;
    CU(cudaSetDevice(ctx->device));
    long long done = 0;
    const auto w0 = std::chrono::steady_clock::now();
    // ordinary calls on the context since the last run (an energy evaluation, say) may have re-predicted the j-store
    // to another time: predict to the pending block time again (one launch per s2_bts_run, not per step)
    if (int rc = bts_predict_dev_time(b); rc != S2_OK) return rc;
    // the small-step kernel computes in fp64 pair arithmetic: fp64 contexts only (s2_set_tuning key 9 = 6 switches it off)
    bool small_ok = ctx->precision == S2_FP64 && ctx->tune[9] != 6;
    ForceArgs small{};
    const int kSmallCap = ctx->tune[10] > 0 ? std::min(ctx->tune[10], 1024) : kSmallCapDefault;
    if (small_ok) {
        const int nc = ctx->order == 6 ? 10 : 7, rw = ctx->order == 6 ? 20 : 14;
        small.nj = b->n;
        small.eps2 = b->eps2;
        small.order = ctx->order;
        const size_t was[3] = {b->xrows.bytes, b->xrec.bytes, b->xhdr.bytes};
        int rc = dev_reserve(ctx, b->xrows, (size_t)ctx->sm_count * kSmallCap * nc * 2 * sizeof(unsigned long long));
        if (rc == S2_OK) rc = dev_reserve(ctx, b->xrec, (size_t)b->n * rw * sizeof(unsigned long long));
        if (rc == S2_OK) rc = dev_reserve(ctx, b->xhdr, (size_t)ctx->sm_count * ctx->sm_count * sizeof(unsigned long long));
        if (rc != S2_OK) return rc;
        // sequence tags are 32 bits: long before they wrap, start again from clean buffers
        const bool wrap = b->h_ctl->tag > 0x70000000LL;
        if (wrap) {
            CU(cudaMemsetAsync(&((BtsCtl *)b->misc.p)->tag, 0, sizeof(long long), ctx->stream));
            b->h_ctl->tag = 0;
        }
        if (wrap || !b->x_clean || was[0] != b->xrows.bytes || was[1] != b->xrec.bytes || was[2] != b->xhdr.bytes) {
            CU(cudaMemsetAsync(b->xrows.p, 0, b->xrows.bytes, ctx->stream));
            CU(cudaMemsetAsync(b->xrec.p, 0, b->xrec.bytes, ctx->stream));
            CU(cudaMemsetAsync(b->xhdr.p, 0, b->xhdr.bytes, ctx->stream));
            b->x_clean = true;
        }
    }
    while (done < max_block_steps && b->h_ctl->t_next <= t_end) {
        const double t_new = b->h_ctl->t_next;
        const int n_act = b->h_ctl->n_next;
        if (n_act <= 0 || n_act > b->n) return S2_ESTATE;
        // the j-particles were already predicted to t_new (by the previous select, or by the small-step kernel)
        if (small_ok && n_act <= kSmallCap) {
            const int K = (int)std::min<long long>(kBtsLog, max_block_steps - done);
            const long long steps0 = b->h_ctl->steps;
            BtsArgs a = bts_args(b);
            a.spec_cap = kSmallCap;
            a.max_steps = K;
            a.t_end = t_end;
            a.xrows = (unsigned long long *)b->xrows.p;
            a.xrec = (unsigned long long *)b->xrec.p;
            a.xhdr = (unsigned long long *)b->xhdr.p;
            if (time_device) CU(cudaEventRecord(b->ev[0], ctx->stream));
            const cudaError_t e = launch_bts_small_steps(small, a, bts_predict_args(b), ctx->device, ctx->sm_count, ctx->stream);
            if (e == cudaErrorNotSupported || e == cudaErrorCooperativeLaunchTooLarge || e == cudaErrorLaunchOutOfResources) {
                // this device (or the share of it this process has right now) cannot hold one CTA per SM at once:
                // every step the ordinary way -- nothing was launched, nothing is lost
                cudaGetLastError();
                small_ok = false;
                continue;
            }
            CU(e);
            ctx->launches++;
            if (time_device) CU(cudaEventRecord(b->ev[1], ctx->stream));
            CU(cudaStreamSynchronize(ctx->stream));      // one synchronisation per run of small steps
            const int ran = (int)(b->h_ctl->steps - steps0);
            if (b->h_ctl->error || ran < 1 || ran > K) return S2_ESTATE;   // (the first step of a launch always qualifies)
            if (time_device) {
                float ms = 0.f;
                CU(cudaEventElapsedTime(&ms, b->ev[0], b->ev[1]));
                b->device_ms += ms;
                b->small_device_ms += ms;
                b->timed_steps += ran;
            }
            for (int k = 0; k < ran; ++k) {
                b->particle_steps += b->h_log[k];
                b->hist_ni.push_back(b->h_log[k]);
            }
            b->time = b->h_ctl->t_done;
            b->block_steps += ran;
            b->small_steps += ran;
            b->small_launches++;
            done += ran;
            ctx->predicted = true;
            ctx->nj_pred = b->n;
            ctx->calc_done = false;
            continue;
        }
        if (time_device) CU(cudaEventRecord(b->ev[0], ctx->stream));
        BtsArgs a = bts_args(b);
        a.n_act = n_act;
        ctx->bts_hook = &a;                  // if the force call combines with reduce_kernel, that kernel corrects as well
        ctx->bts_hook_done = false;
        int rc = run_force(ctx, n_act, (const int *)b->ilist.p, nullptr, false, b->eps2, 0, false);
        ctx->bts_hook = nullptr;
        if (rc != S2_OK) return rc;
        if (!ctx->bts_hook_done) {
            CU(launch_pdl(bts_correct_kernel, dim3((n_act + 127) / 128), dim3(128), ctx->stream, a));
            ctx->launches++;
        }
        rc = bts_select_predict(b, 0.0, false);
        if (rc != S2_OK) return rc;
        if (time_device) CU(cudaEventRecord(b->ev[1], ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));          // the one synchronisation of a block step: 12 bytes in pinned memory
        if (time_device) {
            float ms = 0.f;
            CU(cudaEventElapsedTime(&ms, b->ev[0], b->ev[1]));
            b->device_ms += ms;
            b->timed_steps++;
        }
        b->time = t_new;
        b->block_steps++;
        b->particle_steps += n_act;
        b->hist_ni.push_back(n_act);
        ++done;
    }
    CU(cudaGetLastError());
    b->wall_ms += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - w0).count();
    if (steps_done) *steps_done = done;
    return S2_OK;
}

extern "C" int s2_bts_get_state(s2_bts *b, double *time, double *t, double *dt, double *pos, double *vel, double *acc,
                                double *jerk, double *pot)
{
    if (!b) return S2_EINVAL;
    if (!b->ready) return S2_ESTATE;
    s2_ctx *ctx = b->ctx;
    const int n = b->n;
    CU(cudaSetDevice(ctx->device));
    std::vector<double> h((size_t)15 * n);
    CU(cudaMemcpyAsync(h.data(), base_field(ctx, 0), (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    for (int f = 2; f < 14; ++f)
        CU(cudaMemcpyAsync(h.data() + (size_t)(f - 1) * n, base_field(ctx, f), (size_t)n * sizeof(double), cudaMemcpyDeviceToHost,
                           ctx->stream));
    CU(cudaMemcpyAsync(h.data() + (size_t)13 * n, b->dt.p, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaMemcpyAsync(h.data() + (size_t)14 * n, b->pot.p, (size_t)n * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (time) *time = b->time;
    double *vecs[4] = {pos, vel, acc, jerk};
    for (int i = 0; i < n; ++i) {
        if (t) t[i] = h[i];
        if (dt) dt[i] = h[(size_t)13 * n + i];
        if (pot) pot[i] = h[(size_t)14 * n + i];
        for (int v = 0; v < 4; ++v)
            if (vecs[v])
                for (int c = 0; c < 3; ++c) vecs[v][3 * (size_t)i + c] = h[(size_t)(1 + 3 * v + c) * n + i];
    }
    return S2_OK;
}

extern "C" int s2_bts_stats(const s2_bts *b, double *time, double *t_next, int *n_next, long long *block_steps,
                            long long *particle_steps, double *wall_ms, double *device_ms, long long *timed_steps)
{
    if (!b) return S2_EINVAL;
    if (time) *time = b->time;
    if (t_next) *t_next = b->ready ? b->h_ctl->t_next : 0.0;
    if (n_next) *n_next = b->ready ? b->h_ctl->n_next : 0;
    if (block_steps) *block_steps = b->block_steps;
    if (particle_steps) *particle_steps = b->particle_steps;
    if (wall_ms) *wall_ms = b->wall_ms;
    if (device_ms) *device_ms = b->device_ms;
    if (timed_steps) *timed_steps = b->timed_steps;
    return S2_OK;
}

extern "C" int s2_bts_small_profile(s2_bts *b, int on, long long out[10])
{
    if (!b) return S2_EINVAL;
    s2_ctx *ctx = b->ctx;
    CU(cudaSetDevice(ctx->device));
    long long *dev = (long long *)((char *)b->misc.p + 640);
    if (out) {
        CU(cudaMemcpyAsync(out, dev, 10 * sizeof(long long), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    if (on < 0 || on > ctx->sm_count) return S2_EINVAL;
    if (on) CU(cudaMemsetAsync(dev, 0, 10 * sizeof(long long), ctx->stream));
    b->profile = on != 0;
    b->profile_cta = on ? on - 1 : 0;
    return S2_OK;
}

extern "C" int s2_bts_small_stats(const s2_bts *b, long long *launches, long long *steps, double *device_ms)
{
    if (!b) return S2_EINVAL;
    if (launches) *launches = b->small_launches;
    if (steps) *steps = b->small_steps;
    if (device_ms) *device_ms = b->small_device_ms;
    return S2_OK;
}

extern "C" int s2_bts_get_history(const s2_bts *b, long long first, int count, int *n_active)
{
    if (!b || first < 0 || count < 0 || (count > 0 && !n_active)) return S2_EINVAL;
    if (first + count > (long long)b->hist_ni.size()) return S2_ERANGE;
    for (int k = 0; k < count; ++k) n_active[k] = b->hist_ni[(size_t)first + k];
    return S2_OK;
}
