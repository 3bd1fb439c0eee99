// s2_api.cu -- the C ABI of include/s2b200.h: context, device buffers, staging, the launch
// balancer that picks (lanes per i, warp columns, j-slices), and result read-back.
// Every arithmetic step of the hot path runs in the kernels; this file only moves bytes and
// chooses launch shapes.
#include <math.h>
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include <algorithm>
#include <chrono>
#include <map>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "s2_internal.h"
#include "../../include/s2b200_test.h"

namespace s2 {
cudaError_t launch_csr_scan(const double *rec, int ni, int cap, int *len, long long *block_sum, long long *total,
                            long long *offsets, cudaStream_t st);
cudaError_t launch_csr_fill(const int *list, const int *len, const long long *offsets, int ni, int cap, int *out, cudaStream_t st);
int csr_blocks(int ni);
cudaError_t launch_fp32_fix(const ForceArgs &a, int sm_count, cudaStream_t st);
cudaError_t launch_fp32_flag(const double *rec, const F32Flag &f, int ni, cudaStream_t st);
cudaError_t launch_compare_records(const double *a, const double *b, int ni, int order, double tol, int *bad, cudaStream_t st);
cudaError_t launch_unpack_records(const double *rec, int ni, int order, double *acc, double *jerk, double *snap, double *pot,
                                  int *nn_id, double *nn_r2, int *ngb_count, cudaStream_t st);
cudaError_t dispatch_force_fp64(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                                cudaStream_t st, bool query, int *ctas_per_sm);
cudaError_t dispatch_force_fp32(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                                cudaStream_t st, bool query, int *ctas_per_sm);
cudaError_t dispatch_force_ds(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                              cudaStream_t st, bool query, int *ctas_per_sm);
cudaError_t dispatch_force_fp64_bank0(int order, unsigned flags, const ForceArgs &a, cudaStream_t st, int *geom);
cudaError_t dispatch_force_fp64_bank1(int order, unsigned flags, const ForceArgs &a, cudaStream_t st, int *geom);
cudaError_t force_bank_address0(void **p);
cudaError_t force_bank_address1(void **p);
int force_nplanes(int precision, int order, unsigned flags);
cudaError_t run_ds_ops(int n, const double *d_a, const double *d_b, double *d_out, cudaStream_t st);
}  // namespace s2

using namespace s2;

#include "s2_ctx.h"

// ---- helpers ----------------------------------------------------------------------------

int fail_cuda(s2_ctx *c, cudaError_t e)
{
    if (c) c->cuda_err = cudaGetErrorString(e);
    return S2_ECUDA;
}

int dev_reserve(s2_ctx *ctx, Buf &b, size_t bytes)
{
    if (bytes <= b.bytes) return S2_OK;
    // grow-only; contents are not preserved (callers refill)
    if (b.p) {
        // the old block may still be in use by enqueued kernels: drain the stream first
        CU(cudaStreamSynchronize(ctx->stream));
        if (ctx->has_alloc)
            ctx->alloc.free(b.p, ctx->alloc.user);
        else
            cudaFree(b.p);
        b.p = nullptr;
        b.bytes = 0;
    }
    size_t want = bytes + bytes / 4;   // 25 % head-room against repeated growth
    want = (want + 255) & ~(size_t)255;
    void *p = nullptr;
    if (ctx->has_alloc) {
        p = ctx->alloc.alloc(want, ctx->alloc.user);
        if (!p) return S2_ENOMEM;
    } else {
        cudaError_t e = cudaMalloc(&p, want);
        if (e == cudaErrorMemoryAllocation) {
            cudaGetLastError();
            return S2_ENOMEM;
        }
        if (e != cudaSuccess) return fail_cuda(ctx, e);
    }
    b.p = p;
    b.bytes = want;
    return S2_OK;
}

void dev_release(s2_ctx *ctx, Buf &b)
{
    if (!b.p) return;
    if (ctx->has_alloc)
        ctx->alloc.free(b.p, ctx->alloc.user);
    else
        cudaFree(b.p);
    b.p = nullptr;
    b.bytes = 0;
}

int pinned_reserve(s2_ctx *ctx, void **p, size_t *have, size_t used, size_t bytes)
{
    if (bytes <= *have) return S2_OK;
    size_t want = std::max(bytes + bytes / 2, (size_t)1 << 16);
    void *q = nullptr;
    cudaError_t e = cudaHostAlloc(&q, want, cudaHostAllocDefault);
    if (e == cudaErrorMemoryAllocation) {
        cudaGetLastError();
        return S2_ENOMEM;
    }
    if (e != cudaSuccess) return fail_cuda(ctx, e);
    if (*p) {
        if (used) memcpy(q, *p, used);
        cudaFreeHost(*p);
    }
    *p = q;
    *have = want;
    return S2_OK;
}

// Host-side copies of the staging path (a1, a9) run on a few threads once they are large: one core moves ~8 GB/s,
// and at N = 2^18 the 32 MB in + 25 MB out were 5 % of an end-to-end step.
template <class F>
static void par_ranges(size_t n, size_t min_per_thread, F fn)
{
    size_t nt = std::min<size_t>({(size_t)8, std::max<size_t>(1, std::thread::hardware_concurrency()), n / std::max<size_t>(1, min_per_thread)});
    if (nt <= 1) { fn((size_t)0, n); return; }
    std::vector<std::thread> th;
    const size_t per = (n + nt - 1) / nt;
    for (size_t k = 1; k < nt; ++k) {
        const size_t lo = std::min(n, k * per), hi = std::min(n, lo + per);
        if (lo < hi) th.emplace_back([=] { fn(lo, hi); });
    }
    fn((size_t)0, std::min(n, per));
    for (auto &t : th) t.join();
}
static void par_memcpy(void *dst, const void *src, size_t bytes)
{
    par_ranges(bytes, (size_t)1 << 20, [=](size_t lo, size_t hi) { memcpy((char *)dst + lo, (const char *)src + lo, hi - lo); });
}

static inline size_t align16(size_t x) { return (x + 15) & ~(size_t)15; }

// ---- state shared by the contexts of one device: the two constant banks of the uniform-operand sweep ------------
// (see run_force_bank below)
struct BankOwner {
    cudaEvent_t ev = nullptr;
    cudaStream_t stream = nullptr;
    bool used = false;
    unsigned *flags = nullptr;   // device words {ready[2], -, -, arrived[2]} of the bank hand-over (run_force_bank)
    unsigned ticket = 0;         // tickets handed out so far (chunk sequence numbers, cyclic)
    int refs = 0;                // open contexts on this device; the last s2_close frees flags and event
    // How the banks are refilled on this device (DESIGN.md 5.2 "what the uniform-operand sweep assumes"):
    //   0 not yet decided; 1 by the sweep's own last CTA through the bank's global address, launches overlapped
    //   (relies on behaviour CUDA does not document, so it is only used after bank_selftest has seen it produce the
    //   shared-memory sweep's results on this device and driver); 2 by cudaMemcpyAsync between ordinary launches
    //   (documented semantics; ~4 % slower)
    int mode = 0;
};
static std::mutex g_bank_mu;
static std::map<int, BankOwner> g_bank;
enum { kBankSelfRefill = 1, kBankHostRefill = 2 };

// ---- life cycle ---------------------------------------------------------------------------

extern "C" int s2_open(s2_ctx **out, int device, int order, int precision, int nj_capacity, int ngb_cap,
                       const s2_allocator *a, void *cuda_stream)
{
    if (!out) return S2_EINVAL;
    *out = nullptr;
    if ((order != 2 && order != 4 && order != 6) || precision < S2_FP64 || precision > S2_FP32 || nj_capacity <= 0 || ngb_cap < 0)
        return S2_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || device < 0 || device >= ndev) {
        cudaGetLastError();
        return S2_ECUDA;   // no CPU fallback
    }
    if (cudaSetDevice(device) != cudaSuccess) return S2_ECUDA;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, device) != cudaSuccess) return S2_ECUDA;
    if (prop.major < 10) return S2_ECUDA;   // kernels are built for sm_100a only

    s2_ctx *ctx = new s2_ctx();
    ctx->device = device;
    ctx->order = order;
    ctx->precision = precision;
    ctx->nj_cap = nj_capacity;
    ctx->ngb_cap = ngb_cap;
    ctx->stream = (cudaStream_t)cuda_stream;
    ctx->sm_count = prop.multiProcessorCount;
    if (a && a->alloc && a->free) {
        ctx->alloc = *a;
        ctx->has_alloc = true;
    }
    int rc = S2_OK;
    const size_t nf = nfields(order), np = nplanes(order), nq = n_qplanes(precision, order);
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->base, nf * nj_capacity * sizeof(double) + (size_t)nj_capacity * sizeof(int));
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->planes, np * nj_capacity * sizeof(double2));
    if (rc == S2_OK && nq) rc = dev_reserve(ctx, ctx->qplanes, nq * nj_capacity * sizeof(float4));
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->flags, 256);
    if (rc == S2_OK) {
        cudaError_t e = cudaMemsetAsync(ctx->flags.p, 0, 256, ctx->stream);
        if (e == cudaSuccess) e = cudaHostAlloc((void **)&ctx->h_flags, 64, cudaHostAllocDefault);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_stage, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_io, cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_il[0], cudaEventDisableTiming);
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&ctx->ev_il[1], cudaEventDisableTiming);
        for (int k = 0; k < 6 && e == cudaSuccess; ++k) e = cudaEventCreate(&ctx->ev_t[k]);
        for (int k = 0; k < 4 && e == cudaSuccess; ++k) e = cudaEventCreate(&ctx->ev_csr[k]);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e != cudaSuccess) rc = fail_cuda(ctx, e);
    }
    {
        std::lock_guard<std::mutex> lock(g_bank_mu);
        g_bank[device].refs++;
    }
    if (rc != S2_OK) {
        s2_close(ctx);
        return rc;
    }
    *out = ctx;
    return S2_OK;
}

extern "C" int s2_close(s2_ctx *ctx)
{
    if (!ctx) return S2_EINVAL;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (Buf *b : {&ctx->base, &ctx->planes, &ctx->qplanes, &ctx->stage_dev, &ctx->iplanes, &ctx->iqplanes,
                   &ctx->i_addr, &ctx->i_h2, &ctx->part, &ctx->result, &ctx->seg, &ctx->list, &ctx->flags, &ctx->counters,
                   &ctx->csr_len, &ctx->csr_bsum, &ctx->csr_off, &ctx->csr_list, &ctx->wq, &ctx->fix, &ctx->fixpart, &ctx->fixarr})
        dev_release(ctx, *b);
    for (auto &e : ctx->ev_csr)
        if (e) cudaEventDestroy(e);
    if (ctx->h_stage) cudaFreeHost(ctx->h_stage);
    if (ctx->h_io) cudaFreeHost(ctx->h_io);
    if (ctx->h_flags) cudaFreeHost(ctx->h_flags);
    if (ctx->ev_stage) cudaEventDestroy(ctx->ev_stage);
    if (ctx->ev_io) cudaEventDestroy(ctx->ev_io);
    for (int k = 0; k < 2; ++k) {
        if (ctx->ev_il[k]) cudaEventDestroy(ctx->ev_il[k]);
        if (ctx->h_il[k]) cudaFreeHost(ctx->h_il[k]);
    }
    if (ctx->h_res) cudaFreeHost(ctx->h_res);
    for (auto &e : ctx->ev_t)
        if (e) cudaEventDestroy(e);
    {   // the last context of a device releases what the device's contexts share (bank hand-over words, event)
        std::lock_guard<std::mutex> lock(g_bank_mu);
        auto it = g_bank.find(ctx->device);
        if (it != g_bank.end() && --it->second.refs <= 0) {
            if (it->second.used) cudaEventSynchronize(it->second.ev);
            if (it->second.flags) cudaFree(it->second.flags);
            if (it->second.ev) cudaEventDestroy(it->second.ev);
            const int mode = it->second.mode;
            g_bank.erase(it);
            g_bank[ctx->device].mode = mode;   // the verdict of the self-test is a property of device + driver: kept
        }
    }
    cudaGetLastError();
    delete ctx;
    return S2_OK;
}

extern "C" int s2_set_stream(s2_ctx *ctx, void *cuda_stream)
{
    if (!ctx) return S2_EINVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->stream = (cudaStream_t)cuda_stream;
    return S2_OK;
}

extern "C" int s2_synchronize(s2_ctx *ctx)
{
    if (!ctx) return S2_EINVAL;
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaGetLastError());
    return S2_OK;
}

// ---- a1: set / commit -------------------------------------------------------------------

extern "C" int s2_set_j(s2_ctx *ctx, int n, const int *address, const int *id, const double *t, const double *mass,
                        const double *pos, const double *vel, const double *acc, const double *jerk,
                        const double *snap, const double *crackle)
{
    if (!ctx || n < 0) return S2_EINVAL;
    if (n == 0) return S2_OK;
    if (!address || !id || !t || !mass || !pos || !vel) return S2_EINVAL;
    if (ctx->order != 2 && (!acc || !jerk)) return S2_EINVAL;   // 2nd order: missing derivatives are stored as zero
    if (ctx->order == 6 && (!snap || !crackle)) return S2_EINVAL;
    if (n > ctx->nj_cap) return S2_ERANGE;
    for (int k = 0; k < n; ++k)
        if (address[k] < 0 || address[k] >= ctx->nj_cap) return S2_ERANGE;
    for (int k = 0; k < n; ++k)
        if (id[k] < 0) return S2_EINVAL;

    // the previous commit may still be reading the staging buffer
    if (ctx->batches.empty()) CU(cudaEventSynchronize(ctx->ev_stage));

    const int nf = nfields(ctx->order);
    const size_t off = align16(ctx->h_stage_used);
    const size_t ints = align16((size_t)2 * n * sizeof(int));
    const size_t bytes = ints + (size_t)nf * n * sizeof(double);
    int rc = pinned_reserve(ctx, &ctx->h_stage, &ctx->h_stage_bytes, ctx->h_stage_used, off + bytes);
    if (rc != S2_OK) return rc;
    char *blk = (char *)ctx->h_stage + off;
    par_memcpy(blk, address, (size_t)n * sizeof(int));
    par_memcpy(blk + (size_t)n * sizeof(int), id, (size_t)n * sizeof(int));
    double *f = (double *)(blk + ints);
    par_memcpy(f, t, (size_t)n * sizeof(double));
    par_memcpy(f + n, mass, (size_t)n * sizeof(double));
    // vector fields are staged verbatim, (n,3) row-major; the scatter kernel does the transposition into the SoA
    const double *vecs[6] = {pos, vel, acc, jerk, snap, crackle};
    const int nvec = ctx->order == 6 ? 6 : 4;
    for (int v = 0; v < nvec; ++v) {
        double *dst = f + (size_t)(2 + 3 * v) * n;
        if (vecs[v])
            par_memcpy(dst, vecs[v], (size_t)3 * n * sizeof(double));
        else   // 2nd-order context without acc / jerk
            memset(dst, 0, (size_t)3 * n * sizeof(double));
    }
    ctx->batches.push_back({off, n});
    ctx->h_stage_used = off + bytes;
    return S2_OK;
}

extern "C" int s2_commit_j(s2_ctx *ctx)
{
    if (!ctx) return S2_EINVAL;
    if (ctx->batches.empty()) return S2_OK;
    CU(cudaSetDevice(ctx->device));
    int rc = dev_reserve(ctx, ctx->stage_dev, ctx->h_stage_used);
    if (rc != S2_OK) return rc;
    CU(cudaMemcpyAsync(ctx->stage_dev.p, ctx->h_stage, ctx->h_stage_used, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaEventRecord(ctx->ev_stage, ctx->stream));
    const int nf = nfields(ctx->order);
    for (const Batch &b : ctx->batches) {
        ScatterArgs a{};
        const char *blk = (const char *)ctx->stage_dev.p + b.offset;
        a.address = (const int *)blk;
        a.id = a.address + b.n;
        const double *f = (const double *)(blk + align16((size_t)2 * b.n * sizeof(int)));
        a.src[0] = f;
        a.src[1] = f + b.n;
        for (int k = 2; k < nf; ++k)   // component c of vector field v: row-major (n,3) block, stride 3
            a.src[k] = f + (size_t)(2 + 3 * ((k - 2) / 3)) * b.n + (k - 2) % 3;
        for (int k = 0; k < nf; ++k) a.dst[k] = base_field(ctx, k);
        a.dst_id = base_id(ctx);
        a.n = b.n;
        a.nfields = nf;
        a.nj_cap = ctx->nj_cap;
        a.erange_flag = (int *)ctx->flags.p + 1;
        CU(launch_scatter(a, ctx->stream));
        ctx->launches++;
    }
    ctx->batches.clear();
    ctx->h_stage_used = 0;
    ctx->have_j = true;
    ctx->predicted = false;
    return S2_OK;
}

extern "C" int s2_commit_j_device(s2_ctx *ctx, int n, const int *d_address, const int *d_id, const double *d_t,
                                  const double *d_mass, const double *d_pos, const double *d_vel,
                                  const double *d_acc, const double *d_jerk, const double *d_snap,
                                  const double *d_crackle)
{
    if (!ctx || n < 0) return S2_EINVAL;
    if (n == 0) return S2_OK;
    if (!d_address || !d_id || !d_t || !d_mass || !d_pos || !d_vel) return S2_EINVAL;
    if (ctx->order != 2 && (!d_acc || !d_jerk)) return S2_EINVAL;   // 2nd order: missing derivatives are stored as zero (as s2_set_j)
    if (ctx->order == 6 && (!d_snap || !d_crackle)) return S2_EINVAL;
    if (n > ctx->nj_cap) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    ScatterArgs a{};
    a.address = d_address;
    a.id = d_id;
    a.src[0] = d_t;
    a.src[1] = d_mass;
    const double *vecs[6] = {d_pos, d_vel, d_acc, d_jerk, d_snap, d_crackle};
    const int nvec = ctx->order == 6 ? 6 : 4;
    for (int v = 0; v < nvec; ++v)
        for (int c = 0; c < 3; ++c) a.src[2 + 3 * v + c] = vecs[v] ? vecs[v] + c : nullptr;
    const int nf = nfields(ctx->order);
    for (int k = 0; k < nf; ++k) a.dst[k] = base_field(ctx, k);
    a.dst_id = base_id(ctx);
    a.n = n;
    a.nfields = nf;
    a.nj_cap = ctx->nj_cap;
    a.erange_flag = (int *)ctx->flags.p + 1;
    CU(launch_scatter(a, ctx->stream));
    ctx->launches++;
    ctx->have_j = true;
    ctx->flags_dirty = true;   // the scatter kernel raises flag 1 on an out-of-range address
    ctx->predicted = false;
    return S2_OK;
}

// ---- a2: predict ------------------------------------------------------------------------

extern "C" int s2_predict(s2_ctx *ctx, double t, int nj)
{
    if (!ctx) return S2_EINVAL;
    if (nj <= 0 || nj > ctx->nj_cap) return S2_ERANGE;
    if (!ctx->have_j || !ctx->batches.empty()) return S2_ESTATE;   // staged but uncommitted particles
    CU(cudaSetDevice(ctx->device));
    PredictArgs a{};
    const int nf = nfields(ctx->order), np = nplanes(ctx->order), nq = n_qplanes(ctx->precision, ctx->order);
    for (int k = 0; k < nf; ++k) a.f[k] = base_field(ctx, k);
    a.id = base_id(ctx);
    for (int k = 0; k < np; ++k) a.p[k] = plane(ctx, k);
    for (int k = 0; k < nq; ++k) a.q[k] = qplane(ctx, k);
    a.t = t;
    a.nj = nj;
    a.order = ctx->order;
    a.precision = ctx->precision;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[0], ctx->stream));
    CU(launch_predict(a, ctx->stream));
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[1], ctx->stream));
    ctx->ran_predict = true;
    ctx->launches++;
    ctx->predicted = true;
    ctx->nj_pred = nj;
    ctx->t_pred = t;
    ctx->calc_done = false;
    return S2_OK;
}

extern "C" int s2_set_j_range(s2_ctx *ctx, int first, int count)
{
    if (!ctx || first < 0 || count < 0) return S2_EINVAL;
    if ((long long)first + count > ctx->nj_cap) return S2_ERANGE;
    ctx->j_first = count > 0 ? first : 0;
    ctx->j_count = count;
    return S2_OK;
}

// ---- launch balancer ----------------------------------------------------------------------

static cudaError_t dispatch(int precision, int order, unsigned flags, int L, dim3 grid, size_t smem,
                            const ForceArgs &a, cudaStream_t st, bool query, int *occ)
{
    switch (precision) {
    case S2_FP64: return dispatch_force_fp64(order, flags, L, grid, smem, a, st, query, occ);
    case S2_FP32: return dispatch_force_fp32(order, flags, L, grid, smem, a, st, query, occ);
    case S2_DS: return dispatch_force_ds(order, flags, L, grid, smem, a, st, query, occ);
    }
    return cudaErrorInvalidValue;
}

// Launch-shape model.  All times in SM cycles:
//   an SM receives n = ceil(CTAs / SMs) CTAs; with `occ` resident at a time it pays the fixed per-CTA latency
//   (first bulk copy, i-gather, epilogue) once per residency round, and one CTA-iteration (256 lanes x 1 pair)
//   costs t_iter cycles of the arithmetic pipe, whoever shares the SM;
//   the combine costs one launch gap when it is a separate kernel, or a short serial tail in the last CTA of
//   each i-group when it is fused.
struct ShapeCost {
    double t_iter, c_cta, c_row, c_launch, tiled_gain;
};
static ShapeCost cost_params(int precision, int order)
{
    ShapeCost c;
    c.t_iter = precision == S2_FP64 ? 146.0 : (precision == S2_FP32 ? 100.0 : 1400.0);
    if (order == 6) c.t_iter *= 1.7;
    if (order == 2) c.t_iter *= 0.6;
    c.tiled_gain = 0.93;  // measured: pairs of the register-tiled sweep cost this fraction of the plain ones
    c.c_cta = 4000.0;     // ~2 us: launch ramp, first tile, i-gather, shuffles, record write
    c.c_row = 1000.0;     // ~0.5 us per round of 32 partial rows (L2 latency bound)
    c.c_launch = 3000.0;  // ~1.5 us: second launch (programmatic dependent launch hides part of it)
    return c;
}

static int query_occ(s2_ctx *ctx, unsigned flags, int L, int npl, int *occ_out)
{
    int occ = ctx->tune[3];
    if (occ <= 0) {
        const long long key = ((long long)flags << 32) | (unsigned)(L & 0xffff);
        auto it = ctx->occ_cache.find(key);
        if (it == ctx->occ_cache.end()) {
            ForceArgs dummy{};
            cudaError_t e = dispatch(ctx->precision, ctx->order, flags, L, dim3(1), force_smem_bytes(npl, 256, 2),
                                     dummy, ctx->stream, true, &occ);
            if (e != cudaSuccess) return fail_cuda(ctx, e);
            if (occ < 1) occ = 1;
            ctx->occ_cache[key] = occ;
        } else {
            occ = it->second;
        }
    }
    *occ_out = occ;
    return S2_OK;
}

// Chooses lanes per i (L), warp columns (Wj), number of j-slices (S), the tile length and the number of tile
// buffers.  Automatic choices are cached per (n_i, n_j, flags); s2_set_tuning overrides any of them.
static int choose_shape(s2_ctx *ctx, int ni, int nj, unsigned flags, ForceShape *out)
{
    const bool tuned = ctx->tune[0] || ctx->tune[1] || ctx->tune[2] || ctx->tune[3] || ctx->tune[4] || ctx->tune[5] || ctx->tune[6] || ctx->tune[7];
    const long long ckey = ((long long)ni << 34) ^ ((long long)nj << 3) ^ (long long)flags;
    if (!tuned) {
        auto it = ctx->shape_cache.find(ckey);
        if (it != ctx->shape_cache.end()) {
            *out = it->second.first;
            ctx->last_info[7] = it->second.second;
            return S2_OK;
        }
    }
    const int npl = force_nplanes(ctx->precision, ctx->order, flags);
    const ShapeCost C_ = cost_params(ctx->precision, ctx->order);
    const bool want_ngb = flags & S2_WANT_NGB;
    const int tile_max = std::min(2048, (int)((232448 - kSmemHeader) / (2 * npl * 16)) / 32 * 32);

    double best = 1e300;
    int bL = 1, bTL = 0, bWj = 1, bS = 1, bocc = 1, bfused = 0, bC = 1;
    const int ipt_max = force_ipt(ctx->precision);
    for (int Lc = -5; Lc <= 6; ++Lc) {
        // Lc <= 0: register-tiled sweep (ipt_max i per thread) with TL = 1, 2, .., 32 lanes per i-slot (TL > 1: plain sums
        // only); Lc = 1..6: one i per thread, L = 1, 2, 4, .., 32 lanes per i
        const int L = Lc <= 0 ? 0 : 1 << (Lc - 1);
        const int TL = Lc <= 0 ? 1 << (-Lc) : 0;
        const int ipt = L == 0 ? ipt_max : 1;
        if (L == 0 && (ipt_max < 2 || ctx->tune[7] == 1 || (TL > 1 && flags != 0))) continue;
        // lanes per i-slot pay in fp32, where the tiled sweep's packed FFMA2 pairs halve the issue slots (measured at
        // N = 65536: n_i = 256: 32.1 -> 27.8 us, 1024: 101.9 -> 88.9 us); in fp64 they measure within 1 % of the one-i-per-
        // thread shapes (the LDS.128 they save is a small part of an FP64-pipe-bound loop), so there only when forced
        if (L == 0 && TL > 1 && ctx->precision != S2_FP32 && ctx->tune[7] < 2) continue;
        if (ctx->tune[7] >= 2 && L != 0) continue;
        if (ctx->tune[1] > 0 && (L == 0 ? TL : L) != ctx->tune[1]) continue;
        int occ;
        int rc = query_occ(ctx, flags, L == 0 ? (TL > 1 ? -TL : 0) : L, npl, &occ);
        if (rc != S2_OK) return rc;
        for (int Wj = 1; Wj <= kWarps; Wj <<= 1) {
            // warp columns: warps of a CTA share i-particles and split every tile (the paper's 2D blocks, L104);
            // used only while the i-list cannot fill one CTA with L lanes per i (measured: otherwise the extra
            // i-groups re-stream the j range from L2 and lose, profiles/r01_small_ni.md)
            if (ctx->tune[2] > 0 ? Wj != ctx->tune[2] : (Wj > 1 && (L <= 1 || (long long)ni * L * Wj > kThreads))) continue;
            if (Wj > 1 && L <= 1) continue;
            const int icta = L == 0 ? kThreads * ipt / TL : (kWarps / Wj) * (32 / L);
            const int Gi = (ni + icta - 1) / icta;
            const int lanes_j = (L == 0 ? TL : L) * Wj;          // lanes (over all warp columns) sharing one i
            const int min_slice = std::max(32, 2 * lanes_j);
            const int smax = std::min(65535, std::max(1, nj / min_slice));
            // candidate slice counts: 1, and those that make the grid k x SMs (k = 1..16)
            int cand[40], nc = 0;
            if (ctx->tune[0] > 0) {
                cand[nc++] = ctx->tune[0];
            } else {
                cand[nc++] = 1;
                for (int k = 1; k <= 16; ++k) {
                    const int s1 = (int)(((long long)k * ctx->sm_count) / Gi);          // floor: grid <= k SMs
                    if (s1 >= 1 && s1 <= smax) cand[nc++] = s1;
                }
            }
            for (int q = 0; q < nc; ++q) {
                int S = cand[q];
                // neighbour segments must stay ascending per record: a warp column may then only take a part of ONE tile
                if (want_ngb && Wj > 1 && (nj + S - 1) / S > tile_max) S = (nj + tile_max - 1) / tile_max;
                const bool fusable = !want_ngb && (ctx->tune[5] == 0 || ctx->tune[5] == 3) && S * Wj > 1 && L != 0;
                // clusters of C CTAs along the slice axis pre-combine their records through distributed shared
                // memory (j-split shapes only: their record block, <= 128 x 96 B, always fits the tile buffers)
                int C = 1;
                if (fusable && lanes_j > 1 && S > 1) {
                    C = ctx->tune[6] > 0 ? ctx->tune[6] : 1;   // opt-in: measured slower than no cluster
                    if (C != 1 && C != 2 && C != 4 && C != 8) return S2_EINVAL;
                    if (S < C) C = 1;
                    S = S / C * C;
                }
                int sl = (nj + S - 1) / S;
                if (C == 1) S = (nj + sl - 1) / sl;             // no empty slices (a cluster grid may keep some)
                const long long ctas = (long long)Gi * S;
                const double n_sm = (double)((ctas + ctx->sm_count - 1) / ctx->sm_count);
                const double iters = (double)((sl + lanes_j - 1) / lanes_j);
                // measured (profiles/r01_small_ni.md): a lone CTA per SM is latency-bound (~1.1x); lanes that share an i
                // read different j, and LDS.128 is conflict-free only up to 8 distinct addresses (4-way at L = 32)
                double t_iter = C_.t_iter * (n_sm >= 2 ? 1.0 : 1.1) * (1.0 + 0.01 * L) * (L == 32 ? 1.3 : 1.0);
                // register-tiled: ipt pairs per lane and j, fewer shared-memory reads each
                if (L == 0) t_iter = C_.t_iter * ipt * C_.tiled_gain * (n_sm >= 2 ? 1.0 : 1.09) * (1.0 + 0.03 * (-Lc)) * (TL == 32 ? 1.3 : 1.0);
                // every i-group streams the whole j range from L2 (~2500 B per SM-cycle over the chip)
                const double stream = (double)Gi * nj * npl * 16.0 / 2500.0;
                double cost = std::ceil(n_sm / occ) * C_.c_cta + std::max(n_sm * iters * t_iter, stream);
                const int nst = S * Wj;
                int fused = 0;
                if (nst > 1) {
                    const double rounds_f = std::ceil(std::min(icta, ni) / (double)kWarps) * std::ceil((S / C) / 32.0);
                    // the fused tail (fence, arrival counter, the last CTA's serial reduce; nothing overlaps it) costs
                    // ~2 us more than the same rounds in the separate launch, whose latency programmatic dependent
                    // launch hides (measured at N = 65536, same sweep shape: n_i = 8: 12.0 vs 9.9 us, n_i = 1: 8.9 vs 8.5)
                    const double fused_cost = (1.0 + rounds_f) * C_.c_row + (C > 1 ? C_.c_row : 0.0) + 4000.0;
                    // the partial records are written by every CTA at the end of a one-wave sweep and read back by the
                    // reduce: ~600 B per cycle for the round trip (measured: n_i = 512, 296 rows: 14.5 MB, +12 us)
                    const double sep_cost = C_.c_launch + std::ceil(nst / 32.0) * C_.c_row * 0.5 +
                                            (double)ni * nst * (REC * 8.0) / 600.0;
                    fused = fusable && (fused_cost < sep_cost || ctx->tune[6] > 1 || ctx->tune[5] == 3);
                    if (!fused && C > 1) continue;              // a cluster shape only makes sense fused
                    // warp columns only pay when the CTA adds them up in shared memory (the fused path); unfused, every
                    // column writes its own partial row (measured at N = 2^18, n_i = 1: 16.7 us against 10.4 us fused)
                    if (!fused && Wj > 1 && !want_ngb && ctx->tune[2] == 0 && ctx->tune[5] == 0) continue;
                    cost += fused ? fused_cost : sep_cost;
                }
                if (cost < best * (1 - 1e-9)) {
                    best = cost;
                    bL = L; bTL = TL; bWj = Wj; bS = S; bocc = occ; bfused = fused; bC = fused ? C : 1;
                }
            }
        }
    }
    if (best >= 1e300) return S2_EINVAL;

    ForceShape sh{};
    sh.L = bL;
    sh.TL = bTL;
    sh.Wj = bWj;
    sh.S = bS;
    sh.slice_len = (nj + bS - 1) / bS;
    // tiles: a ring of up to 4 buffers (<= ~96 KB per CTA so two CTAs still fit an SM); short slices are cut
    // into as many tiles as there are buffers so that every bulk copy is in flight from the start
    int tile = ctx->tune[4] > 0 ? ctx->tune[4] : 256;
    if (tile % 32 || tile < 32 || tile > tile_max) return S2_EINVAL;
    int stages;
    if (bWj > 1 && want_ngb) {   // one tile per CTA
        tile = std::max(32, (sh.slice_len + 31) / 32 * 32);
        if (tile > tile_max) return S2_EINVAL;
        stages = 1;
    } else {
        if (bWj > 1 && ctx->tune[4] == 0) tile = std::min(tile_max, 64 * bWj);   // >= 64 j per warp column and tile
        stages = std::max(2, std::min(4, (int)(98304 / ((size_t)npl * tile * 16))));
        if (ctx->tune[4] == 0 && sh.slice_len < stages * tile)
            tile = std::max(32, ((sh.slice_len + stages - 1) / stages + 31) / 32 * 32);
    }
    sh.tile = tile;
    sh.stages = stages;
    sh.fused = bfused;
    sh.cluster = bC;
    ctx->last_info[7] = bocc;
    if (!tuned) ctx->shape_cache[ckey] = std::make_pair(sh, bocc);
    *out = sh;
    return S2_OK;
}

// ---- a3-a8: force calls -------------------------------------------------------------------

// ---- a4 at the largest n_i: the uniform-operand sweep (force_sweep_bank_kernel, s2_force_fp64.cu) -----------
// The constant bank is one per device and module, shared by every context of the process: a sweep that uses it
// on another stream first waits for the event the previous user recorded after its last chunk.

// When the chunked sweep beats the shared-memory one (measured on B200 at N = 2^18, fp64 4th order, Gpairs/s
// bank / shared-memory): n_i = 49152: 481 / 488, 57344: 492 / 487, 61440: 502 / 489, 65536: 506 / 489, 81920: 510 / 489,
// 114688: 513 / 478, 131072: 517 / 482, 262144: 518 / 482 (with NN + lists 441 / 420).  Its launches overlap and a
// launch moves into the CTA slots its predecessor leaves free (the CTAs look for the next chunk's ticket at their
// start and 15 more times on their way through the chunk), so unlike the shared-memory sweep it does not care whether
// the grid is a whole number of residency rounds; below ~0.6 rounds (296 CTAs of 256 threads each) the per-launch
// costs win (n_i = 40960: 452 / 488 with 128-thread CTAs, 49152: 502 / 488).
// The 2nd-order variant measures -4 % and stays on the shared-memory sweep.
static bool bank_applies(const s2_ctx *ctx, int ni, int nj)
{
    if (ctx->precision != S2_FP64 || ctx->tune[8] == 1) return false;
    if (ctx->tune[8] >= 2) return true;   // 3: forced, without overlapping launches (A/B measurements); 4: forced, refilled
                                          // by stream-ordered copies (the documented-semantics fallback)
    for (int k = 0; k < 8; ++k)
        if (ctx->tune[k]) return false;   // an explicit launch shape was asked for
    // 6th order (round 2: two 126-register CTAs per SM instead of one of 158): N = 2^18, bank / shared-memory Gpairs/s:
    // n_i = 49152: 278 / 292, 65536: 294 / 293, 131072: 301 / 290, 262144: 302 / 290
    if (ctx->order == 6) return nj >= 8192 && ni >= 100000;
    return ctx->order == 4 && nj >= 8192 && ni >= 48000;
}

static cudaError_t dispatch_bank(int b, int order, unsigned flags, const ForceArgs &a, cudaStream_t st, int *geom)
{
    return b ? dispatch_force_fp64_bank1(order, flags, a, st, geom) : dispatch_force_fp64_bank0(order, flags, a, st, geom);
}

// Chunk c lives in bank c & 1 and carries ticket base + c + 1.  The host copies chunks 0 and 1 into the banks; from
// then on the sweep feeds itself: the last CTA of the launch of chunk c copies chunk c + 2 into the bank it has just
// swept and publishes ready[bank] = ticket(c + 2) (see force_sweep_bank_kernel).  Nothing but kernels sits in the
// stream, so the launches carry programmatic stream serialisation and overlap: the next one fills the SMs while this
// one drains (event-ordered refills: 498 Gpairs/s at n_i = 2^18; overlapped: 512).
static int run_force_bank(s2_ctx *ctx, ForceArgs &a, int ni, unsigned flags, int mode)
{
    int geom[3] = {0, 0, 0};
    CU(dispatch_bank(0, ctx->order, flags, a, ctx->stream, geom));
    const int chunk = geom[0];
    void *bank[2] = {nullptr, nullptr};
    CU(force_bank_address0(&bank[0]));
    CU(force_bank_address1(&bank[1]));
    const int npl = force_nplanes(S2_FP64, ctx->order, flags);
    const int nj = a.nj;
    const int nchunks = (nj + chunk - 1) / chunk;
    // CTAs of 128 threads (4 per SM) fill the rounds that consecutive launches share more finely; measured at N = 2^18
    // (128 / 256 threads, Gpairs/s): n_i = 49152: 502 / 481, 65536: 512 / 506, 81920: 514 / 510, 131072: 518 / 517,
    // 262144: 516 / 518.  Launches with decisions do not share rounds (they wait at their start): 256.
    const int threads = (flags == 0 && ctx->order == 4 && ni < 200000 && ctx->tune[8] != 3 && mode == kBankSelfRefill) ? 128 : geom[1];
    a.bank_threads = threads;
    a.bank_state = (double *)ctx->part.p;
    a.is_final = 1;
    a.rec = (double *)ctx->result.p;
    a.seg = (int *)ctx->list.p;
    a.segcap = ctx->ngb_cap;
    a.nslices_total = 1;
    // the planes of the predicted store are equally spaced unless some are skipped (2nd order)
    const size_t pitch = npl > 1 ? (size_t)((const char *)a.jp[1] - (const char *)a.jp[0]) : 0;
    bool equal_stride = npl > 1;
    for (int p = 1; p < npl; ++p)
        equal_stride = equal_stride && (const char *)a.jp[p] == (const char *)a.jp[0] + p * pitch;

    std::lock_guard<std::mutex> lock(g_bank_mu);
    BankOwner &own = g_bank[ctx->device];
    if (!own.ev) CU(cudaEventCreateWithFlags(&own.ev, cudaEventDisableTiming));
    if (!own.flags) {   // 64 bytes shared by every context of the device (not a context's buffer): freed by the last s2_close
        CU(cudaMalloc((void **)&own.flags, 64));
        CU(cudaMemsetAsync(own.flags, 0, 64, ctx->stream));   // ordered before this stream's first sweep; others wait on own.ev
    }
    // inside a stream capture (CUDA graph) events cannot tie the graph to work outside it: the caller orders
    // replays of such a graph against other users of the banks himself
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    CU(cudaStreamIsCapturing(ctx->stream, &cap));
    const bool capturing = cap != cudaStreamCaptureStatusNone;
    if (!capturing && own.used && own.stream != ctx->stream) CU(cudaStreamWaitEvent(ctx->stream, own.ev, 0));
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[2], ctx->stream));
    const unsigned base = own.ticket;
    if (mode == kBankSelfRefill) own.ticket += (unsigned)nchunks;
    auto copy_chunk = [&](int c) -> cudaError_t {   // chunk c of every plane -> bank c & 1, in stream order
        const int cnt = std::min(chunk, nj - c * chunk);
        if (equal_stride)   // one strided copy moves the chunk of every plane
            return cudaMemcpy2DAsync(bank[c & 1], (size_t)chunk * sizeof(double2), (const double2 *)a.jp[0] + a.j_first + (size_t)c * chunk, pitch,
                                     (size_t)cnt * sizeof(double2), npl, cudaMemcpyDeviceToDevice, ctx->stream);
        for (int p = 0; p < npl; ++p) {
            cudaError_t e = cudaMemcpyAsync((double2 *)bank[c & 1] + (size_t)p * chunk, (const double2 *)a.jp[p] + a.j_first + (size_t)c * chunk,
                                            (size_t)cnt * sizeof(double2), cudaMemcpyDeviceToDevice, ctx->stream);
            if (e != cudaSuccess) return e;
        }
        return cudaSuccess;
    };
    if (mode == kBankSelfRefill)
        for (int c = 0; c < std::min(2, nchunks); ++c) CU(copy_chunk(c));   // the later chunks are copied by the kernels
    // launch -1 sweeps nothing: it gathers the i-particles, parks them and zeroes the running state, so that every
    // chunk launch finds its inputs complete and may overlap its predecessor
    a.bank_j0 = 0; a.bank_cnt = 0; a.bank_first = 1; a.bank_last = 0; a.bank_pdl = 0; a.bank_wait_early = 0;
    a.bank_id = 0; a.bank_flags = nullptr; a.bank_ticket = 0; a.bank_spin = 0; a.bank_next_known = 1;
    a.bank_self = nullptr; a.bank_next_j0 = 0; a.bank_next_cnt = 0;
    CU(dispatch_bank(0, ctx->order, flags, a, ctx->stream, nullptr));
    ctx->launches++;
    const bool overlap = !capturing && ctx->tune[8] != 3;   // 3: forced, plain launches (A/B measurements)
    for (int c = 0; c < nchunks; ++c) {
        const int b = c & 1;
        a.bank_j0 = a.j_first + c * chunk;
        a.bank_cnt = std::min(chunk, nj - c * chunk);
        a.bank_first = 0;
        a.bank_last = c == nchunks - 1;
        a.bank_id = b;
        if (mode == kBankHostRefill) {
            // Documented semantics only: the bank is written by a stream-ordered copy between two ordinary launches
            // (the copy follows the launch of chunk c - 2, the last reader of this bank, and precedes this launch).
            CU(copy_chunk(c));
            a.bank_flags = nullptr; a.bank_ticket = 0; a.bank_spin = 0; a.bank_next_known = 1; a.bank_self = nullptr;
            a.bank_next_j0 = 0; a.bank_next_cnt = 0; a.bank_pdl = 0; a.bank_wait_early = 0;
            CU(dispatch_bank(b, ctx->order, flags, a, ctx->stream, nullptr));
            ctx->launches++;
            continue;
        }
        a.bank_flags = own.flags;
        a.bank_ticket = base + (unsigned)c + 1u;
        a.bank_spin = c >= 2;
        a.bank_next_known = c == 0 || c == nchunks - 1;
        a.bank_self = (double2 *)bank[b];
        a.bank_next_j0 = a.j_first + (c + 2) * chunk;
        a.bank_next_cnt = c + 2 < nchunks ? std::min(chunk, nj - (c + 2) * chunk) : 0;
        a.bank_pdl = overlap && c > 0;
        a.bank_wait_early = c == 0 || flags != 0;   // decisions (thresholds) are carried from chunk to chunk
        CU(dispatch_bank(b, ctx->order, flags, a, ctx->stream, nullptr));
        ctx->launches++;
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[3], ctx->stream));
    if (!capturing) {
        CU(cudaEventRecord(own.ev, ctx->stream));
        own.stream = ctx->stream;
        own.used = true;
    }

    int *li = ctx->last_info;
    li[0] = nchunks; li[1] = 1; li[2] = 1; li[3] = (ni + threads - 1) / threads; li[4] = threads; li[5] = 0;
    li[6] = mode == kBankSelfRefill ? 3 : 5;
    li[7] = geom[2] * geom[1] / threads; li[8] = 1; li[9] = 1;
    return S2_OK;
}


// First use of the self-refilling sweep on a device: run it once next to the shared-memory sweep on (a part of) the
// caller's own problem -- at least three chunks, so that the last-CTA refill, the ticket hand-over and the
// overlapping launches are all exercised -- and compare every record.  The self-refill writes the constant bank from
// device code and relies on the next launch seeing the new contents; CUDA documents neither, so the
// library only keeps using it where it has just seen it work, and otherwise falls back for good to refilling the banks
// with stream-ordered copies between ordinary launches (documented semantics, measured ~4 % slower).
static int bank_selftest(s2_ctx *ctx, int ni, const int *d_i_addr, bool explicit_i, double eps2, bool *ok)
{
    const int nj_save = ctx->nj_pred, t8 = ctx->tune[8], jc_save = ctx->j_count;
    ctx->j_count = 0;
    const int ni_t = std::min(ni, 65536);
    const int nj_t = std::min(nj_save, 8 * 1024);
    *ok = false;
    Buf ref;
    int rc = dev_reserve(ctx, ref, (size_t)ni_t * REC * sizeof(double));
    if (rc != S2_OK) return rc;
    ctx->in_selftest = true;
    ctx->nj_pred = nj_t;
    ctx->tune[8] = 1;
    rc = run_force(ctx, ni_t, d_i_addr, nullptr, explicit_i, eps2, 0, false);
    if (rc == S2_OK) {
        cudaError_t e = cudaMemcpyAsync(ref.p, ctx->result.p, (size_t)ni_t * REC * sizeof(double), cudaMemcpyDeviceToDevice, ctx->stream);
        if (e != cudaSuccess) rc = fail_cuda(ctx, e);
    }
    ctx->tune[8] = 2;
    for (int rep = 0; rep < 2 && rc == S2_OK; ++rep) {   // twice back to back: the second sweep starts on banks the first one left
        rc = run_force(ctx, ni_t, d_i_addr, nullptr, explicit_i, eps2, 0, false);
        if (rc == S2_OK) {
            cudaError_t e = launch_compare_records((const double *)ref.p, (const double *)ctx->result.p, ni_t, ctx->order, 1e-11,
                                                   (int *)ctx->flags.p + 2, ctx->stream);
            if (e != cudaSuccess) rc = fail_cuda(ctx, e);
            ctx->launches++;
        }
    }
    ctx->tune[8] = t8;
    ctx->nj_pred = nj_save;
    ctx->j_count = jc_save;
    ctx->in_selftest = false;
    ctx->calc_done = false;
    if (rc == S2_OK) {
        cudaError_t e = cudaMemcpyAsync(ctx->h_flags + 2, (int *)ctx->flags.p + 2, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream);
        if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
        if (e == cudaSuccess) e = cudaMemsetAsync((int *)ctx->flags.p + 2, 0, sizeof(int), ctx->stream);
        if (e != cudaSuccess) rc = fail_cuda(ctx, e);
        else *ok = ctx->h_flags[2] == 0;
    }
    dev_release(ctx, ref);
    return rc;
}

static int bank_choose_mode(s2_ctx *ctx, int ni, const int *d_i_addr, bool explicit_i, double eps2, int *mode)
{
    if (ctx->in_selftest) { *mode = kBankSelfRefill; return S2_OK; }
    if (ctx->tune[8] == 4) { *mode = kBankHostRefill; return S2_OK; }
    int m;
    {
        std::lock_guard<std::mutex> lock(g_bank_mu);
        m = g_bank[ctx->device].mode;
    }
    if (m == 0) {
        // a sweep of at most two chunks never refills a bank from a kernel (the host copies both): nothing to verify yet
        int geom[3] = {0, 0, 0};
        ForceArgs dummy{};
        CU(dispatch_force_fp64_bank0(ctx->order, 0, dummy, ctx->stream, geom));
        if ((ctx->j_count > 0 ? ctx->j_count : ctx->nj_pred) <= 2 * geom[0]) { *mode = kBankSelfRefill; return S2_OK; }
        cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
        CU(cudaStreamIsCapturing(ctx->stream, &cap));
        if (cap != cudaStreamCaptureStatusNone) { *mode = kBankHostRefill; return S2_OK; }   // cannot test inside a capture
        bool ok = false;
        int rc = bank_selftest(ctx, ni, d_i_addr, explicit_i, eps2, &ok);
        if (rc != S2_OK) return rc;
        m = ok ? kBankSelfRefill : kBankHostRefill;
        std::lock_guard<std::mutex> lock(g_bank_mu);
        g_bank[ctx->device].mode = m;
    }
    *mode = m;
    return S2_OK;
}

// fp32 fix-up (reading R-F32): an i-particle is re-evaluated in fp64 when sqrt(sum q^2) (|v_i| + v_esc) > 8 |jerk_i|.
// Measured on configs 1, 3, 4, 5: the estimate is 0.46 ... 7 times the true rms pair term R_i, so every particle with
// R_i > 17 |jerk_i| is caught (fp32 then stays below 4e-7 x 17 = 7e-6 of the total) and 0.3-0.8 % of the particles are flagged.
constexpr double kF32FlagThreshold = 8.0;

// Calls with at most this many i-particles keep their i-list and their final records in pinned host memory that the
// kernels access directly (transfers dominate small calls).  Measured host round trip
// (calc + get_results): N = 64: 38-41 -> 26 us; N = 65536, n_i = 1: 37 -> 27.5, n_i = 32: 40 -> 34, n_i = 256: 72 -> 73
// (the record writes over the host link start to cost more than the copy they save), hence the limit
constexpr int kZeroCopyNi = 128;

int run_force(s2_ctx *ctx, int ni, const int *d_i_addr, const double *d_h2, bool explicit_i, double eps2,
              unsigned flags, bool host_call)
{
    // the j-range summed over: all predicted particles, or one rank's share under j-sharding (s2_set_j_range)
    const int j_first = ctx->j_count > 0 ? ctx->j_first : 0;
    const int nj_eff = ctx->j_count > 0 ? ctx->j_count : ctx->nj_pred;
    if ((long long)j_first + nj_eff > ctx->nj_pred) return S2_ERANGE;
    const bool bank = bank_applies(ctx, ni, nj_eff);
    ForceShape sh{};
    int rc = S2_OK;
    ctx->csr_valid = false;
    int bank_mode = 0;
    if (bank) {
        rc = bank_choose_mode(ctx, ni, d_i_addr, explicit_i, eps2, &bank_mode);
        if (rc != S2_OK) return rc;
    }
    if (bank) {   // one lane per i, one "slice": the chunks of the constant bank are swept launch by launch
        sh.L = 1; sh.TL = 0; sh.Wj = 1; sh.S = 1; sh.slice_len = nj_eff; sh.tile = 256; sh.stages = 2; sh.cluster = 1;
        rc = dev_reserve(ctx, ctx->part, (size_t)ni * (REC + 10) * sizeof(double));   // running sums + parked i-state
    } else {
        rc = choose_shape(ctx, ni, nj_eff, flags, &sh);
    }
    if (rc != S2_OK) return rc;
    const int nst = sh.S * sh.Wj;
    const bool want_ngb = flags & S2_WANT_NGB;
    const bool final_direct = nst == 1;
    // without neighbour lists the combine is fused into the sweep launch (last CTA of an i-group reduces)
    const int icta_ = sh.L == 0 ? kThreads * force_ipt(ctx->precision) / std::max(1, sh.TL) : (kWarps / sh.Wj) * (32 / sh.L);
    const int Gi_ = (ni + icta_ - 1) / icta_;
    const bool fused = sh.fused != 0;
    // opt-in (s2_set_tuning key 5 = 2): combine the j-slices with fp64 atomics instead of the reduce kernel
    const bool atomic = ctx->tune[5] == 2 && flags == 0 && nst > 1 && !fused && !bank;
    // small calls: the final records are written straight into pinned host memory
    // (calls made with host arrays only: a caller that keeps its i-list on the device is not latency-bound by copies)
    const bool host_res = host_call && ni <= kZeroCopyNi && !bank && !atomic && ctx->tune[9] != 1 && ctx->tune[9] != 3;

    rc = host_res ? pinned_reserve(ctx, &ctx->h_res, &ctx->h_res_bytes, 0, (size_t)kZeroCopyNi * REC * sizeof(double))
                  : dev_reserve(ctx, ctx->result, (size_t)ni * REC * sizeof(double));
    double *const resp = host_res ? (double *)ctx->h_res : (double *)ctx->result.p;
    if (rc == S2_OK && !final_direct && !atomic) rc = dev_reserve(ctx, ctx->part, (size_t)nst * ni * REC * sizeof(double));
    if (rc == S2_OK && fused && (size_t)Gi_ * sizeof(unsigned) > ctx->counters.bytes) {
        rc = dev_reserve(ctx, ctx->counters, (size_t)Gi_ * sizeof(unsigned));
        if (rc == S2_OK) CU(cudaMemsetAsync(ctx->counters.p, 0, ctx->counters.bytes, ctx->stream));
    }
    int segcap = 0;
    if (want_ngb) {
        if (ctx->ngb_cap <= 0) return S2_EINVAL;
        // a record covers at most one slice (a warp column takes a part of every tile of the slice)
        segcap = final_direct ? ctx->ngb_cap : std::min(ctx->ngb_cap, sh.slice_len);
        if (rc == S2_OK) rc = dev_reserve(ctx, ctx->list, (size_t)ni * ctx->ngb_cap * sizeof(int));
        if (rc == S2_OK && !final_direct) rc = dev_reserve(ctx, ctx->seg, (size_t)ni * nst * segcap * sizeof(int));
    }
    if (rc != S2_OK) return rc;

    ForceArgs a{};
    const int np = nplanes(ctx->order), nq = n_qplanes(ctx->precision, ctx->order);
    // planes staged per tile, in the order the policy reads them.  A 2nd-order sweep skips the velocity planes:
    // fp64 P0 P1 P3, fp32 F0 F1, double-single D0 D1 D3 (P3 / D3 carry the id).
    int nsel = 0;
    int sel[kMaxPlanes];
    if (ctx->precision == S2_FP64) {
        if (ctx->order == 2) { sel[0] = 0; sel[1] = 1; sel[2] = 3; nsel = 3; }
        else for (int k = 0; k < np; ++k) sel[nsel++] = k;
        for (int k = 0; k < nsel; ++k) {
            a.jp[k] = plane(ctx, sel[k]);
            a.ip[k] = explicit_i ? (const void *)((double2 *)ctx->iplanes.p + (size_t)sel[k] * ni) : a.jp[k];
        }
    } else {
        if (ctx->order == 2 && ctx->precision == S2_FP32) { sel[0] = 0; sel[1] = 1; nsel = 2; }
        else if (ctx->order == 2) { sel[0] = 0; sel[1] = 1; sel[2] = 3; nsel = 3; }
        else for (int k = 0; k < nq; ++k) sel[nsel++] = k;
        for (int k = 0; k < nsel; ++k) {
            a.jp[k] = qplane(ctx, sel[k]);
            a.ip[k] = explicit_i ? (const void *)((float4 *)ctx->iqplanes.p + (size_t)sel[k] * ni) : a.jp[k];
        }
    }
    if (ctx->precision != S2_FP64 && flags) {   // decisions are taken on fp64 positions in every mode
        for (int k = 0; k < 2; ++k) {
            a.jp[nsel + k] = plane(ctx, k);
            a.ip[nsel + k] = explicit_i ? (const void *)((double2 *)ctx->iplanes.p + (size_t)k * ni) : a.jp[nsel + k];
        }
    }
    a.i_addr = explicit_i ? nullptr : d_i_addr;
    a.h2 = d_h2;
    if (host_call && !explicit_i && ni <= kZeroCopyNi && ctx->tune[9] != 1) {
        // d_i_addr / d_h2 point into pinned host memory (s2_calc_ilist).  A few CTAs read them in place; a wide grid
        // (every CTA of every j-slice gathers its i-particles) would queue a thousand reads on the host link
        // (measured +11 us at 148 CTAs), so there they are copied once to the device first
        const long long ctas = (long long)Gi_ * sh.S;
        if (ctas > 8 || ctx->tune[9] == 2) {
            const size_t b_addr = align16((size_t)ni * sizeof(int)), b_h2 = d_h2 ? (size_t)ni * sizeof(double) : 0;
            rc = dev_reserve(ctx, ctx->i_addr, b_addr + b_h2);
            if (rc != S2_OK) return rc;
            CU(cudaMemcpyAsync(ctx->i_addr.p, d_i_addr, b_addr + b_h2, cudaMemcpyHostToDevice, ctx->stream));
            a.i_addr = (const int *)ctx->i_addr.p;
            a.h2 = d_h2 ? (const double *)((char *)ctx->i_addr.p + b_addr) : nullptr;
        }
    }
    a.jid_plane = plane(ctx, 3);
    a.ni = ni;
    a.nj = nj_eff;
    a.j_first = j_first;
    a.eps2 = eps2;
    a.S = sh.S;
    a.slice_len = sh.slice_len;
    a.Wj = sh.Wj;
    a.tile = sh.tile;
    a.stages = sh.stages;
    a.nslices_total = nst;
    a.is_final = final_direct ? 1 : 0;
    a.rec = final_direct ? resp : (double *)ctx->part.p;
    a.seg = final_direct ? (int *)ctx->list.p : (int *)ctx->seg.p;
    a.segcap = segcap;
    a.overflow_flag = (int *)ctx->flags.p;
    a.ngb_cap = ctx->ngb_cap;
    a.fused = fused ? 1 : 0;
    a.cluster = fused ? sh.cluster : 1;
    a.counters = (unsigned *)ctx->counters.p;
    a.out_final = resp;
    a.order = ctx->order;
    a.atomic = atomic ? 1 : 0;
    // fp32, reading R-F32: the sweep leaves sum_j q_j^2 per (slice, i); particles whose jerk is a strongly cancelling sum
    // are then re-evaluated in fp64 (tune key 9 = 4 switches the fix-up off, for A/B measurements)
    const bool fixup = ctx->precision == S2_FP32 && ctx->order != 2 && !atomic && ctx->tune[9] != 4;
    F32Flag f32{};
    int fix_S = 1, fix_slice = nj_eff, fix_kcap = 2;
    if (fixup) {
        // j-slices of the fix-up sweep: <= 256 particles each, so that even one flagged particle is spread over many
        // warps; at most 2^20 partial rows [slice][flagged particle], with room for n_i / 16 flagged particles (any beyond
        // that are swept unsliced by the same kernel)
        fix_kcap = std::min((ni + 1) / 2 * 2, std::max(64, ni / 16 / 2 * 2));   // room for 6 % flagged (measured: 0.3-0.8 %)
        // slice length: ~4096 j keeps the sweep near 290 Gpairs/s once there is an item per warp (measured: n_i = 65536,
        // N = 65536: 185 Gpairs/s with 4096-particle slices, 83 with 256-particle ones; N = n_i = 2^18: 291 against 195 with
        // 65536-particle ones); a short i-list flags a handful of particles (~n_i / 200), which want short slices instead
        {
            const int warps = 16 * ctx->sm_count, groups = std::max(1, ni / 400);
            const int s_long = std::max(1, nj_eff / 4096), s_short = std::max(1, (nj_eff + 255) / 256);
            fix_S = (long long)groups * s_long >= warps ? s_long : std::min(s_short, std::max(s_long, (warps + groups - 1) / groups));
            fix_S = std::max(1, std::min(fix_S, std::max(1, (1 << 20) / fix_kcap)));
        }
        fix_slice = (nj_eff + fix_S - 1) / fix_S;
        fix_S = (nj_eff + fix_slice - 1) / fix_slice;
        rc = dev_reserve(ctx, ctx->wq, (size_t)nst * ni * sizeof(float));
        if (rc == S2_OK) rc = dev_reserve(ctx, ctx->fix, 16 + (size_t)ni * sizeof(int));
        // arrival counters of the fix-up groups: a buffer of their own (nothing else is ever written there), zeroed when
        // it is allocated; the kernel resets every counter it used, so they are zero between calls
        const size_t b_arr = (size_t)(ni / 2 + 1) * sizeof(unsigned);
        if (rc == S2_OK && b_arr > ctx->fixarr.bytes) {
            rc = dev_reserve(ctx, ctx->fixarr, b_arr);
            if (rc == S2_OK) CU(cudaMemsetAsync(ctx->fixarr.p, 0, ctx->fixarr.bytes, ctx->stream));
        }
        if (rc == S2_OK && fix_S > 1) rc = dev_reserve(ctx, ctx->fixpart, (size_t)fix_S * fix_kcap * (ctx->order == 6 ? 10 : 7) * sizeof(double));
        if (rc != S2_OK) return rc;
        a.wq = (float *)ctx->wq.p;
        a.fix_count = (int *)ctx->fix.p;   // zeroed by the sweep itself
        f32.wq = (const float *)ctx->wq.p;
        f32.nst = nst;
        f32.v2 = explicit_i ? (const double2 *)ctx->iplanes.p + (size_t)2 * ni : plane(ctx, 2);
        f32.v3 = explicit_i ? (const double2 *)ctx->iplanes.p + (size_t)3 * ni : plane(ctx, 3);
        f32.thresh = ctx->tune[9] == 5 ? 0.0 : kF32FlagThreshold;   // 5: flag every i-particle (tests of the fix-up itself)
        f32.count = (int *)ctx->fix.p;
        f32.pos_list = (int *)((char *)ctx->fix.p + 16);
    }
    if (atomic) CU(cudaMemsetAsync(ctx->result.p, 0, (size_t)ni * REC * sizeof(double), ctx->stream));

    if (want_ngb) CU(cudaMemsetAsync(ctx->flags.p, 0, sizeof(int), ctx->stream));   // overflow flag of this call
    if (bank) {
        rc = run_force_bank(ctx, a, ni, flags, bank_mode);
        if (rc != S2_OK) return rc;
        ctx->ran_force = true;
        ctx->ran_reduce = false;
        ctx->calc_done = true;
        ctx->res_on_host = false;
        ctx->ni_last = ni;
        ctx->flags_last = flags;
        return S2_OK;
    }
    const int icta = icta_;
    dim3 grid((ni + icta - 1) / icta, sh.S);
    size_t smem = force_smem_bytes(force_nplanes(ctx->precision, ctx->order, flags), sh.tile, sh.stages);
    smem = std::max(smem, (size_t)kSmemHeader + (size_t)icta * sh.Wj * REC * sizeof(double));   // record block of the combines
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[2], ctx->stream));
    CU(dispatch(ctx->precision, ctx->order, flags, sh.L == 0 ? (sh.TL > 1 ? -sh.TL : 0) : sh.L, grid, smem, a, ctx->stream, false, nullptr));
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[3], ctx->stream));
    ctx->launches++;
    ctx->ran_force = true;
    ctx->ran_reduce = false;
    bool flagged_inline = false;
    if (!final_direct && !fused && !atomic) {
        ReduceArgs r{};
        r.part = (const double *)ctx->part.p;
        r.out = resp;
        r.seg = (const int *)ctx->seg.p;
        r.list = (int *)ctx->list.p;
        r.jid_plane = plane(ctx, 3);
        r.ni = ni;
        r.nslices_total = nst;
        r.segcap = segcap;
        r.ngb_cap = ctx->ngb_cap;
        r.order = ctx->order;
        r.flags = flags;
        r.overflow_flag = (int *)ctx->flags.p;
        ctx->bts_hook_done = false;
        if (ctx->bts_hook && !ctx->in_selftest && !fixup && flags == 0 && !host_res && reduce_by_warp_kernel(r)) {
            r.bts = *ctx->bts_hook;          // the integrator's corrector rides on the combine (fp32: the fix-up must run first)
            r.has_bts = 1;
            ctx->bts_hook_done = true;
        }
        if (fixup && reduce_by_warp_kernel(r)) {   // reduce_kernel flags while it has the final sums at hand: no flag launch
            r.f32 = f32;
            r.f32.i_addr = a.i_addr;
            flagged_inline = true;
        }
        if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[4], ctx->stream));
        CU(launch_reduce(r, ctx->stream));
        if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[5], ctx->stream));
        ctx->launches++;
        ctx->ran_reduce = true;
    }
    if (fixup) {
        if (!ctx->ran_reduce && ctx->timing) CU(cudaEventRecord(ctx->ev_t[4], ctx->stream));
        const int np64 = nplanes(ctx->order);
        f32.i_addr = a.i_addr;
        if (!flagged_inline) {
            CU(launch_fp32_flag(resp, f32, ni, ctx->stream));
            ctx->launches++;
        }
        // the flagged particles through the fp64 fix-up sweep (fp32_fix_sweep_kernel, s2_force_fp64.cu)
        ForceArgs b = a;
        for (int k = 0; k < kMaxPlanes; ++k) b.jp[k] = b.ip[k] = nullptr;
        for (int k = 0; k < np64; ++k) {
            b.jp[k] = plane(ctx, k);
            b.ip[k] = explicit_i ? (const void *)((double2 *)ctx->iplanes.p + (size_t)k * ni) : b.jp[k];
        }
        b.S = fix_S; b.slice_len = fix_slice;
        b.h2 = nullptr; b.rec = resp; b.wq = nullptr; b.pos_list = f32.pos_list; b.ni_dev = f32.count;
        b.fix_part = (double *)ctx->fixpart.p;
        b.fix_kcap = fix_kcap;
        b.fix_arrive = (unsigned *)ctx->fixarr.p;
        CU(launch_fp32_fix(b, ctx->sm_count, ctx->stream));
        if (ctx->timing) CU(cudaEventRecord(ctx->ev_t[5], ctx->stream));
        ctx->launches++;
        ctx->ran_reduce = true;
        ctx->fix_last = -1;
    }
    int *li = ctx->last_info;
    li[0] = sh.S; li[1] = sh.L == 0 ? std::max(1, sh.TL) : sh.L; li[2] = sh.Wj; li[3] = (int)(grid.x * grid.y); li[4] = kThreads;
    li[5] = (int)smem; li[6] = final_direct ? 0 : (fused ? 2 : (atomic ? 4 : 1));
    li[8] = sh.L == 0 ? force_ipt(ctx->precision) : 1; li[9] = a.cluster;
    ctx->calc_done = true;
    ctx->res_on_host = host_res;
    ctx->ni_last = ni;
    ctx->flags_last = flags;
    return S2_OK;
}

static int check_calc(s2_ctx *ctx, int ni, unsigned flags, const void *h2)
{
    if (!ctx || ni <= 0) return S2_EINVAL;
    if (flags & ~(unsigned)(S2_WANT_NN | S2_WANT_NGB)) return S2_EINVAL;
    if ((flags & S2_WANT_NGB) && (!h2 || ctx->ngb_cap <= 0)) return S2_EINVAL;
    if (!ctx->predicted) return S2_ESTATE;
    return S2_OK;
}

extern "C" int s2_calc_ilist_device(s2_ctx *ctx, int ni, const int *d_i_address, const double *d_h2, double eps2,
                                    unsigned flags)
{
    int rc = check_calc(ctx, ni, flags, d_h2);
    if (rc != S2_OK) return rc;
    if (!d_i_address) return S2_EINVAL;
    CU(cudaSetDevice(ctx->device));
    return run_force(ctx, ni, d_i_address, d_h2, false, eps2, flags, false);
}

extern "C" int s2_calc_ilist(s2_ctx *ctx, int ni, const int *i_address, const double *h2, double eps2,
                             unsigned flags)
{
    int rc = check_calc(ctx, ni, flags, h2);
    if (rc != S2_OK) return rc;
    if (!i_address) return S2_EINVAL;
    for (int k = 0; k < ni; ++k)
        if (i_address[k] < 0 || i_address[k] >= ctx->nj_pred) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    const bool ngb = flags & S2_WANT_NGB;
    const size_t b_addr = align16((size_t)ni * sizeof(int)), b_h2 = ngb ? (size_t)ni * sizeof(double) : 0;
    if (ni <= kZeroCopyNi && ctx->tune[9] != 1) {
        // small call: the kernels read the i-list (and h2) from pinned host memory; two buffers alternate, each
        // guarded by an event recorded behind the kernels that read it
        const int k = ctx->il_turn;
        ctx->il_turn ^= 1;
        CU(cudaEventSynchronize(ctx->ev_il[k]));
        rc = pinned_reserve(ctx, &ctx->h_il[k], &ctx->h_il_bytes[k], 0,
                            align16((size_t)kZeroCopyNi * sizeof(int)) + (size_t)kZeroCopyNi * sizeof(double));
        if (rc != S2_OK) return rc;
        memcpy(ctx->h_il[k], i_address, (size_t)ni * sizeof(int));
        if (ngb) memcpy((char *)ctx->h_il[k] + b_addr, h2, b_h2);
        rc = run_force(ctx, ni, (const int *)ctx->h_il[k], ngb ? (const double *)((char *)ctx->h_il[k] + b_addr) : nullptr,
                       false, eps2, flags, true);
        if (rc != S2_OK) return rc;
        CU(cudaEventRecord(ctx->ev_il[k], ctx->stream));
        return S2_OK;
    }
    CU(cudaEventSynchronize(ctx->ev_io));
    rc = pinned_reserve(ctx, &ctx->h_io, &ctx->h_io_bytes, 0, b_addr + b_h2);
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->i_addr, b_addr + b_h2);
    if (rc != S2_OK) return rc;
    memcpy(ctx->h_io, i_address, (size_t)ni * sizeof(int));
    if (ngb) memcpy((char *)ctx->h_io + b_addr, h2, b_h2);
    CU(cudaMemcpyAsync(ctx->i_addr.p, ctx->h_io, b_addr + b_h2, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaEventRecord(ctx->ev_io, ctx->stream));
    return run_force(ctx, ni, (const int *)ctx->i_addr.p,
                     ngb ? (const double *)((char *)ctx->i_addr.p + b_addr) : nullptr, false, eps2, flags, true);
}

extern "C" int s2_calc_ilist_batch(s2_ctx *ctx, int k, const int *ni, const int *i_address, const double *h2, double eps2,
                                   unsigned flags)
{
    if (!ctx || k <= 0 || !ni) return S2_EINVAL;
    long long tot = 0;
    for (int b = 0; b < k; ++b) {
        if (ni[b] <= 0) return S2_EINVAL;
        tot += ni[b];
    }
    if (tot > 0x7fffffffLL) return S2_ERANGE;
    // i-particles are independent of one another: the concatenation is one i-list
    return s2_calc_ilist(ctx, (int)tot, i_address, h2, eps2, flags);
}

static inline void split_ds_host(double x, float *hi, float *lo)
{
    *hi = (float)x;
    *lo = (float)(x - (double)*hi);
}

extern "C" int s2_calc_explicit(s2_ctx *ctx, int ni, const int *id, const double *pos, const double *vel,
                                const double *acc, const double *h2, double eps2, unsigned flags)
{
    int rc = check_calc(ctx, ni, flags, h2);
    if (rc != S2_OK) return rc;
    if (!id || !pos || (ctx->order != 2 && !vel) || (ctx->order == 6 && !acc)) return S2_EINVAL;
    CU(cudaSetDevice(ctx->device));
    const bool ngb = flags & S2_WANT_NGB;
    const int np = nplanes(ctx->order), nq = n_qplanes(ctx->precision, ctx->order);
    const size_t b_p = (size_t)np * ni * sizeof(double2), b_q = (size_t)nq * ni * sizeof(float4);
    const size_t b_h2 = ngb ? (size_t)ni * sizeof(double) : 0;
    CU(cudaEventSynchronize(ctx->ev_io));
    rc = pinned_reserve(ctx, &ctx->h_io, &ctx->h_io_bytes, 0, b_p + b_q + b_h2);
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->iplanes, b_p);
    if (rc == S2_OK && nq) rc = dev_reserve(ctx, ctx->iqplanes, b_q);
    if (rc == S2_OK && ngb) rc = dev_reserve(ctx, ctx->i_h2, b_h2);
    if (rc != S2_OK) return rc;
    // pack the i-particles into the same plane layout the predictor writes for j (pure data movement
    // plus the fp64 -> (hi, lo) float split of the storage format)
    double2 *P = (double2 *)ctx->h_io;
    float4 *Q = (float4 *)((char *)ctx->h_io + b_p);
    for (int k = 0; k < ni; ++k) {
        static const double zero3[3] = {0.0, 0.0, 0.0};
        const double *x = pos + 3 * (size_t)k, *v = vel ? vel + 3 * (size_t)k : zero3;
        int idk = id[k];
        double idbits;
        memset(&idbits, 0, sizeof idbits);
        memcpy(&idbits, &idk, sizeof idk);   // little-endian: low word = id, high word = 0
        P[k] = make_double2(x[0], x[1]);
        P[(size_t)ni + k] = make_double2(x[2], 0.0);
        P[(size_t)2 * ni + k] = make_double2(v[0], v[1]);
        P[(size_t)3 * ni + k] = make_double2(v[2], idbits);
        const double *ac = ctx->order == 6 ? acc + 3 * (size_t)k : nullptr;
        if (ac) {
            P[(size_t)4 * ni + k] = make_double2(ac[0], ac[1]);
            P[(size_t)5 * ni + k] = make_double2(ac[2], 0.0);
        }
        float idf;
        memcpy(&idf, &idk, sizeof idf);
        if (ctx->precision == S2_FP32) {
            float xh[3], xl[3];
            for (int c = 0; c < 3; ++c) split_ds_host(x[c], &xh[c], &xl[c]);
            Q[k] = make_float4(xh[0], xh[1], xh[2], 0.f);
            Q[(size_t)ni + k] = make_float4(xl[0], xl[1], xl[2], idf);
            Q[(size_t)2 * ni + k] = make_float4((float)v[0], (float)v[1], (float)v[2], 0.f);
            if (ac) Q[(size_t)3 * ni + k] = make_float4((float)ac[0], (float)ac[1], (float)ac[2], 0.f);
        } else if (ctx->precision == S2_DS) {
            float h[9], l[9];
            for (int c = 0; c < 3; ++c) {
                split_ds_host(x[c], &h[c], &l[c]);
                split_ds_host(v[c], &h[3 + c], &l[3 + c]);
                if (ac) split_ds_host(ac[c], &h[6 + c], &l[6 + c]);
            }
            Q[k] = make_float4(h[0], l[0], h[1], l[1]);
            Q[(size_t)ni + k] = make_float4(h[2], l[2], 0.f, 0.f);
            Q[(size_t)2 * ni + k] = make_float4(h[3], l[3], h[4], l[4]);
            Q[(size_t)3 * ni + k] = make_float4(h[5], l[5], idf, 0.f);
            if (ac) {
                Q[(size_t)4 * ni + k] = make_float4(h[6], l[6], h[7], l[7]);
                Q[(size_t)5 * ni + k] = make_float4(h[8], l[8], 0.f, 0.f);
            }
        }
    }
    if (ngb) memcpy((char *)ctx->h_io + b_p + b_q, h2, b_h2);
    CU(cudaMemcpyAsync(ctx->iplanes.p, ctx->h_io, b_p, cudaMemcpyHostToDevice, ctx->stream));
    if (nq) CU(cudaMemcpyAsync(ctx->iqplanes.p, (char *)ctx->h_io + b_p, b_q, cudaMemcpyHostToDevice, ctx->stream));
    if (ngb) CU(cudaMemcpyAsync(ctx->i_h2.p, (char *)ctx->h_io + b_p + b_q, b_h2, cudaMemcpyHostToDevice, ctx->stream));
    CU(cudaEventRecord(ctx->ev_io, ctx->stream));
    return run_force(ctx, ni, nullptr, ngb ? (const double *)ctx->i_h2.p : nullptr, true, eps2, flags, true);
}

// ---- a9: results --------------------------------------------------------------------------

// flag 0: a neighbour list overflowed in the last call; flag 1: a device-side commit dropped an address.  Neither
// can be set unless lists were asked for or s2_commit_j_device ran, and then the copy is skipped (small calls)
static int fetch_flags(s2_ctx *ctx)
{
    if (!(ctx->flags_last & S2_WANT_NGB) && !ctx->flags_dirty) {
        ctx->h_flags[0] = ctx->h_flags[1] = 0;
        return S2_OK;
    }
    CU(cudaMemcpyAsync(ctx->h_flags, ctx->flags.p, 2 * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    ctx->flags_dirty = false;
    return S2_OK;
}

static int post_sync_status(s2_ctx *ctx)
{
    if (ctx->h_flags[1]) {   // a device-side commit dropped out-of-range addresses
        cudaMemsetAsync((int *)ctx->flags.p + 1, 0, sizeof(int), ctx->stream);
        return S2_ERANGE;
    }
    if ((ctx->flags_last & S2_WANT_NGB) && ctx->h_flags[0]) return S2_EOVERFLOW;
    return S2_OK;
}

extern "C" int s2_get_results(s2_ctx *ctx, int ni, double *acc, double *jerk, double *snap, double *pot, int *nn_id,
                              double *nn_r2, int *ngb_count)
{
    if (!ctx || ni < 0) return S2_EINVAL;
    if (!ctx->calc_done) return S2_ESTATE;
    if (ni > ctx->ni_last) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    const size_t bytes = (size_t)ni * REC * sizeof(double);
    int rc = S2_OK;
    if (!ctx->res_on_host) {
        CU(cudaEventSynchronize(ctx->ev_io));
        rc = pinned_reserve(ctx, &ctx->h_io, &ctx->h_io_bytes, 0, bytes);
        if (rc != S2_OK) return rc;
        if (ni) CU(cudaMemcpyAsync(ctx->h_io, ctx->result.p, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    }
    rc = fetch_flags(ctx);
    if (rc != S2_OK) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    CU(cudaGetLastError());
    const double *r0 = (const double *)(ctx->res_on_host ? ctx->h_res : ctx->h_io);   // small calls: written by the kernels
    const int order = ctx->order;
    par_ranges((size_t)ni, (size_t)16384, [=](size_t lo, size_t hi) {
    const double *r = r0 + lo * REC;
    for (size_t k = lo; k < hi; ++k, r += REC) {
        if (acc) { acc[3 * (size_t)k] = r[0]; acc[3 * (size_t)k + 1] = r[1]; acc[3 * (size_t)k + 2] = r[2]; }
        if (jerk) { jerk[3 * (size_t)k] = r[3]; jerk[3 * (size_t)k + 1] = r[4]; jerk[3 * (size_t)k + 2] = r[5]; }
        if (pot) pot[k] = r[6];
        if (nn_r2) nn_r2[k] = r[7];
        int packed[2];
        memcpy(packed, &r[8], sizeof packed);   // low word = nn id, high word = neighbour count
        if (nn_id) nn_id[k] = packed[0];
        if (ngb_count) ngb_count[k] = packed[1];
        if (snap && order == 6) { snap[3 * (size_t)k] = r[9]; snap[3 * (size_t)k + 1] = r[10]; snap[3 * (size_t)k + 2] = r[11]; }
    }
    });
    return post_sync_status(ctx);
}

extern "C" int s2_get_results_device(s2_ctx *ctx, int ni, double *d_acc, double *d_jerk, double *d_snap, double *d_pot,
                                     int *d_nn_id, double *d_nn_r2, int *d_ngb_count)
{
    if (!ctx || ni < 0) return S2_EINVAL;
    if (!ctx->calc_done) return S2_ESTATE;
    if (ni > ctx->ni_last) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    const double *rec = (const double *)(ctx->res_on_host ? ctx->h_res : ctx->result.p);
    CU(launch_unpack_records(rec, ni, ctx->order, d_acc, d_jerk, d_snap, d_pot, d_nn_id, d_nn_r2, d_ngb_count, ctx->stream));
    ctx->launches++;
    return S2_OK;
}

extern "C" int s2_get_neighbours(s2_ctx *ctx, int i, int cap, int *n_out, int *list)
{
    if (!ctx || !n_out || cap < 0 || (cap > 0 && !list)) return S2_EINVAL;
    if (!ctx->calc_done || !(ctx->flags_last & S2_WANT_NGB)) return S2_ESTATE;
    if (i < 0 || i >= ctx->ni_last) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    double rec8 = 0.0;
    if (!ctx->res_on_host)
        CU(cudaMemcpyAsync(&rec8, (double *)ctx->result.p + (size_t)i * REC + 8, sizeof(double), cudaMemcpyDeviceToHost,
                           ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    if (ctx->res_on_host) rec8 = ((const double *)ctx->h_res)[(size_t)i * REC + 8];
    int packed[2];
    memcpy(packed, &rec8, sizeof packed);
    const int have = std::min(packed[1], ctx->ngb_cap);
    const int n = std::min(have, cap);
    if (n > 0) {
        CU(cudaMemcpyAsync(list, (int *)ctx->list.p + (size_t)i * ctx->ngb_cap, (size_t)n * sizeof(int),
                           cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
    }
    *n_out = n;
    return packed[1] > ctx->ngb_cap ? S2_EOVERFLOW : S2_OK;
}

// Compacts the fixed-stride lists of the last force call into CSR form on the device (count -> scan -> fill) and
// caches the result until the next s2_calc_*.  One 8-byte read-back (the total) sits between scan and fill.
static int build_csr(s2_ctx *ctx)
{
    if (ctx->csr_valid) return S2_OK;
    const int ni = ctx->ni_last;
    const int nb = csr_blocks(ni);
    int rc = dev_reserve(ctx, ctx->csr_len, (size_t)ni * sizeof(int));
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->csr_bsum, (size_t)(nb + 1) * sizeof(long long));
    if (rc == S2_OK) rc = dev_reserve(ctx, ctx->csr_off, (size_t)(ni + 1) * sizeof(long long));
    if (rc != S2_OK) return rc;
    const double *rec = (const double *)(ctx->res_on_host ? ctx->h_res : ctx->result.p);   // pinned records are device-readable
    long long *bsum = (long long *)ctx->csr_bsum.p, *d_total = bsum + nb;
    long long *h_total = (long long *)(ctx->h_flags + 4);
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_csr[0], ctx->stream));
    CU(launch_csr_scan(rec, ni, ctx->ngb_cap, (int *)ctx->csr_len.p, bsum, d_total, (long long *)ctx->csr_off.p, ctx->stream));
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_csr[1], ctx->stream));
    ctx->launches += 3;
    CU(cudaMemcpyAsync(h_total, d_total, sizeof(long long), cudaMemcpyDeviceToHost, ctx->stream));
    rc = fetch_flags(ctx);
    if (rc != S2_OK) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    ctx->csr_total = *h_total;
    rc = dev_reserve(ctx, ctx->csr_list, (size_t)std::max<long long>(ctx->csr_total, 1) * sizeof(int));
    if (rc != S2_OK) return rc;
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_csr[2], ctx->stream));
    if (ctx->csr_total > 0) {
        CU(launch_csr_fill((const int *)ctx->list.p, (const int *)ctx->csr_len.p, (const long long *)ctx->csr_off.p, ni,
                           ctx->ngb_cap, (int *)ctx->csr_list.p, ctx->stream));
        ctx->launches++;
    }
    if (ctx->timing) CU(cudaEventRecord(ctx->ev_csr[3], ctx->stream));
    ctx->ran_csr = true;
    ctx->csr_valid = true;
    return S2_OK;
}

extern "C" int s2_get_neighbours_csr(s2_ctx *ctx, int ni, long long *offsets, int *list, long long list_cap)
{
    if (!ctx || ni < 0 || !offsets || list_cap < 0) return S2_EINVAL;
    if (!ctx->calc_done || !(ctx->flags_last & S2_WANT_NGB)) return S2_ESTATE;
    if (ni > ctx->ni_last) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    int rc = build_csr(ctx);
    if (rc != S2_OK) return rc;
    // offsets and (when the caller's list can hold every member) the compacted list in one go; a prefix request
    // (ni < n_i of the call) may need fewer members than csr_total, which offsets[ni] then says
    const size_t b_off = align16((size_t)(ni + 1) * sizeof(long long));
    const bool with_list = list && list_cap >= ctx->csr_total && ctx->csr_total > 0;
    CU(cudaEventSynchronize(ctx->ev_io));
    rc = pinned_reserve(ctx, &ctx->h_io, &ctx->h_io_bytes, 0, b_off + (with_list ? (size_t)ctx->csr_total * sizeof(int) : 0));
    if (rc != S2_OK) return rc;
    CU(cudaMemcpyAsync(ctx->h_io, ctx->csr_off.p, (size_t)(ni + 1) * sizeof(long long), cudaMemcpyDeviceToHost, ctx->stream));
    if (with_list)
        CU(cudaMemcpyAsync((char *)ctx->h_io + b_off, ctx->csr_list.p, (size_t)ctx->csr_total * sizeof(int), cudaMemcpyDeviceToHost,
                           ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    par_memcpy(offsets, ctx->h_io, (size_t)(ni + 1) * sizeof(long long));
    const long long tot = offsets[ni];
    if (tot > list_cap || (tot > 0 && !list)) return S2_ERANGE;
    if (tot > 0) {
        if (!with_list) {   // prefix request with a list shorter than the whole call's: copy just the prefix
            rc = pinned_reserve(ctx, &ctx->h_io, &ctx->h_io_bytes, 0, b_off + (size_t)tot * sizeof(int));
            if (rc != S2_OK) return rc;
            CU(cudaMemcpyAsync((char *)ctx->h_io + b_off, ctx->csr_list.p, (size_t)tot * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
            CU(cudaStreamSynchronize(ctx->stream));
        }
        par_memcpy(list, (const char *)ctx->h_io + b_off, (size_t)tot * sizeof(int));
    }
    return ctx->h_flags[0] ? S2_EOVERFLOW : S2_OK;
}

extern "C" int s2_get_neighbours_csr_device(s2_ctx *ctx, int ni, const long long **d_offsets, const int **d_list, long long *total)
{
    if (!ctx || ni < 0 || !d_offsets || !d_list || !total) return S2_EINVAL;
    if (!ctx->calc_done || !(ctx->flags_last & S2_WANT_NGB)) return S2_ESTATE;
    if (ni > ctx->ni_last) return S2_ERANGE;
    CU(cudaSetDevice(ctx->device));
    int rc = build_csr(ctx);
    if (rc != S2_OK) return rc;
    *d_offsets = (const long long *)ctx->csr_off.p;
    *d_list = (const int *)ctx->csr_list.p;
    *total = ctx->csr_total;
    if (ni < ctx->ni_last) {
        long long *h = (long long *)(ctx->h_flags + 4);
        CU(cudaMemcpyAsync(h, (const long long *)ctx->csr_off.p + ni, sizeof(long long), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        *total = *h;
    }
    return ctx->h_flags[0] ? S2_EOVERFLOW : S2_OK;
}

extern "C" int s2_get_csr_timing(s2_ctx *ctx, float *scan_ms, float *fill_ms)
{
    if (!ctx) return S2_EINVAL;
    if (!ctx->timing || !ctx->ran_csr) return S2_ESTATE;
    CU(cudaStreamSynchronize(ctx->stream));
    float a = 0.f, b = 0.f;
    CU(cudaEventElapsedTime(&a, ctx->ev_csr[0], ctx->ev_csr[1]));
    CU(cudaEventElapsedTime(&b, ctx->ev_csr[2], ctx->ev_csr[3]));
    if (scan_ms) *scan_ms = a;
    if (fill_ms) *fill_ms = b;
    return S2_OK;
}

// ---- hooks and diagnostics ----------------------------------------------------------------

extern "C" int s2_get_predicted_j(s2_ctx *ctx, int first, int n, double *pos, double *vel, double *acc)
{
    if (!ctx || n < 0 || first < 0) return S2_EINVAL;
    if (!ctx->predicted) return S2_ESTATE;
    if ((long long)first + n > ctx->nj_pred) return S2_ERANGE;
    if (n == 0) return S2_OK;
    CU(cudaSetDevice(ctx->device));
    const int np = nplanes(ctx->order);
    std::vector<double2> h((size_t)np * n);
    for (int p = 0; p < np; ++p)
        CU(cudaMemcpyAsync(h.data() + (size_t)p * n, plane(ctx, p) + first, (size_t)n * sizeof(double2),
                           cudaMemcpyDeviceToHost, ctx->stream));
    CU(cudaStreamSynchronize(ctx->stream));
    for (int k = 0; k < n; ++k) {
        if (pos) { pos[3 * (size_t)k] = h[k].x; pos[3 * (size_t)k + 1] = h[k].y; pos[3 * (size_t)k + 2] = h[(size_t)n + k].x; }
        if (vel) { vel[3 * (size_t)k] = h[(size_t)2 * n + k].x; vel[3 * (size_t)k + 1] = h[(size_t)2 * n + k].y; vel[3 * (size_t)k + 2] = h[(size_t)3 * n + k].x; }
        if (acc && np == 6) { acc[3 * (size_t)k] = h[(size_t)4 * n + k].x; acc[3 * (size_t)k + 1] = h[(size_t)4 * n + k].y; acc[3 * (size_t)k + 2] = h[(size_t)5 * n + k].x; }
    }
    return S2_OK;
}

extern "C" int s2_get_j(s2_ctx *ctx, int first, int n, int *id, double *t, double *mass, double *pos)
{
    if (!ctx || n < 0 || first < 0) return S2_EINVAL;
    if (!ctx->have_j) return S2_ESTATE;
    if ((long long)first + n > ctx->nj_cap) return S2_ERANGE;
    if (n == 0) return S2_OK;
    CU(cudaSetDevice(ctx->device));
    std::vector<double> h((size_t)5 * n);
    for (int f = 0; f < 5; ++f)
        CU(cudaMemcpyAsync(h.data() + (size_t)f * n, base_field(ctx, f) + first, (size_t)n * sizeof(double),
                           cudaMemcpyDeviceToHost, ctx->stream));
    if (id) CU(cudaMemcpyAsync(id, base_id(ctx) + first, (size_t)n * sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    int rc = fetch_flags(ctx);
    if (rc != S2_OK) return rc;
    CU(cudaStreamSynchronize(ctx->stream));
    for (int k = 0; k < n; ++k) {
        if (t) t[k] = h[k];
        if (mass) mass[k] = h[(size_t)n + k];
        if (pos) for (int c = 0; c < 3; ++c) pos[3 * (size_t)k + c] = h[(size_t)(2 + c) * n + k];
    }
    if (ctx->h_flags[1]) {
        cudaMemsetAsync((int *)ctx->flags.p + 1, 0, sizeof(int), ctx->stream);
        return S2_ERANGE;
    }
    return S2_OK;
}

extern "C" int s2_set_tuning(s2_ctx *ctx, int key, int value)
{
    if (!ctx || key < 0 || key > 10 || value < 0) return S2_EINVAL;
    ctx->tune[key] = value;
    return S2_OK;
}

extern "C" int s2_last_launch_info(const s2_ctx *ctx, int out[10])
{
    if (!ctx || !out) return S2_EINVAL;
    memcpy(out, ctx->last_info, sizeof ctx->last_info);
    return S2_OK;
}

extern "C" long long s2_kernel_launches(const s2_ctx *ctx) { return ctx ? ctx->launches : 0; }

extern "C" int s2_enable_timing(s2_ctx *ctx, int on)
{
    if (!ctx) return S2_EINVAL;
    ctx->timing = on != 0;
    ctx->ran_predict = ctx->ran_force = ctx->ran_reduce = false;
    return S2_OK;
}

extern "C" int s2_get_timing(s2_ctx *ctx, float *predict_ms, float *force_ms, float *reduce_ms)
{
    if (!ctx) return S2_EINVAL;
    if (!ctx->timing) return S2_ESTATE;
    CU(cudaStreamSynchronize(ctx->stream));
    float v[3] = {0.f, 0.f, 0.f};
    const bool ran[3] = {ctx->ran_predict, ctx->ran_force, ctx->ran_reduce};
    for (int k = 0; k < 3; ++k)
        if (ran[k]) CU(cudaEventElapsedTime(&v[k], ctx->ev_t[2 * k], ctx->ev_t[2 * k + 1]));
    if (predict_ms) *predict_ms = v[0];
    if (force_ms) *force_ms = v[1];
    if (reduce_ms) *reduce_ms = v[2];
    return S2_OK;
}

// Host wall time of one small force call as a C caller sees it: s2_calc_ilist + s2_get_results (which synchronises),
// `reps` times in a row, measured with the steady clock here so that no binding layer is in the loop.
extern "C" int s2_time_host_roundtrip(s2_ctx *ctx, int ni, const int *i_address, double eps2, unsigned flags, int reps,
                                      double *us_per_call)
{
    if (!ctx || !i_address || !us_per_call || ni <= 0 || reps <= 0 || (flags & S2_WANT_NGB)) return S2_EINVAL;
    std::vector<double> acc((size_t)ni * 3), jerk((size_t)ni * 3), snap((size_t)ni * 3), pot((size_t)ni), nn_r2((size_t)ni);
    std::vector<int> nn_id((size_t)ni);
    for (int k = 0; k < 3; ++k) {   // warm-up: shape cache, pinned buffers
        int rc = s2_calc_ilist(ctx, ni, i_address, nullptr, eps2, flags);
        if (rc != S2_OK) return rc;
        rc = s2_get_results(ctx, ni, acc.data(), jerk.data(), snap.data(), pot.data(), nn_id.data(), nn_r2.data(), nullptr);
        if (rc != S2_OK) return rc;
    }
    const auto t0 = std::chrono::steady_clock::now();
    for (int k = 0; k < reps; ++k) {
        int rc = s2_calc_ilist(ctx, ni, i_address, nullptr, eps2, flags);
        if (rc != S2_OK) return rc;
        rc = s2_get_results(ctx, ni, acc.data(), jerk.data(), snap.data(), pot.data(), nn_id.data(), nn_r2.data(), nullptr);
        if (rc != S2_OK) return rc;
    }
    const auto t1 = std::chrono::steady_clock::now();
    *us_per_call = std::chrono::duration<double, std::micro>(t1 - t0).count() / reps;
    return S2_OK;
}

extern "C" int s2_fp32_fixup_count(s2_ctx *ctx, int *n)
{
    if (!ctx || !n) return S2_EINVAL;
    *n = 0;
    if (!ctx->calc_done) return S2_ESTATE;
    if (ctx->precision != S2_FP32 || !ctx->fix.p || ctx->order == 2) return S2_OK;
    if (ctx->fix_last < 0) {
        CU(cudaMemcpyAsync(ctx->h_flags + 3, ctx->fix.p, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
        CU(cudaStreamSynchronize(ctx->stream));
        ctx->fix_last = ctx->h_flags[3];
    }
    *n = ctx->fix_last;
    return S2_OK;
}

extern "C" int s2_peak_fma(s2_ctx *ctx, int kind, int iters, double *fma_per_s)
{
    if (!ctx || !fma_per_s || iters <= 0 || kind < 0 || kind > 8) return S2_EINVAL;
    CU(cudaSetDevice(ctx->device));
    CU(run_peak_fma(kind, iters, ctx->sm_count, ctx->stream, fma_per_s));
    ctx->launches += 2;
    return S2_OK;
}

extern "C" int s2_hop_latency(s2_ctx *ctx, int ctas, int iters, double *cycles_per_round_trip)
{
    if (!ctx || !cycles_per_round_trip || iters <= 0 || ctas < 2 || ctas > ctx->sm_count) return S2_EINVAL;   // co-resident: one CTA per SM at most
    CU(cudaSetDevice(ctx->device));
    Buf tmp;
    const size_t bytes = (size_t)(ctas + 2) * 128;
    int rc = dev_reserve(ctx, tmp, bytes);
    if (rc != S2_OK) return rc;
    long long h = 0;
    cudaError_t e = cudaMemsetAsync(tmp.p, 0, bytes, ctx->stream);
    if (e == cudaSuccess) e = run_hop_latency(ctas, iters, (unsigned long long *)tmp.p + 16, (long long *)tmp.p, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(&h, tmp.p, sizeof h, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    ctx->launches++;
    dev_release(ctx, tmp);
    if (e != cudaSuccess) return fail_cuda(ctx, e);
    *cycles_per_round_trip = (double)h / iters;
    return S2_OK;
}

extern "C" int s2_test_ds_ops(s2_ctx *ctx, int n, const double *a, const double *b, double *out)
{
    if (!ctx || n < 0 || (n > 0 && (!a || !b || !out))) return S2_EINVAL;
    if (n == 0) return S2_OK;
    CU(cudaSetDevice(ctx->device));
    Buf tmp;
    const size_t bytes = (size_t)n * sizeof(double);
    int rc = dev_reserve(ctx, tmp, 10 * bytes);
    if (rc != S2_OK) return rc;
    double *d_a = (double *)tmp.p, *d_b = d_a + n, *d_out = d_b + n;
    cudaError_t e = cudaMemcpyAsync(d_a, a, bytes, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(d_b, b, bytes, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = run_ds_ops(n, d_a, d_b, d_out, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out, d_out, 8 * bytes, cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    ctx->launches++;
    dev_release(ctx, tmp);
    if (e != cudaSuccess) return fail_cuda(ctx, e);
    return S2_OK;
}

extern "C" const char *s2_strerror(int code)
{
    switch (code) {
    case S2_OK: return "ok";
    case S2_EINVAL: return "invalid argument";
    case S2_ERANGE: return "address or count out of range";
    case S2_ENOMEM: return "out of device or pinned memory";
    case S2_ECUDA: return "CUDA error or no CUDA device (there is no CPU fallback)";
    case S2_ESTATE: return "call order violated (commit -> predict -> calc -> get)";
    case S2_EOVERFLOW: return "a neighbour list exceeded ngb_cap (results valid, lists truncated)";
    }
    return "unknown error code";
}

extern "C" const char *s2_last_cuda_error(const s2_ctx *ctx) { return ctx ? ctx->cuda_err.c_str() : ""; }

extern "C" const char *s2_version(void) { return "s2b200 0.1 (sm_100a)"; }
