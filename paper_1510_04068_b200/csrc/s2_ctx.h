// s2_ctx.h -- the context behind the opaque s2_ctx of include/s2b200.h, shared by the translation units that
// implement the ABI (s2_api.cu: the GRAPE-style calls; s2_bts.cu: the device-resident block-time-step integrator).
// Not part of the ABI.
#pragma once

#include <map>
#include <string>
#include <vector>

#include "s2_internal.h"

using namespace s2;   // private header of the library's own translation units

struct Buf {
    void *p = nullptr;
    size_t bytes = 0;
};

struct Batch {
    size_t offset;   // byte offset of the batch block in the staging buffer
    int n;
};

struct s2_ctx {
    int device = 0, order = 4, precision = S2_FP64, nj_cap = 0, ngb_cap = 0;
    s2_allocator alloc{};
    bool has_alloc = false;
    cudaStream_t stream = nullptr;
    int sm_count = 148;
    std::string cuda_err;
    long long launches = 0;

    // device buffers
    Buf base, planes, qplanes, stage_dev, iplanes, iqplanes, i_addr, i_h2, part, result, seg, list, flags, counters;
    // device-side CSR of the neighbour lists of the last force call (built on first request, s2_ngb.cu)
    Buf csr_len, csr_bsum, csr_off, csr_list;
    Buf fixarr;                       // fp32 fix-up: arrival counters of the groups (zero between calls)
    Buf fixpart;                      // fp32 fix-up: partial rows [S][ni][7|10] of the flagged particles' j-slices
    Buf wq, fix;                       // fp32 fix-up (R-F32): sum of q^2 per (slice, i); {count, flagged positions}
    int fix_last = -1;                // flagged i-particles of the last fp32 call once read back (-1: not read)
    bool csr_valid = false;
    long long csr_total = 0;
    cudaEvent_t ev_csr[4] = {nullptr, nullptr, nullptr, nullptr};
    bool ran_csr = false;
    // pinned host buffers
    void *h_stage = nullptr;
    size_t h_stage_bytes = 0, h_stage_used = 0;
    void *h_io = nullptr;
    size_t h_io_bytes = 0;
    int *h_flags = nullptr;           // pinned, 4 ints
    // zero-copy small calls (n_i <= kZeroCopyNi): the kernels read the i-list from, and write the final records to,
    // pinned host memory directly (device-accessible under unified addressing) -- no copy operations on the stream
    void *h_res = nullptr;            // final records of the last small call
    size_t h_res_bytes = 0;
    bool res_on_host = false;
    void *h_il[2] = {nullptr, nullptr};   // i-list (+ h2) of small calls, alternating so that a call can be
    size_t h_il_bytes[2] = {0, 0};        // prepared while the previous one still runs
    cudaEvent_t ev_il[2] = {nullptr, nullptr};
    int il_turn = 0;
    bool flags_dirty = false;         // a device-side commit may have raised the range flag
    const BtsArgs *bts_hook = nullptr;   // set by s2_bts_run around run_force: corrector to apply inside reduce_kernel
    bool bts_hook_done = false;       // run_force took the hook (the force call went through reduce_kernel)
    bool in_selftest = false;         // inside bank_selftest (run_force re-entered with a reduced problem)
    cudaEvent_t ev_stage = nullptr;   // H2D of the staging buffer finished
    cudaEvent_t ev_io = nullptr;      // H2D of the i-list upload finished
    std::vector<Batch> batches;

    // state
    bool have_j = false, predicted = false, calc_done = false, results_fetched = false;
    int nj_pred = 0, ni_last = 0;
    int j_first = 0, j_count = 0;     // j-range of the force sums (s2_set_j_range); count 0 = every predicted particle
    unsigned flags_last = 0;
    double t_pred = 0.0;

    // tuning overrides and last launch
    int tune[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    int last_info[10] = {0, 0, 0, 0, 0, 0, 0, 0, 1, 1};
    std::map<long long, int> occ_cache;
    std::map<long long, std::pair<ForceShape, int>> shape_cache;

    // timing
    bool timing = false;
    cudaEvent_t ev_t[6] = {nullptr, nullptr, nullptr, nullptr, nullptr, nullptr};
    bool ran_predict = false, ran_force = false, ran_reduce = false;
};


// where the arrays of the j-store live inside the context's buffers
static inline double *base_field(const s2_ctx *c, int f) { return (double *)c->base.p + (size_t)f * c->nj_cap; }
static inline int *base_id(const s2_ctx *c) { return (int *)((double *)c->base.p + (size_t)s2::nfields(c->order) * c->nj_cap); }
static inline double2 *plane(const s2_ctx *c, int p) { return (double2 *)c->planes.p + (size_t)p * c->nj_cap; }
static inline float4 *qplane(const s2_ctx *c, int p) { return (float4 *)c->qplanes.p + (size_t)p * c->nj_cap; }
static inline int n_qplanes(int precision, int order)
{
    if (precision == S2_FP32) return order == 6 ? 4 : 3;
    if (precision == S2_DS) return order == 6 ? 6 : 4;
    return 0;
}

int fail_cuda(s2_ctx *c, cudaError_t e);
#define CU(call)                                           \
    do {                                                   \
        cudaError_t e__ = (call);                          \
        if (e__ != cudaSuccess) return fail_cuda(ctx, e__); \
    } while (0)

// device buffers grow on demand through the context's allocator (contents are not preserved)
int dev_reserve(s2_ctx *ctx, Buf &b, size_t bytes);
void dev_release(s2_ctx *ctx, Buf &b);
int pinned_reserve(s2_ctx *ctx, void **p, size_t *have, size_t used, size_t bytes);
// a3-a8 on an i-list that already lives where the kernels can read it (s2_api.cu)
int run_force(s2_ctx *ctx, int ni, const int *d_i_addr, const double *d_h2, bool explicit_i, double eps2, unsigned flags,
              bool host_call);
