// s2_internal.h -- shared declarations of the CUDA library behind include/s2b200.h.
// Not part of the ABI.  Nothing here is shared with oracle/.
#pragma once

#include <cuda_runtime.h>
#include <stdint.h>

#include <vector>

#include "../../include/s2b200.h"

namespace s2 {

// ---- data layout in HBM ----------------------------------------
//
// Base j-store (fp64 SoA, one array per scalar field, capacity nj_cap each):
//   field 0 t_j, 1 m, 2-4 x, 5-7 v, 8-10 a, 11-13 jerk, [14-16 snap, 17-19 crackle], + int id[]
// Predicted j-store, fp64 "planes" of 16-byte elements (one element per particle per plane):
//   P0 (x, y)   P1 (z, m)   P2 (vx, vy)   P3 (vz, id bits)   [6th order: P4 (ax, ay)  P5 (az, 0)]
// fp32 planes (float4 per particle):
//   F0 (x_hi, y_hi, z_hi, m)   F1 (x_lo, y_lo, z_lo, id bits)   F2 (vx, vy, vz, 0)   [F3 (ax, ay, az, 0)]
// double-single planes (float4 per particle, value = hi + lo):
//   D0 (x_hi, x_lo, y_hi, y_lo)  D1 (z_hi, z_lo, m_hi, m_lo)  D2 (vx_hi, vx_lo, vy_hi, vy_lo)
//   D3 (vz_hi, vz_lo, id bits, 0)   [D4 (ax_hi, ax_lo, ay_hi, ay_lo)  D5 (az_hi, az_lo, 0, 0)]
// Result / partial record: REC doubles per (slice, i):
//   0-2 acc, 3-5 jerk, 6 pot, 7 nn_d2, 8 {int nn (address in partials, id in finals), int ngb_count},
//   9-11 snap (6th order)

constexpr int kMaxFields = 20;
constexpr int kMaxPlanes = 8;      // up to 6 arithmetic planes + 2 fp64 position planes for decisions
constexpr int REC = 12;            // doubles per result record (96 B = three 32-byte sectors)
constexpr int kThreads = 256;   // threads per force CTA
constexpr int kWarps = kThreads / 32;
// i-particles per thread of the register-tiled full-occupancy sweep (force_sweep_tiled_kernel); 1 = not built
constexpr int kIptF64 = 2, kIptF32 = 2, kIptDS = 1;
inline int force_ipt(int precision) { return precision == S2_FP64 ? kIptF64 : (precision == S2_FP32 ? kIptF32 : kIptDS); }

// a 2nd-order context (acc + pot only) stores and predicts like a 4th-order one (missing derivatives are zero);
// only the force sweep differs (fewer planes staged, no jerk terms)
inline int nfields(int order) { return order == 6 ? 20 : 14; }
inline int nplanes(int order) { return order == 6 ? 6 : 4; }

struct PredictArgs {
    const double *f[kMaxFields];   // base fields
    const int *id;
    double2 *p[kMaxPlanes];        // fp64 planes (always written)
    float4 *q[kMaxPlanes];         // precision-specific planes or nullptr
    double t;
    const double *t_dev;           // when non-null the prediction time is read from device memory (block-step integrator)
    int pdl;                       // launch with programmatic stream serialisation (the kernel waits for its predecessor itself)
    int nj;
    int order;
    int precision;
};

struct ScatterArgs {
    const int *address;
    const int *id;
    const double *src[kMaxFields]; // scalar fields (t, m) have stride 1; vector fields are (n,3) row-major
    double *dst[kMaxFields];
    int *dst_id;
    int n;
    int nfields;
    int nj_cap;
    int *erange_flag;
};

struct ForceArgs {
    const void *jp[kMaxPlanes];    // j planes staged per tile: the pair-arithmetic planes, then (non-fp64
                                   // modes with NN/NGB) the fp64 position planes P0, P1 for the decisions
    const void *ip[kMaxPlanes];    // same list for the i side (== jp in address mode)
    const int *i_addr;             // nullptr: i-th i-particle lives at index i of ip
    const double *h2;              // per i, or nullptr
    const double2 *jid_plane;      // fp64 plane P3 of j (id lookup for final nn)
    int ni;
    int nj;                        // number of j-particles summed over ...
    int j_first;                   // ... starting at this address of the predicted store
    double eps2;
    int S;                         // CTA slices over j
    int slice_len;                 // j per CTA slice
    int Wj;                        // warp columns over j inside a CTA (1,2,4,8)
    int tile;                      // j per shared-memory tile
    int stages;                    // tile buffers in the ring (2..kMaxStages)
    int nslices_total;             // S * Wj
    int is_final;                  // 1: write final records (nn as id), no reduce kernel follows
    double *rec;                   // [nslices_total][ni][REC]
    int *seg;                      // [ni][nslices_total][segcap] neighbour segments
    int segcap;
    int *overflow_flag;
    int ngb_cap;
    // fused combine (no neighbour lists): the warp columns of a CTA are summed in shared memory, so there is one
    // partial row per j-slice, and the last CTA of an i-group to finish reduces the S rows in a fixed order
    int fused;
    int cluster;                   // CTAs per cluster along the slice axis (1, 2, 4, 8); > 1 only when fused
    unsigned *counters;            // [number of i-groups], zero between calls (the reducing CTA resets its entry)
    double *out_final;             // [ni][REC]
    int order;
    // fp32 path, reading R-F32 (s2_api.cu fp32_fixup): the sweep leaves sum_j q_j^2 per (slice, i) so that particles whose
    // jerk is a strongly cancelling sum can be found and re-evaluated in fp64
    float *wq;                     // [nslices_total][ni], or nullptr
    int *fix_count;                // number of flagged i-particles: the sweep zeroes it (saves a memset node per call)
    // fp32 fix-up (fp32_fix_sweep_kernel, s2_force_fp64.cu): the flagged i-particles, as positions in the i-list, their
    // number (device memory: known only after the flag kernel ran), and the partial rows [S][ni][NC] of their j-slices
    const int *pos_list;
    const int *ni_dev;
    double *fix_part;              // [S][fix_kcap][NC]
    int fix_kcap;                  // flagged particles the partial rows have room for (even); the rest is swept unsliced
    unsigned *fix_arrive;          // [ceil(ni / 2)] arrival counters of the fix-up groups, zero between calls
    int atomic;                    // 1: j-slices add their sums to the zeroed final records with fp64 atomics (opt-in,
                                   // the paper's Sapporo2 combine L88; not bit-reproducible; no NN / neighbour lists)
    // uniform-operand sweep (force_sweep_bank_kernel): the chunk of j now in the constant bank
    int bank_j0, bank_cnt;         // address of its first particle, number of particles
    int bank_first, bank_last;     // first chunk: start from zero; last chunk: write final records to rec
    double *bank_state;            // [REC][ni] running sums and decisions between chunk launches (SoA)
    int bank_id;                   // which of the two constant banks (modules) this launch reads
    unsigned *bank_flags;          // device words {ready[2], -, -, arrived[2]} of the bank hand-over, or nullptr for the
                                   // launch that only parks the i-particles
    unsigned bank_ticket;          // sequence number of this chunk: ready[bank] >= ticket when the chunk is in its bank
    int bank_spin;                 // 0 for the first two chunks (copied by the host before the first launch)
    int bank_next_known;           // 1: the next chunk is known to be in its bank (first chunks) or there is none
    double2 *bank_self;            // this launch's bank through its address in global memory (refill target)
    int bank_next_j0, bank_next_cnt;   // the chunk after next, which the last CTA copies into this bank (cnt 0: none)
    int bank_pdl;                  // launch with programmatic stream serialisation (overlaps the previous chunk's tail)
    int bank_wait_early;           // wait for the previous launch before anything is read (decisions carried, chunk 0)
    int bank_threads;              // threads per CTA of the chunk launches (128 or 256; 0: the policy's default)
};

// ---- block-time-step integrator (s2_bts.cu): state handed to its kernels ----------------------------------------
constexpr int kBtsLog = 1024;        // block steps one launch of the small-step kernel may run (entries of its pinned log)
struct BtsCtl {                      // device control block (mirrored to pinned host memory by the kernels that change it)
    double t_next;                   // time of the block step that is about to run
    int n_next;                      // number of active particles of that step
    int error;                       // != 0: a wait inside the small-step kernel timed out (the state is then undefined)
    long long steps;                 // block steps the small-step kernel has run since s2_bts_init
    double t_done;                   // time of the last block step it completed
    long long tag;                   // last sequence tag the small-step kernel used in its exchange buffers
};

struct BtsArgs {
    double *f[kMaxFields];           // base j-store fields (t, m, x, v, a, jerk [, snap, crackle])
    double *dt;                      // [n] current step of every particle
    double *pot;                     // [n] potential at the particle's last force evaluation
    const double *rec;               // result records of the force call on the active list
    int *ilist;                      // active list (addresses, ascending)
    int *stage;                      // [n] per-block compaction staging of the select kernel
    int *bcnt;                       // [nblocks] active particles found by each block
    unsigned *arrive;                // arrival counter of the select kernel (zero between launches)
    int *hist;                       // [kLevels] particles per step level
    BtsCtl *ctl;                     // device control block
    BtsCtl *h_ctl;                   // the same, in pinned host memory
    int n, n_act, order;
    double eta, eta_start, dt_max, dt_min;
    double eta4;                     // 6th order, averaged criterion: eta of the 4th-order Aarseth step it is averaged with
    int averaged;
    // small-step kernel (bts_small_steps_kernel, s2_force_fp64.cu): runs block steps of at most spec_cap active particles
    // that lie at or before t_end, at most max_steps of them, and logs each step's active count to pinned h_log
    int spec_cap, max_steps;
    double t_end;
    int *h_log;                      // pinned, kBtsLog entries
    // exchange buffers of that kernel, 64-bit words {32 bits of payload, 32-bit sequence tag}: a reader polls the words it
    // needs until they carry the tag of the step, so the data is its own flag (no fence, no counter)
    unsigned long long *xrows;       // partial sums [CTA][spec_cap][7 | 10][2 words]
    unsigned long long *xrec;        // the active particles of the coming step, by owner: [address of first own + q][14 | 20 words]
    unsigned long long *xhdr;        // [reader CTA][owner CTA] {number of the owner's active particles}: one copy per reader
    unsigned *bar;                   // bar[0] grid-barrier counter, bar[1] exit counter; both 0 between launches
    long long *prof;                 // null, or 10 sums: SM cycles CTA prof_cta spent in each part of a step (s2b200_test.h), steps
    int prof_cta;
};

// fp32 path, reading R-F32: what is needed to decide whether an i-particle's jerk is a strongly cancelling sum
struct F32Flag {
    const float *wq;               // [nst][ni] sum of q^2 per (slice, i), or nullptr: no flagging
    int nst;
    const double2 *v2, *v3;        // fp64 planes P2 (vx, vy), P3 (vz, id) of the i side
    const int *i_addr;             // nullptr: i-th i-particle lives at index i of the planes
    double thresh;
    int *pos_list;                 // out: positions (in the i-list) of the flagged particles, any order
    int *count;                    // out: their number
};

struct ReduceArgs {
    const double *part;            // [nslices_total][ni][REC]
    double *out;                   // [ni][REC]
    const int *seg;                // [ni][nslices_total][segcap]
    int *list;                     // [ni][ngb_cap]
    const double2 *jid_plane;      // P3 of j
    int ni;
    int nslices_total;
    int segcap;
    int ngb_cap;
    int order;
    unsigned flags;
    int *overflow_flag;
    F32Flag f32;                   // fp32 contexts: flag ill-conditioned jerk sums while the final sums are at hand (wq != nullptr)
    int has_bts;                   // block-step integrator: lane 0 applies the corrector to its particle right after the combine
    BtsArgs bts;
};

// kernels' host-side launchers (each returns the cudaError_t of the launch)
cudaError_t launch_scatter(const ScatterArgs &a, cudaStream_t st);
cudaError_t launch_predict(const PredictArgs &a, cudaStream_t st);
cudaError_t launch_reduce(const ReduceArgs &a, cudaStream_t st);
bool reduce_by_warp_kernel(const ReduceArgs &a);   // true: launch_reduce takes reduce_kernel (one warp per i), which flags inline

struct ForceShape {                // chosen by the balancer in s2_api.cu
    int L;                         // lanes per i (1..32); 0: register-tiled sweep (several i per thread)
    int TL;                        // register-tiled sweep: lanes per i-slot (1..32)
    int Wj;                        // warp columns
    int S;
    int slice_len;
    int tile;
    int stages;
    int fused;                     // combine inside the sweep launch (last CTA of each i-group)
    int cluster;                   // CTAs per cluster along the slice axis when fused (1 = no cluster)
};
constexpr int kSmemHeader = 64;   // mbarriers live in the first 64 bytes of dynamic shared memory
constexpr int kMaxStages = 8;
inline size_t force_smem_bytes(int nplanes, int tile, int stages)
{
    return (size_t)kSmemHeader + (size_t)stages * nplanes * tile * 16;
}

cudaError_t run_peak_fma(int kind, int iters, int sm_count, cudaStream_t st, double *fma_per_s);
cudaError_t run_hop_latency(int ctas, int iters, unsigned long long *buf, long long *d_cycles, cudaStream_t st);

}  // namespace s2
