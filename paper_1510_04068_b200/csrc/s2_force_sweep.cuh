// s2_force_sweep.cuh -- the i x j force sweep (a3-a5, a7, a8), generic over a precision policy.
//
// PAPER.md sec 2.1 (L46-L54): sinks (i) x sources (j); "parallelisation over the sink particles"
// when there are many sinks, Sapporo1's "parallelize over the source particles ... split into
// subsets" when there are few, and sec 3.1 (L104) "2D thread-blocks ... multiple threads per
// i-particle whereby each thread computes a part of the j-particles".  Two kernel templates cover
// the whole range:
//   force_sweep_tiled_kernel<P, IPT>  full-occupancy path: one lane per i, IPT i-particles per thread,
//                                     so every j read from shared memory feeds IPT pair evaluations;
//   force_sweep_kernel<P, L>          j-split path: L lanes share one i-particle and take interleaved j
//                                     (L = 1: plain one lane per i); when the i-list cannot fill a CTA the
//                                     8 warps also become warp columns (Wj) that split every tile.
// Common to both:
//   - a CTA owns a group of i-particles (blockIdx.x) and a contiguous j-slice (blockIdx.y);
//   - j tiles are staged global -> shared with 1-D bulk async copies (TMA, cp.async.bulk) that complete on
//     an mbarrier, in a ring of up to 4 buffers (TilePipe);
//   - i-particles and accumulators live in registers; per-tile partial sums are added to running totals;
//     each (slice, i) writes one 96-byte record;
//   - slices are combined in a fixed order, never by floating-point atomics: by reduce_kernel
//     (s2_reduce.cu, launched with programmatic dependent launch) or, for small i-groups, by the last CTA
//     of the i-group inside the sweep launch (fused), optionally after a cluster / DSMEM pre-combine;
//   - nearest-neighbour and neighbour decisions sit behind one exact compare (Dec::thr); hits are appended in
//     ascending j order: per thread for L = 1, by warp ballot + population-count prefix for L > 1.
#pragma once

#include <math_constants.h>

#include <atomic>

#include "s2_force_common.cuh"

namespace s2 {

// decision state: nearest neighbour (squared distance, j address) and neighbour count, plus the rejection
// threshold of the one-lane-per-i paths: a pair can only change a decision if d2 < thr = max(h2, nn_d2), which is
// rare (a few dozen neighbours and ~ln N nearest-neighbour updates per i), so everything else sits behind one compare
struct Dec {
    double nn_d2;
    double thr;    // max(h2 if neighbour lists are wanted, nn_d2 if the nearest neighbour is wanted)
    float thrf;    // thr rounded up with a 2^-10 guard band: prefilter on an fp32 estimate of d2 (fp32 / DS sweeps)
    int nn_j;
    int cnt;

    template <bool NN, bool NGB>
    __device__ __forceinline__ void set_thr(double h2)
    {
        thr = NN ? (NGB ? fmax(h2, nn_d2) : nn_d2) : h2;
        thrf = __double2float_ru(thr) * 1.0009765625f;
    }
    template <bool NN, bool NGB>
    __device__ __forceinline__ void init(double h2)
    {
        nn_d2 = CUDART_INF;
        nn_j = -1;
        cnt = 0;
        set_thr<NN, NGB>(h2);
    }
};

// d2: unsoftened squared distance in fp64 (reading R-D2); skip: self or padding lane.
template <int L, bool NN, bool NGB>
__device__ __forceinline__ void decide(double d2, int jaddr, bool skip, double h2, Dec &D,
                                       const Decomp &d, int *seg, int segcap)
{
    if (L == 1) {
        if (!(d2 < D.thr)) return;   // exact: no decision below can fire when d2 >= max(h2, nn_d2)
    }
    const double d2m = skip ? CUDART_INF : d2;
    if (NN) {
        if (d2m < D.nn_d2) {   // strict: the first (lowest-address) minimum of this lane is kept
            D.nn_d2 = d2m;
            D.nn_j = jaddr;
            if (L == 1) D.template set_thr<NN, NGB>(h2);
        }
    }
    if (NGB) {
        const bool hit = d2m < h2;
        if (L == 1) {
            if (hit) {
                if (D.cnt < segcap && d.i_valid) seg[D.cnt] = jaddr;
                D.cnt++;
            }
        } else {
            const unsigned b = __ballot_sync(0xffffffffu, hit);
            if (b) {   // warp-uniform
                const unsigned g = (L == 32) ? b : ((b >> (d.il * L)) & ((1u << L) - 1u));
                const int pos = D.cnt + __popc(g & ((1u << d.jl) - 1u));
                if (hit && pos < segcap && d.i_valid) seg[pos] = jaddr;
                D.cnt += __popc(g);
            }
        }
    }
}

// Opt-in combine by atomics (sec 2.2.4: Sapporo2 "uses atomic operations" instead of a second kernel):
// every (slice, i) record is added to the zeroed final record.  The order of the additions is whatever the
// hardware makes it, so the last bits differ run to run (L84, L164) -- which is why it is not the default.
__device__ __forceinline__ void atomic_add_record(double *r, const double out[10], int order, bool first_slice)
{
#pragma unroll
    for (int c = 0; c < 7; ++c) atomicAdd(r + c, out[c]);
    if (order == 6) {
#pragma unroll
        for (int c = 0; c < 3; ++c) atomicAdd(r + 9 + c, out[7 + c]);
    }
    if (first_slice) {   // decisions are not computed on this path: "none"
        r[7] = CUDART_INF;
        r[8] = __hiloint2double(0, -1);
    }
}

// Sum of the partial rows of one i-particle by one warp, in a fixed order (P17): lane l adds rows l, l+32, ...
// sequentially, then the 32 lanes combine by an xor-butterfly; nn by (d2, address) lexicographic minimum.
// Rows were written by other CTAs of the same launch: read through L2 (ld.global.cg), after a fence.
template <bool NN>
__device__ __forceinline__ void reduce_rows_warp(const double *part, double *outp, const double2 *jid_plane, int i,
                                                 int ni, int rows, int order, int lane)
{
    double v[10];
#pragma unroll
    for (int c = 0; c < 10; ++c) v[c] = 0.0;
    double nn_d2 = CUDART_INF;
    int nn_j = -1;
    // rows are fetched four at a time (independent loads in flight) and added in row order
    for (int s0 = lane; s0 < rows; s0 += 4 * 32) {
        double2 q[4][6];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int s = s0 + 32 * u;
            if (s < rows) {
                const double2 *r = reinterpret_cast<const double2 *>(part + ((size_t)s * ni + i) * REC);
#pragma unroll
                for (int c = 0; c < 5; ++c) q[u][c] = __ldcg(r + c);
                if (order == 6) q[u][5] = __ldcg(r + 5);
            }
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            if (s0 + 32 * u < rows) {
                v[0] += q[u][0].x; v[1] += q[u][0].y; v[2] += q[u][1].x; v[3] += q[u][1].y;
                v[4] += q[u][2].x; v[5] += q[u][2].y; v[6] += q[u][3].x;
                if (order == 6) { v[7] += q[u][4].y; v[8] += q[u][5].x; v[9] += q[u][5].y; }
                if (NN) {
                    const int j = __double2loint(q[u][4].x);
                    if (q[u][3].y < nn_d2 || (q[u][3].y == nn_d2 && (unsigned)j < (unsigned)nn_j)) {
                        nn_d2 = q[u][3].y;
                        nn_j = j;
                    }
                }
            }
        }
    }
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
#pragma unroll
        for (int c = 0; c < 10; ++c) v[c] += shfl_xor_d(v[c], m);
        if (NN) {
            const double od2 = shfl_xor_d(nn_d2, m);
            const int oj = __shfl_xor_sync(0xffffffffu, nn_j, m);
            if (od2 < nn_d2 || (od2 == nn_d2 && (unsigned)oj < (unsigned)nn_j)) {
                nn_d2 = od2;
                nn_j = oj;
            }
        }
    }
    if (lane == 0) {
        int nn = nn_j;
        if (NN && nn >= 0) nn = __double2loint(jid_plane[nn].y);
        double2 *o = reinterpret_cast<double2 *>(outp + (size_t)i * REC);
        o[0] = make_double2(v[0], v[1]);
        o[1] = make_double2(v[2], v[3]);
        o[2] = make_double2(v[4], v[5]);
        o[3] = make_double2(v[6], nn_d2);
        o[4] = make_double2(__hiloint2double(0, nn), v[7]);
        o[5] = make_double2(v[8], v[9]);
    }
}

// fp32 path, reading R-F32: is the jerk of i-particle i a strongly cancelling sum?  Each fp32 pair term is good to
// ~4e-7, so the error of the sum is ~4e-7 sqrt(sum_j |t_j|^2), and sqrt(sum_j |t_j|^2) ~ sqrt(sum_j q_j^2) V with
// V = |v_i| + sqrt(2 |pot_i|) (own speed + local escape speed bound the relative speeds that matter).  Called by a whole
// warp that has just written the final record of i (lane 0); the rows of sum q^2 are added lane-parallel in a fixed order.
__device__ __forceinline__ void fp32_flag_warp(const F32Flag &f, const double *rec, int i, int ni, int lane)
{
    double w = 0.0;
    for (int s = lane; s < f.nst; s += 32) w += (double)f.wq[(size_t)s * ni + i];
#pragma unroll
    for (int m = 1; m < 32; m <<= 1) w += shfl_xor_d(w, m);
    if (lane == 0) {
        const double *r = rec + (size_t)i * REC;
        const double J = sqrt(r[3] * r[3] + r[4] * r[4] + r[5] * r[5]);
        const int ia = f.i_addr ? f.i_addr[i] : i;
        const double2 a = f.v2[ia], b = f.v3[ia];
        const double V = sqrt(a.x * a.x + a.y * a.y + b.x * b.x) + sqrt(2.0 * fabs(r[6]));
        if (sqrt(w) * V > f.thresh * J) f.pos_list[atomicAdd(f.count, 1)] = i;
    }
}

// Ring of ST shared-memory tile buffers filled by 1-D bulk copies (one per plane) that complete on an mbarrier.
// Thread 0 issues; everybody waits on the barrier of the tile it is about to read.
template <int NPL>
struct TilePipe {
    uint64_t *full;
    unsigned char *tiles;
    const ForceArgs *a;
    int ST, tile, j0, j1, ntiles;
    size_t stage_bytes;

    __device__ __forceinline__ void init(unsigned char *smem_raw, const ForceArgs &args)
    {
        a = &args;
        full = reinterpret_cast<uint64_t *>(smem_raw);
        tiles = smem_raw + kSmemHeader;
        ST = args.stages;
        tile = args.tile;
        stage_bytes = (size_t)NPL * tile * 16;
        j0 = args.j_first + blockIdx.y * args.slice_len;
        j1 = min(args.j_first + args.nj, j0 + args.slice_len);
        ntiles = j1 > j0 ? (j1 - j0 + tile - 1) / tile : 0;
        if (threadIdx.x == 0) {
            for (int s = 0; s < ST; ++s) mbar_init(&full[s], 1);
            mbar_fence_init();
        }
        __syncthreads();
        if (threadIdx.x == 0)
            for (int t = 0; t < min(ntiles, ST - 1); ++t) issue(t);   // prologue: ST-1 tiles in flight
    }
    __device__ __forceinline__ void issue(int t) const
    {
        const int st = t % ST;
        const int jt = j0 + t * tile;
        const uint32_t bytes = (uint32_t)min(tile, j1 - jt) * 16u;
        mbar_arrive_expect_tx(&full[st], bytes * NPL);
#pragma unroll
        for (int p = 0; p < NPL; ++p)
            bulk_g2s(tiles + st * stage_bytes + (size_t)p * tile * 16,
                     reinterpret_cast<const unsigned char *>(a->jp[p]) + (size_t)jt * 16, bytes, &full[st]);
    }
    // start of tile t: refill the stage released by the barrier that ended tile t-1, then wait for tile t
    __device__ __forceinline__ const unsigned char *acquire(int t) const
    {
        if (threadIdx.x == 0 && t + ST - 1 < ntiles) issue(t + ST - 1);
        mbar_wait(&full[t % ST], (t / ST) & 1);
        return tiles + (t % ST) * stage_bytes;
    }
    // end of tile t: a barrier is only needed when this stage will be refilled
    __device__ __forceinline__ void release(int t) const
    {
        if (t + ST < ntiles) __syncthreads();
    }
};

// Policy interface (see PolicyF64 in s2_force_fp64.cu):
//   NPL, kMinBlocks, NN, NGB, ORDER
//   struct IState; static void load_i(const ForceArgs&, int i, IState&)
//   struct Part { void zero(); }   per-tile partial sums, updated by pair()
//   struct Acc { void zero(); void add(const Part&); void shfl_add(int mask); void to_f64(double out[10]) }
//   template <int L, bool MASKED> static void pair(const unsigned char *stage, int tile, int k, bool valid,
//                                                  int jaddr, const IState&, Part&, Dec&, const Decomp&, int *seg, int segcap)
template <class P, int L>
__global__ void __launch_bounds__(kThreads, P::kMinBlocks) force_sweep_kernel(const ForceArgs a)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int NPL = P::NPL;
    const Decomp d = decompose<L>(a.Wj, a.ni);
    if constexpr (P::kTrackW)   // fp32: the flagged count of this call starts at zero (it is only raised by later launches)
        if (a.fix_count && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *a.fix_count = 0;
    TilePipe<NPL> pipe;
    pipe.init(smem_raw, a);
    unsigned char *tiles = pipe.tiles;
    const int tile = a.tile, j0 = pipe.j0, j1 = pipe.j1, ntiles = pipe.ntiles;
    typename P::IState I;
    P::load_i(a, d.i, I);

    typename P::Acc tot;     // running totals (fp64 / double-single)
    typename P::Part part;   // per-tile partial sums in the pair-arithmetic type
    tot.zero();
    Dec D;
    D.template init<P::NN, P::NGB>(I.h2);
    int *seg = nullptr;
    if (P::NGB) seg = a.seg + ((size_t)d.i * a.nslices_total + d.slice) * a.segcap;

    for (int t = 0; t < ntiles; ++t) {
        const unsigned char *stage = pipe.acquire(t);
        const int jt = j0 + t * tile;
        const int cnt = min(tile, j1 - jt);
        // this warp column's sub-range of the tile
        int beg = 0, end = cnt;
        if (a.Wj > 1) {
            const int sub = (cnt + a.Wj - 1) / a.Wj;
            beg = min(cnt, d.wj * sub);
            end = min(cnt, beg + sub);
        }
        const int len = end - beg;
        part.zero();
        if (L == 1) {
#pragma unroll P::kUnroll
            for (int k = beg; k < end; ++k)
                P::template pair<L, false>(stage, tile, k, true, jt + k, I, part, D, d, seg, a.segcap);
        } else {
            const int nfull = len / L;
            int k = beg + d.jl;
#pragma unroll P::kUnroll
            for (int it = 0; it < nfull; ++it, k += L)
                P::template pair<L, false>(stage, tile, k, true, jt + k, I, part, D, d, seg, a.segcap);
            if (len - nfull * L > 0) {   // ragged tail: lanes past the end re-read the last j, masked
                const bool valid = k < end;
                const int kk = valid ? k : end - 1;
                P::template pair<L, true>(stage, tile, kk, valid, jt + kk, I, part, D, d, seg, a.segcap);
            }
        }
        tot.add(part);   // two-level accumulation: per-tile partial sums, then the running total
        pipe.release(t);
    }

    // The sweep is over: let a dependent launch (the reduce kernel, launched with programmatic stream
    // serialisation) be staged while the epilogue runs; it waits for this grid's completion itself
    // (griddepcontrol.wait).  Not earlier: staged CTAs hold registers that a second sweep CTA per SM needs.
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");

    // combine the L lanes of each i in a fixed (butterfly) order
    if (L > 1) {
#pragma unroll
        for (int m = 1; m < L; m <<= 1) {
            tot.shfl_add(m);
            if (P::NN) {
                const double od2 = shfl_xor_d(D.nn_d2, m);
                const int oj = __shfl_xor_sync(0xffffffffu, D.nn_j, m);
                if (od2 < D.nn_d2 || (od2 == D.nn_d2 && (unsigned)oj < (unsigned)D.nn_j)) {
                    D.nn_d2 = od2;
                    D.nn_j = oj;
                }
            }
        }
    }

    if constexpr (P::kTrackW)
        if (a.wq && d.jl == 0 && d.i_valid) a.wq[(size_t)d.slice * a.ni + d.i] = (float)tot.wq();

    double out[10];
    tot.to_f64(out);
    int nn = D.nn_j;
    int row = d.slice;                      // partial row this thread's record goes to
    bool writer = d.jl == 0 && d.i_valid;

    if (a.fused && a.Wj > 1) {
        // warp columns: the Wj warps that hold the same i-particles (different j sub-ranges of every tile) add
        // their records in shared memory, in column order 0, 1, ...; column 0 carries the sum on
        double *sm = reinterpret_cast<double *>(tiles);
        const int il_cta = d.wi * (32 / L) + d.il;         // index of this thread's i inside the CTA
        __syncthreads();                                   // every warp is done reading the tile buffers
        if (d.jl == 0) {
            double *r = sm + (il_cta * a.Wj + d.wj) * REC;
#pragma unroll
            for (int c = 0; c < 10; ++c) r[c] = out[c];
            r[10] = D.nn_d2;
            r[11] = __hiloint2double(0, nn);
        }
        __syncthreads();
        writer = writer && d.wj == 0;
        if (d.jl == 0 && d.wj == 0) {
            for (int c = 1; c < a.Wj; ++c) {
                const double *r = sm + (il_cta * a.Wj + c) * REC;
#pragma unroll
                for (int k = 0; k < 10; ++k) out[k] += r[k];
                if (P::NN) {
                    const int oj = __double2loint(r[11]);
                    if (r[10] < D.nn_d2 || (r[10] == D.nn_d2 && (unsigned)oj < (unsigned)nn)) {
                        D.nn_d2 = r[10];
                        nn = oj;
                    }
                }
            }
        }
        row = blockIdx.y;
    }

    if (a.cluster > 1) {
        // Thread-block cluster of a.cluster CTAs along the slice axis: every CTA parks its records in its own
        // shared memory, the cluster synchronises, and CTA rank r sums the records of its share of the i-particles
        // over the ranks 0, 1, ... in that order through distributed shared memory.  One partial row per cluster.
        const int C = a.cluster;
        const int icta = (kWarps / a.Wj) * (32 / L);
        const int il_cta = d.wi * (32 / L) + d.il;            // index of this thread's i inside the CTA
        double *sm = reinterpret_cast<double *>(tiles);
        __syncthreads();                                       // tile buffers are dead from here on
        if (d.jl == 0 && (a.Wj == 1 || d.wj == 0)) {
            double *r = sm + il_cta * REC;
#pragma unroll
            for (int c = 0; c < 10; ++c) r[c] = out[c];
            r[10] = D.nn_d2;
            r[11] = __hiloint2double(0, nn);
        }
        cluster_sync();
        const uint32_t rank = cluster_ctarank();
        const int per = (icta + C - 1) / C;                    // i-particles summed by one rank
        for (int t = threadIdx.x; t < per * REC; t += kThreads) {
            const int li = t / REC, comp = t % REC;
            const int il_sum = rank * per + li;
            const int gi = blockIdx.x * icta + il_sum;
            if (il_sum >= icta || gi >= a.ni || comp == 11) continue;
            const uint32_t base = smem_u32(sm + il_sum * REC);
            double v = ld_dsmem_f64(base + comp * 8, 0);
            int bj = comp == 10 ? __double2loint(ld_dsmem_f64(base + 88, 0)) : 0;
            for (int rk = 1; rk < C; ++rk) {
                const double o = ld_dsmem_f64(base + comp * 8, rk);
                if (comp < 10) {
                    v += o;
                } else {   // nearest neighbour: (d2, address) lexicographic minimum
                    const int oj = __double2loint(ld_dsmem_f64(base + 88, rk));
                    if (o < v || (o == v && (unsigned)oj < (unsigned)bj)) {
                        v = o;
                        bj = oj;
                    }
                }
            }
            // record layout: 0-2 acc, 3-5 jerk, 6 pot, 7 nn_d2, 8 {nn, count}, 9-11 snap
            double *g = a.rec + ((size_t)(blockIdx.y / C) * a.ni + gi) * REC;
            if (comp < 7) g[comp] = v;
            else if (comp < 10) g[comp + 2] = v;
            else {
                g[7] = v;
                g[8] = __hiloint2double(0, bj);
            }
        }
        cluster_sync();                                        // nobody leaves while its shared memory is read
        writer = false;
    }

    if (writer && a.atomic) {
        atomic_add_record(a.out_final + (size_t)d.i * REC, out, a.order, row == 0);
    } else if (writer) {
        double *r = a.rec + ((size_t)row * a.ni + d.i) * REC;
        if (a.is_final) {
            if (P::NN && nn >= 0) nn = __double2loint(a.jid_plane[nn].y);
            if (P::NGB && D.cnt > a.ngb_cap) *a.overflow_flag = 1;
        }
        double2 *r2 = reinterpret_cast<double2 *>(r);
        r2[0] = make_double2(out[0], out[1]);
        r2[1] = make_double2(out[2], out[3]);
        r2[2] = make_double2(out[4], out[5]);
        r2[3] = make_double2(out[6], D.nn_d2);
        r2[4] = make_double2(__hiloint2double(D.cnt, nn), out[7]);
        r2[5] = make_double2(out[8], out[9]);
    }

    if (a.fused) {
        // The last CTA of this i-group to arrive reduces the gridDim.y partial rows (fixed order: lane l adds
        // rows l, l+32, ... then an xor-butterfly -- the same order as reduce_kernel).  No floating-point atomics.
        __shared__ int s_last;
        __threadfence();
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned prev = atomicAdd(&a.counters[blockIdx.x], 1u);
            s_last = prev == gridDim.y - 1;
        }
        __syncthreads();
        if (s_last) {
            __threadfence();
            const int icta = (kWarps / a.Wj) * (32 / L);
            const int i0 = blockIdx.x * icta;
            const int i1 = min(a.ni, i0 + icta);
            const int rows = gridDim.y / max(1, a.cluster);
            const int lane = threadIdx.x & 31;
            for (int i = i0 + (threadIdx.x >> 5); i < i1; i += kWarps)
                reduce_rows_warp<P::NN>(a.rec, a.out_final, a.jid_plane, i, a.ni, rows, a.order, lane);
            if (threadIdx.x == 0) a.counters[blockIdx.x] = 0;
        }
    }
}

// Register-tiled full-occupancy sweep (a4): one lane per i as in force_sweep_kernel<P, 1>, but every thread holds
// IPT i-particles, so each j read from shared memory (4-6 LDS.128 broadcasts) feeds IPT pair evaluations.
// Measured on B200: an LDS.128 costs the FP64 path ~2.75 cycles of register-file bandwidth, so
// halving the loads per pair is worth more than the occupancy it costs.  i-index of slot u of a thread:
// (blockIdx.x * IPT + u) * kThreads + threadIdx.x.  No warp columns, no cluster, no fused combine on this path:
// the grid is large, slices are combined by reduce_kernel (or there is a single slice).
// TL > 1 (plain sums only, no NN / neighbour lists): TL lanes share the IPT i-particles of a thread slot and take
// interleaved j, combined by an xor-butterfly like the lanes of force_sweep_kernel -- the register-tiled pair arithmetic
// (packed FFMA2 pairs in fp32, half the LDS.128 per pair in fp64) for i-lists too short to fill the chip with one lane per i.
template <class P, int IPT, int TL>
__global__ void __launch_bounds__(kThreads, P::kMinBlocksTiled) force_sweep_tiled_kernel(const ForceArgs a)
{
    static_assert(TL == 1 || (!P::NN && !P::NGB), "lanes per i-slot > 1: plain sums only");
    constexpr int IPC = kThreads / TL;   // i-slots per CTA (each holds IPT i-particles)
    const int jl = (threadIdx.x & 31) % TL;
    if constexpr (P::kTrackW)
        if (a.fix_count && blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) *a.fix_count = 0;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    constexpr int NPL = P::NPL;
    TilePipe<NPL> pipe;
    pipe.init(smem_raw, a);
    const int tile = a.tile;

    Decomp d[IPT];
    typename P::IState I[IPT];
    typename P::Acc tot[IPT];
    typename P::Part part[IPT];
    Dec D[IPT];
    int *seg[IPT];
#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        d[u].lane = threadIdx.x & 31;
        d[u].il = d[u].lane / TL; d[u].jl = jl; d[u].wi = threadIdx.x >> 5; d[u].wj = 0;
        d[u].i = (blockIdx.x * IPT + u) * IPC + threadIdx.x / TL;
        d[u].i_valid = d[u].i < a.ni;
        if (!d[u].i_valid) d[u].i = a.ni - 1;   // padding slots recompute the last i and never write
        d[u].slice = blockIdx.y;
        P::load_i(a, d[u].i, I[u]);
        tot[u].zero();
        D[u].template init<P::NN, P::NGB>(I[u].h2);
        seg[u] = P::NGB ? a.seg + ((size_t)d[u].i * a.nslices_total + d[u].slice) * a.segcap : nullptr;
    }

    for (int t = 0; t < pipe.ntiles; ++t) {
        const unsigned char *stage = pipe.acquire(t);
        const int jt = pipe.j0 + t * tile;
        const int cnt = min(tile, pipe.j1 - jt);
#pragma unroll
        for (int u = 0; u < IPT; ++u) part[u].zero();
        const int nfull = cnt / TL;
        int k = jl;
#pragma unroll P::kUnrollTiled
        for (int it = 0; it < nfull; ++it, k += TL) {
            typename P::JData J;
            P::load_j(stage, tile, k, J);
            if constexpr (IPT % 2 == 0 && P::kPacked2) {   // i-particles two by two in packed instructions
#pragma unroll
                for (int u = 0; u < IPT; u += 2)
                    P::interact2(J, true, jt + k, I + u, part + u, D + u, d + u, seg + u, a.segcap);
            } else {
#pragma unroll
                for (int u = 0; u < IPT; ++u)
                    P::template interact<1, false>(J, true, jt + k, I[u], part[u], D[u], d[u], seg[u], a.segcap);
            }
        }
        if (TL > 1 && cnt - nfull * TL > 0) {   // ragged tail: lanes past the end re-read the last j, masked
            const bool valid = k < cnt;
            const int kk = valid ? k : cnt - 1;
            typename P::JData J;
            P::load_j(stage, tile, kk, J);
            if constexpr (IPT % 2 == 0 && P::kPacked2) {
#pragma unroll
                for (int u = 0; u < IPT; u += 2)
                    P::interact2(J, valid, jt + kk, I + u, part + u, D + u, d + u, seg + u, a.segcap);
            } else {
#pragma unroll
                for (int u = 0; u < IPT; ++u)
                    P::template interact<1, true>(J, valid, jt + kk, I[u], part[u], D[u], d[u], seg[u], a.segcap);
            }
        }
#pragma unroll
        for (int u = 0; u < IPT; ++u) tot[u].add(part[u]);
        pipe.release(t);
    }
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");   // see force_sweep_kernel

    if (TL > 1) {   // combine the TL lanes of every i-slot in a fixed (butterfly) order
#pragma unroll
        for (int m = 1; m < TL; m <<= 1) {
#pragma unroll
            for (int u = 0; u < IPT; ++u) tot[u].shfl_add(m);
        }
    }

#pragma unroll
    for (int u = 0; u < IPT; ++u) {
        if (!d[u].i_valid || jl != 0) continue;
        if constexpr (P::kTrackW)
            if (a.wq) a.wq[(size_t)blockIdx.y * a.ni + d[u].i] = (float)tot[u].wq();
        double out[10];
        tot[u].to_f64(out);
        if (a.atomic) {
            atomic_add_record(a.out_final + (size_t)d[u].i * REC, out, a.order, blockIdx.y == 0);
            continue;
        }
        int nn = D[u].nn_j;
        if (a.is_final) {
            if (P::NN && nn >= 0) nn = __double2loint(a.jid_plane[nn].y);
            if (P::NGB && D[u].cnt > a.ngb_cap) *a.overflow_flag = 1;
        }
        double2 *r2 = reinterpret_cast<double2 *>(a.rec + ((size_t)blockIdx.y * a.ni + d[u].i) * REC);
        r2[0] = make_double2(out[0], out[1]);
        r2[1] = make_double2(out[2], out[3]);
        r2[2] = make_double2(out[4], out[5]);
        r2[3] = make_double2(out[6], D[u].nn_d2);
        r2[4] = make_double2(__hiloint2double(D[u].cnt, nn), out[7]);
        r2[5] = make_double2(out[8], out[9]);
    }
}

// Dynamic shared memory above 48 KB needs an opt-in that is per kernel AND per device.  Each kernel is opted in once
// per device to that device's full limit (idempotent, so contexts on different threads may race here harmlessly; a
// process-wide "largest size so far" would leave the kernels of a second device without their opt-in).
constexpr int kMaxDevices = 64;
template <class K>
inline cudaError_t opt_in_smem(K kern, std::atomic<int> *done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= kMaxDevices) return cudaErrorInvalidDevice;
    if (done[dev].load(std::memory_order_acquire)) return cudaSuccess;
    int lim = 0;
    cudaFuncAttributes fa;
    e = cudaDeviceGetAttribute(&lim, cudaDevAttrMaxSharedMemoryPerBlockOptin, dev);
    if (e == cudaSuccess) e = cudaFuncGetAttributes(&fa, kern);
    // static + dynamic shared memory together must stay within the device's opt-in limit
    if (e == cudaSuccess) e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, lim - (int)fa.sharedSizeBytes);
    if (e == cudaSuccess) done[dev].store(1, std::memory_order_release);
    return e;
}

// Host side: instantiate the kernel for a policy and launch it (or query its occupancy) for the
// run-time lane count L.
template <class P>
cudaError_t launch_L(int L, dim3 grid, size_t smem, const ForceArgs &a, cudaStream_t st, bool query,
                            int *ctas_per_sm)
{
#define S2_CASE(LL)                                                                                          \
    case LL: {                                                                                               \
        auto kern = force_sweep_kernel<P, LL>;                                                               \
        static std::atomic<int> s_opted[kMaxDevices];                                                        \
        if (cudaError_t e = opt_in_smem(kern, s_opted); e != cudaSuccess) return e;                          \
        if (query) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, kThreads, smem);  \
        if (a.cluster > 1) {                                                                                 \
            cudaLaunchConfig_t cfg = {};                                                                     \
            cfg.gridDim = grid; cfg.blockDim = dim3(kThreads); cfg.dynamicSmemBytes = smem; cfg.stream = st; \
            cudaLaunchAttribute at[1];                                                                       \
            at[0].id = cudaLaunchAttributeClusterDimension;                                                  \
            at[0].val.clusterDim.x = 1; at[0].val.clusterDim.y = a.cluster; at[0].val.clusterDim.z = 1;      \
            cfg.attrs = at; cfg.numAttrs = 1;                                                                \
            return cudaLaunchKernelEx(&cfg, kern, a);                                                        \
        }                                                                                                    \
        kern<<<grid, kThreads, smem, st>>>(a);                                                               \
        return cudaGetLastError();                                                                           \
    }
    if (L <= 0) {   // register-tiled sweep, P::kIPT i-particles per thread, -L (or 1) lanes per i-slot
        if constexpr (P::kIPT >= 2) {
#define S2_TCASE(TLL)                                                                                        \
    case TLL: {                                                                                              \
        auto kern = force_sweep_tiled_kernel<P, P::kIPT, TLL>;                                               \
        static std::atomic<int> s_opted[kMaxDevices];                                                        \
        if (cudaError_t e = opt_in_smem(kern, s_opted); e != cudaSuccess) return e;                          \
        if (query) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, kThreads, smem);  \
        kern<<<grid, kThreads, smem, st>>>(a);                                                               \
        return cudaGetLastError();                                                                           \
    }
            const int TL = L == 0 ? 1 : -L;
            if constexpr (!P::NN && !P::NGB) {
                switch (TL) {
                    S2_TCASE(1)
                    S2_TCASE(2)
                    S2_TCASE(4)
                    S2_TCASE(8)
                    S2_TCASE(16)
                    S2_TCASE(32)
                }
            } else {
                switch (TL) { S2_TCASE(1) }
            }
#undef S2_TCASE
            return cudaErrorInvalidValue;
        } else {
            return cudaErrorInvalidValue;
        }
    }
    switch (L) {
        S2_CASE(1)
        S2_CASE(2)
        S2_CASE(4)
        S2_CASE(8)
        S2_CASE(16)
        S2_CASE(32)
    }
#undef S2_CASE
    return cudaErrorInvalidValue;
}

}  // namespace s2
