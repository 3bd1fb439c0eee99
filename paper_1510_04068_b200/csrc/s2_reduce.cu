// s2_reduce.cu -- a6: deterministic combine of the per-slice partial records, and the
// neighbour-list compaction across slices.
//
// PAPER.md sec 2.2.4 (L88): Sapporo1 "contains two computational kernels ... the second sums the
// partial results"; Sapporo2 merged them with atomics.  This build keeps the second kernel
// because floating-point atomics make the summation order (and the last digit, L84, L164)
// run-dependent; here the order is fixed: lane l of the warp that owns i adds slices
// l, l+32, l+64, ... in sequence, then the 32 lanes are combined by an xor-butterfly
// (reduce_rows_warp, shared with the fused combine of the sweep, so both give the same bits).
// The kernel streams S*ni records of 96 bytes once: L2/HBM-bound, tiny.  It is launched with
// programmatic stream serialisation: the sweep triggers it after its j loop and this grid waits
// for the sweep's completion itself (griddepcontrol.wait).
#include <math_constants.h>

#include "s2_force_sweep.cuh"
#include "s2_bts_correct.cuh"

namespace s2 {

__global__ void __launch_bounds__(256) reduce_kernel(const ReduceArgs a)
{
    const int warp = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (warp >= a.ni) return;   // whole warp exits together
    const int i = warp;
    const int S = a.nslices_total;
    // programmatic dependent launch: this grid may start while the sweep is still running; wait for its results
    // (and let a dependent launch of its own -- the integrator's corrector -- be staged meanwhile)
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    if (!(a.flags & S2_WANT_NGB)) {   // plain sums (+ nn): the same fixed-order routine the fused combine uses
        if (a.flags & S2_WANT_NN)
            reduce_rows_warp<true>(a.part, a.out, a.jid_plane, i, a.ni, S, a.order, lane);
        else
            reduce_rows_warp<false>(a.part, a.out, a.jid_plane, i, a.ni, S, a.order, lane);
        if (a.f32.wq) fp32_flag_warp(a.f32, a.out, i, a.ni, lane);   // lane 0 reads back the record it has just written
        if (a.has_bts && lane == 0) bts_correct_one(a.bts, i, a.out + (size_t)i * REC);   // integrator: corrector in the same launch
        return;
    }

    double v[10];
#pragma unroll
    for (int c = 0; c < 10; ++c) v[c] = 0.0;
    double nn_d2 = CUDART_INF;
    int nn_j = -1;
    int cnt_total = 0;     // neighbours over my slices
    int written = 0;       // running output position (warp-uniform)

    for (int s0 = 0; s0 < S; s0 += 32) {
        const int s = s0 + lane;
        int c = 0;
        if (s < S) {
            const double2 *r = reinterpret_cast<const double2 *>(a.part + ((size_t)s * a.ni + i) * REC);
            const double2 r0 = r[0], r1 = r[1], r2 = r[2], r3 = r[3], r4 = r[4], r5 = r[5];
            v[0] += r0.x; v[1] += r0.y; v[2] += r1.x; v[3] += r1.y; v[4] += r2.x; v[5] += r2.y;
            v[6] += r3.x;
            if (a.order == 6) { v[7] += r4.y; v[8] += r5.x; v[9] += r5.y; }
            const int j = __double2loint(r4.x);
            c = __double2hiint(r4.x);
            // slices are visited in ascending order by each lane, so strict < keeps the lowest address
            if (r3.y < nn_d2 || (r3.y == nn_d2 && (unsigned)j < (unsigned)nn_j)) {
                nn_d2 = r3.y;
                nn_j = j;
            }
        }
        cnt_total += c;
        if (a.flags & S2_WANT_NGB) {
            // compaction across slices: exclusive prefix of the (clamped) segment lengths in slice
            // order = ascending j order, by warp shuffles; each lane copies its own segment.
            const int len = min(c, a.segcap);
            int incl = len;
#pragma unroll
            for (int m = 1; m < 32; m <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, m);
                if (lane >= m) incl += o;
            }
            const int base = written + incl - len;
            if (len > 0) {
                const int *src = a.seg + ((size_t)i * S + s) * a.segcap;
                int *dst = a.list + (size_t)i * a.ngb_cap;
                for (int k = 0; k < len && base + k < a.ngb_cap; ++k) dst[base + k] = src[k];
            }
            written += __shfl_sync(0xffffffffu, incl, 31);
        }
    }

#pragma unroll
    for (int m = 1; m < 32; m <<= 1) {
#pragma unroll
        for (int c = 0; c < 10; ++c) v[c] += shfl_xor_d(v[c], m);
        const double od2 = shfl_xor_d(nn_d2, m);
        const int oj = __shfl_xor_sync(0xffffffffu, nn_j, m);
        if (od2 < nn_d2 || (od2 == nn_d2 && (unsigned)oj < (unsigned)nn_j)) {
            nn_d2 = od2;
            nn_j = oj;
        }
        cnt_total += __shfl_xor_sync(0xffffffffu, cnt_total, m);
    }

    if (lane == 0) {
        int nn = nn_j;
        if ((a.flags & S2_WANT_NN) && nn >= 0) nn = __double2loint(a.jid_plane[nn].y);
        if ((a.flags & S2_WANT_NGB) && cnt_total > a.ngb_cap) *a.overflow_flag = 1;
        double2 *o = reinterpret_cast<double2 *>(a.out + (size_t)i * REC);
        o[0] = make_double2(v[0], v[1]);
        o[1] = make_double2(v[2], v[3]);
        o[2] = make_double2(v[4], v[5]);
        o[3] = make_double2(v[6], nn_d2);
        o[4] = make_double2(__hiloint2double(cnt_total, nn), v[7]);
        o[5] = make_double2(v[8], v[9]);
    }
    if (a.f32.wq) fp32_flag_warp(a.f32, a.out, i, a.ni, lane);
}

// Few partial rows, many i-particles (the full-occupancy sweeps with 2-16 j-slices): one THREAD per i streams its
// rows with coalesced loads instead of one warp per i with 2-16 active lanes.  The additions follow the same balanced
// tree the warp butterfly of reduce_rows_warp forms (rows beyond NST are its zero lanes), so the sums have the same bits:
//   T(lo, w) = T(lo, w/2) + T(lo + w/2, w/2),  T(l, 1) = row l.
struct RowSum {
    double v[10];
    double nn_d2;
    int nn_j;
};

template <int NST, int LO, int W, bool NN>
__device__ __forceinline__ void tree_rows(const double *part, size_t ni, size_t i, int order, RowSum &out)
{
    if constexpr (W == 1) {
        const double2 *r = reinterpret_cast<const double2 *>(part + ((size_t)LO * ni + i) * REC);
        const double2 r0 = r[0], r1 = r[1], r2 = r[2], r3 = r[3], r4 = r[4];
        out.v[0] = r0.x; out.v[1] = r0.y; out.v[2] = r1.x; out.v[3] = r1.y; out.v[4] = r2.x; out.v[5] = r2.y;
        out.v[6] = r3.x;
        out.v[7] = out.v[8] = out.v[9] = 0.0;
        if (order == 6) {
            const double2 r5 = r[5];
            out.v[7] = r4.y; out.v[8] = r5.x; out.v[9] = r5.y;
        }
        out.nn_d2 = r3.y;
        out.nn_j = __double2loint(r4.x);
    } else {
        tree_rows<NST, LO, W / 2, NN>(part, ni, i, order, out);
        if constexpr (LO + W / 2 < NST) {
            RowSum o;
            tree_rows<NST, LO + W / 2, W / 2, NN>(part, ni, i, order, o);
#pragma unroll
            for (int c = 0; c < 10; ++c) out.v[c] += o.v[c];
            if (NN && (o.nn_d2 < out.nn_d2 || (o.nn_d2 == out.nn_d2 && (unsigned)o.nn_j < (unsigned)out.nn_j))) {
                out.nn_d2 = o.nn_d2;
                out.nn_j = o.nn_j;
            }
        }
    }
}

template <int NST, bool NN>
__global__ void __launch_bounds__(256) reduce_thread_kernel(const ReduceArgs a)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= a.ni) return;
    RowSum t;
    tree_rows<NST, 0, (NST > 8 ? 16 : 8), NN>(a.part, (size_t)a.ni, (size_t)i, a.order, t);
    int nn = NN ? t.nn_j : -1;
    if (NN && nn >= 0) nn = __double2loint(a.jid_plane[nn].y);
    double2 *o = reinterpret_cast<double2 *>(a.out + (size_t)i * REC);
    o[0] = make_double2(t.v[0], t.v[1]);
    o[1] = make_double2(t.v[2], t.v[3]);
    o[2] = make_double2(t.v[4], t.v[5]);
    o[3] = make_double2(t.v[6], NN ? t.nn_d2 : CUDART_INF);
    o[4] = make_double2(__hiloint2double(0, nn), t.v[7]);
    o[5] = make_double2(t.v[8], t.v[9]);
}

template <int NST>
static cudaError_t launch_reduce_thread(const ReduceArgs &a, cudaStream_t st)
{
    const dim3 grid((a.ni + 255) / 256);
    if (a.flags & S2_WANT_NN) reduce_thread_kernel<NST, true><<<grid, 256, 0, st>>>(a);
    else reduce_thread_kernel<NST, false><<<grid, 256, 0, st>>>(a);
    return cudaGetLastError();
}

bool reduce_by_warp_kernel(const ReduceArgs &a)
{
    return !(!(a.flags & S2_WANT_NGB) && a.nslices_total >= 2 && a.nslices_total <= 16 && a.ni >= 4096);
}

cudaError_t launch_reduce(const ReduceArgs &a, cudaStream_t st)
{
    if (a.ni <= 0) return cudaSuccess;
    if (!reduce_by_warp_kernel(a)) {
        switch (a.nslices_total) {   // ordinary stream order (no programmatic launch): the rows are read through L1
        case 2: return launch_reduce_thread<2>(a, st);
        case 3: return launch_reduce_thread<3>(a, st);
        case 4: return launch_reduce_thread<4>(a, st);
        case 5: return launch_reduce_thread<5>(a, st);
        case 6: return launch_reduce_thread<6>(a, st);
        case 7: return launch_reduce_thread<7>(a, st);
        case 8: return launch_reduce_thread<8>(a, st);
        case 9: return launch_reduce_thread<9>(a, st);
        case 10: return launch_reduce_thread<10>(a, st);
        case 11: return launch_reduce_thread<11>(a, st);
        case 12: return launch_reduce_thread<12>(a, st);
        case 13: return launch_reduce_thread<13>(a, st);
        case 14: return launch_reduce_thread<14>(a, st);
        case 15: return launch_reduce_thread<15>(a, st);
        case 16: return launch_reduce_thread<16>(a, st);
        }
    }
    const int warps_per_block = a.ni <= 1024 ? 2 : 8;   // few i: spread the warps over more SMs
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3((a.ni + warps_per_block - 1) / warps_per_block);
    cfg.blockDim = dim3(32 * warps_per_block);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;   // overlap this launch with the sweep's tail
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, reduce_kernel, a);
}

}  // namespace s2
