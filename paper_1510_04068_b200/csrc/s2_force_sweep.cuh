// s2_force_sweep.cuh -- the i x j force sweep (a3-a5, a7, a8), generic over a precision policy.
//
// PAPER.md sec 2.1 (L46-L54): sinks (i) x sources (j); "parallelisation over the sink particles"
// when there are many sinks, Sapporo1's "parallelize over the source particles ... split into
// subsets" when there are few, and sec 3.1 (L104) "2D thread-blocks ... multiple threads per
// i-particle whereby each thread computes a part of the j-particles".  Here one kernel template
// covers the whole range:
//   - a CTA owns a group of i-particles (blockIdx.x) and a contiguous j-slice (blockIdx.y);
//   - inside a warp, L lanes share one i-particle and take interleaved j (L = 1: one lane per i,
//     every lane reads the same j from shared memory as a broadcast);
//   - for very few i (L = 32) the 8 warps may additionally be arranged as warp columns (Wj) that
//     take contiguous sub-ranges of the CTA's (single) tile;
//   - j tiles are staged global -> shared with 1-D bulk async copies (TMA, cp.async.bulk) that
//     complete on an mbarrier, double buffered;
//   - i-particles and accumulators live in registers; the L lanes combine with xor-shuffles in a
//     fixed order; each (slice, i) writes one 96-byte record.  Slices are combined by the
//     deterministic reduce kernel (s2_reduce.cu), never by atomics.
//   - neighbour hits are appended in ascending j order: per thread for L = 1, and for L > 1 by
//     warp ballot + population-count prefix inside the lane group.
#pragma once

#include <math_constants.h>

#include "s2_force_common.cuh"

namespace s2 {

// decision state: nearest neighbour (squared distance, j address) and neighbour count
struct Dec {
    double nn_d2;
    int nn_j;
    int cnt;
};

// d2: unsoftened squared distance in fp64 (reading R-D2); skip: self or padding lane.
template <int L, bool NN, bool NGB>
__device__ __forceinline__ void decide(double d2, int jaddr, bool skip, double h2, Dec &D,
                                       const Decomp &d, int *seg, int segcap)
{
    const double d2m = skip ? CUDART_INF : d2;
    if (NN) {
        if (d2m < D.nn_d2) {   // strict: the first (lowest-address) minimum of this lane is kept
            D.nn_d2 = d2m;
            D.nn_j = jaddr;
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
    uint64_t *full = reinterpret_cast<uint64_t *>(smem_raw);
    unsigned char *tiles = smem_raw + kSmemHeader;
    constexpr int NPL = P::NPL;
    constexpr int ST = 2;   // stages

    const Decomp d = decompose<L>(a.Wj, a.ni);
    const int tile = a.tile;
    const size_t stage_bytes = (size_t)NPL * tile * 16;

    const int j0 = blockIdx.y * a.slice_len;
    const int j1 = min(a.nj, j0 + a.slice_len);
    const int ntiles = j1 > j0 ? (j1 - j0 + tile - 1) / tile : 0;

    if (threadIdx.x == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        mbar_fence_init();
    }
    __syncthreads();

    auto issue = [&](int t) {
        const int st = t & 1;
        const int jt = j0 + t * tile;
        const uint32_t bytes = (uint32_t)min(tile, j1 - jt) * 16u;
        mbar_arrive_expect_tx(&full[st], bytes * NPL);
#pragma unroll
        for (int p = 0; p < NPL; ++p)
            bulk_g2s(tiles + st * stage_bytes + (size_t)p * tile * 16,
                     reinterpret_cast<const unsigned char *>(a.jp[p]) + (size_t)jt * 16, bytes, &full[st]);
    };
    if (threadIdx.x == 0 && ntiles > 0) issue(0);

    typename P::IState I;
    P::load_i(a, d.i, I);

    typename P::Acc tot;     // running totals (fp64 / double-single)
    typename P::Part part;   // per-tile partial sums in the pair-arithmetic type
    tot.zero();
    Dec D;
    D.nn_d2 = CUDART_INF;
    D.nn_j = -1;
    D.cnt = 0;
    int *seg = nullptr;
    if (P::NGB) seg = a.seg + ((size_t)d.i * a.nslices_total + d.slice) * a.segcap;

    for (int t = 0; t < ntiles; ++t) {
        if (threadIdx.x == 0 && t + 1 < ntiles) issue(t + 1);   // stage (t+1)&1 was released by the barrier ending tile t-1
        mbar_wait(&full[t & 1], (t >> 1) & 1);
        const unsigned char *stage = tiles + (t & 1) * stage_bytes;
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
#pragma unroll 2
            for (int it = 0; it < nfull; ++it, k += L)
                P::template pair<L, false>(stage, tile, k, true, jt + k, I, part, D, d, seg, a.segcap);
            if (len - nfull * L > 0) {   // ragged tail: lanes past the end re-read the last j, masked
                const bool valid = k < end;
                const int kk = valid ? k : end - 1;
                P::template pair<L, true>(stage, tile, kk, valid, jt + kk, I, part, D, d, seg, a.segcap);
            }
        }
        tot.add(part);   // two-level accumulation: per-tile partial sums, then the running total
        __syncthreads();
    }

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

    if (d.jl == 0 && d.i_valid) {
        double out[10];
        tot.to_f64(out);
        double *r = a.rec + ((size_t)d.slice * a.ni + d.i) * REC;
        int nn = D.nn_j;
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
        cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        if (e != cudaSuccess) return e;                                                                      \
        if (query) return cudaOccupancyMaxActiveBlocksPerMultiprocessor(ctas_per_sm, kern, kThreads, smem);  \
        kern<<<grid, kThreads, smem, st>>>(a);                                                               \
        return cudaGetLastError();                                                                           \
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
