// s2_force_fp64.cu -- IEEE fp64 pair arithmetic for the force sweep (PAPER.md L76, L128:
// "full native double precision").  Pair terms follow SURVEY sec 8(c) O3:
//   r = x_j - x_i, v = v_j - v_i, a = a_j - a_i
//   s = r.r + eps2;  y = s^(-1/2);  q = m_j y^3
//   acc += q r;  alpha = (r.v) y^2;  jerk += q (v - 3 alpha r)
//   beta = (v.v + r.a) y^2 + alpha^2;  snap += q (a - 6 alpha (v - 3 alpha r) - 3 beta r)
//   pot -= m_j y
// FP64-pipe instruction budget per pair: 32 for 4th order (33 with the
// decision distance kept separate), 54 for 6th order; the reciprocal square root is one
// MUFU.RSQ64H seed (rsqrt.approx.ftz.f64, ~2^-22) plus one third-order Newton step (5 FP64 ops).
#include <algorithm>

#include "s2_force_sweep.cuh"
#include "s2_predict.cuh"
#include "s2_bts_correct.cuh"

namespace s2 {

__device__ __forceinline__ double rsqrt_seed(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    return y;
}

// j-bank of the uniform-operand sweep (force_sweep_bank_kernel below): the whole 64 KB constant bank of this
// module holds one chunk of predicted j-particles, plane p at c_jbank[p * kChunk ..].  Every translation unit is a
// CUDA module of its own with its own bank, so this file is compiled twice (S2_BANK_ID 0 here, 1 through
// s2_force_fp64_bank1.cu): while the sweep reads one bank, the next chunk is copied into the other.
#ifndef S2_BANK_ID
#define S2_BANK_ID 0
#endif
#define S2_CAT2(a, b) a##b
#define S2_CAT(a, b) S2_CAT2(a, b)
constexpr int kBankBytes = 65536;
static __constant__ double2 c_jbank[kBankBytes / 16];

template <int ORDER_, bool NN_, bool NGB_>
struct PolicyF64 {
    static constexpr int ORDER = ORDER_;
    static constexpr bool NN = NN_, NGB = NGB_;
    // planes staged per tile: P0 P1 P2 P3 [P4 P5]; 2nd order (acc + pot only, GRAPE-5 style L34) needs no velocities:
    // P0 P1 P3 (P3 carries the id)
    static constexpr int NPL = ORDER == 6 ? 6 : (ORDER == 2 ? 3 : 4);
    static constexpr int kIdPlane = ORDER == 2 ? 2 : 3;
    // j-particles per chunk of the constant bank (1024 / 680 / 1360 for 4th / 6th / 2nd order)
    static constexpr int kChunk = kBankBytes / (NPL * 16) / 8 * 8;
    static constexpr int kUnrollBank = ORDER == 6 ? 4 : 8;   // pairs in flight there
    static constexpr int kMinBlocksBank = 2;   // 6th order: 126 registers at 4 pairs in flight, no spills (1 CTA of 158 registers: 275 Gpairs/s; 2 CTAs: 302)
    static constexpr int kBankThreads = 256;   // threads per CTA of the uniform-operand sweep
    static constexpr int kMinBlocks = 2;
    static constexpr int kUnroll = 4;   // pairs in flight per thread in the one-lane-per-i loop
    static constexpr int kMinBlocksTiled = ORDER == 6 ? 1 : 2;
    static constexpr int kIPT = kIptF64;                        // i-particles per thread in the register-tiled sweep
    static constexpr bool kPacked2 = false;
    // j per unrolled step there (x kIPT pairs in flight).  The 6th-order pair holds 18 more live doubles: with
    // 128 registers the totals spill inside the loop, so that variant runs one CTA per SM with 208 registers
    // (measured 290 vs 277 Gpairs/s)
    static constexpr int kUnrollTiled = 4;

    struct IState {
        double x, y, z, vx, vy, vz, ax, ay, az, h2, eps2;
        int id;
    };

    static constexpr bool kTrackW = false;
    struct Acc {
        double ax, ay, az, jx, jy, jz, pot, sx, sy, sz;
        __device__ __forceinline__ double wq() const { return 0.0; }
        __device__ __forceinline__ void zero()
        {
            ax = ay = az = jx = jy = jz = pot = 0.0;
            if (ORDER == 6) sx = sy = sz = 0.0;
        }
        __device__ __forceinline__ void add(const Acc &o)
        {
            ax += o.ax; ay += o.ay; az += o.az;
            jx += o.jx; jy += o.jy; jz += o.jz;
            pot += o.pot;
            if (ORDER == 6) { sx += o.sx; sy += o.sy; sz += o.sz; }
        }
        __device__ __forceinline__ void shfl_add(int m)
        {
            ax += shfl_xor_d(ax, m); ay += shfl_xor_d(ay, m); az += shfl_xor_d(az, m);
            jx += shfl_xor_d(jx, m); jy += shfl_xor_d(jy, m); jz += shfl_xor_d(jz, m);
            pot += shfl_xor_d(pot, m);
            if (ORDER == 6) { sx += shfl_xor_d(sx, m); sy += shfl_xor_d(sy, m); sz += shfl_xor_d(sz, m); }
        }
        __device__ __forceinline__ void to_f64(double o[10]) const
        {
            o[0] = ax; o[1] = ay; o[2] = az; o[3] = jx; o[4] = jy; o[5] = jz; o[6] = pot;
            o[7] = ORDER == 6 ? sx : 0.0; o[8] = ORDER == 6 ? sy : 0.0; o[9] = ORDER == 6 ? sz : 0.0;
        }
        __device__ __forceinline__ void from_f64(const double o[10])
        {
            ax = o[0]; ay = o[1]; az = o[2]; jx = o[3]; jy = o[4]; jz = o[5]; pot = o[6];
            if (ORDER == 6) { sx = o[7]; sy = o[8]; sz = o[9]; }
        }
    };

    using Part = Acc;   // fp64 partial sums per tile, added to fp64 totals

    static __device__ __forceinline__ void load_i(const ForceArgs &a, int i, IState &I)
    {
        const int ia = a.i_addr ? a.i_addr[i] : i;
        const double2 p0 = static_cast<const double2 *>(a.ip[0])[ia];
        const double2 p1 = static_cast<const double2 *>(a.ip[1])[ia];
        const double2 p3 = static_cast<const double2 *>(a.ip[kIdPlane])[ia];
        I.x = p0.x; I.y = p0.y; I.z = p1.x;
        if (ORDER != 2) {
            const double2 p2 = static_cast<const double2 *>(a.ip[2])[ia];
            I.vx = p2.x; I.vy = p2.y; I.vz = p3.x;
        }
        I.id = __double2loint(p3.y);
        if (ORDER == 6) {
            const double2 p4 = static_cast<const double2 *>(a.ip[4])[ia];
            const double2 p5 = static_cast<const double2 *>(a.ip[5])[ia];
            I.ax = p4.x; I.ay = p4.y; I.az = p5.x;
        }
        I.h2 = (NGB && a.h2) ? a.h2[i] : 0.0;
        I.eps2 = a.eps2;
    }

    // i-state kept as SoA between the chunk launches of the uniform-operand sweep: the first chunk gathers by
    // address (load_i) and parks it, later chunks read it back coalesced.  kIFields doubles per i.
    static constexpr int kIFields = ORDER == 6 ? 10 : (ORDER == 2 ? 4 : 7);
    static __device__ __forceinline__ void park_i(double *s, size_t ni, const IState &I)
    {
        s[0] = I.x; s[ni] = I.y; s[2 * ni] = I.z; s[3 * ni] = __hiloint2double(0, I.id);
        if (ORDER != 2) { s[4 * ni] = I.vx; s[5 * ni] = I.vy; s[6 * ni] = I.vz; }
        if (ORDER == 6) { s[7 * ni] = I.ax; s[8 * ni] = I.ay; s[9 * ni] = I.az; }
    }
    static __device__ __forceinline__ void unpark_i(const ForceArgs &a, const double *s, size_t ni, int i, IState &I)
    {
        I.x = s[0]; I.y = s[ni]; I.z = s[2 * ni]; I.id = __double2loint(s[3 * ni]);
        if (ORDER != 2) { I.vx = s[4 * ni]; I.vy = s[5 * ni]; I.vz = s[6 * ni]; }
        if (ORDER == 6) { I.ax = s[7 * ni]; I.ay = s[8 * ni]; I.az = s[9 * ni]; }
        I.h2 = (NGB && a.h2) ? a.h2[i] : 0.0;
        I.eps2 = a.eps2;
    }

    struct JData {   // one j-particle as read from the shared-memory planes
        double2 p0, p1, p2, p3, p4, p5;
    };
    static __device__ __forceinline__ void load_j(const unsigned char *stage, int tile, int k, JData &J)
    {
        const double2 *pl = reinterpret_cast<const double2 *>(stage);
        J.p0 = pl[k]; J.p1 = pl[tile + k];
        if (ORDER == 2) { J.p3 = pl[2 * tile + k]; } else { J.p2 = pl[2 * tile + k]; J.p3 = pl[3 * tile + k]; }
        if (ORDER == 6) { J.p4 = pl[4 * tile + k]; J.p5 = pl[5 * tile + k]; }
    }

    // the same particle from the constant bank: the index is warp-uniform, so these become LDCU loads into uniform
    // registers and the pair arithmetic takes them as UR operands -- no shared memory, no register-file write
    static __device__ __forceinline__ void load_j_bank(int k, JData &J)
    {
        J.p0 = c_jbank[k]; J.p1 = c_jbank[kChunk + k];
        if (ORDER == 2) { J.p3 = c_jbank[2 * kChunk + k]; } else { J.p2 = c_jbank[2 * kChunk + k]; J.p3 = c_jbank[3 * kChunk + k]; }
        if (ORDER == 6) { J.p4 = c_jbank[4 * kChunk + k]; J.p5 = c_jbank[5 * kChunk + k]; }
    }

    template <int L, bool MASKED>
    static __device__ __forceinline__ void pair(const unsigned char *stage, int tile, int k, bool valid, int jaddr,
                                                const IState &I, Acc &A, Dec &D, const Decomp &d, int *seg,
                                                int segcap)
    {
        JData J;
        load_j(stage, tile, k, J);
        interact<L, MASKED>(J, valid, jaddr, I, A, D, d, seg, segcap);
    }

    template <int L, bool MASKED>
    static __device__ __forceinline__ void interact(const JData &J, bool valid, int jaddr, const IState &I, Acc &A,
                                                    Dec &D, const Decomp &d, int *seg, int segcap)
    {
        const double2 p0 = J.p0, p1 = J.p1, p2 = J.p2, p3 = J.p3;
        const bool skip = (__double2loint(p3.y) == I.id) || (MASKED && !valid);

        const double dx = p0.x - I.x, dy = p0.y - I.y, dz = p1.x - I.z;
        double dvx = 0.0, dvy = 0.0, dvz = 0.0, rv = 0.0;
        if (ORDER != 2) { dvx = p2.x - I.vx; dvy = p2.y - I.vy; dvz = p3.x - I.vz; }
        double s;
        if (NN || NGB) {
            const double d2 = __fma_rn(dz, dz, __fma_rn(dy, dy, __dmul_rn(dx, dx)));
            decide<L, NN, NGB>(d2, jaddr, skip, I.h2, D, d, seg, segcap);
            s = d2 + I.eps2;
        } else {
            s = fma(dz, dz, fma(dy, dy, fma(dx, dx, I.eps2)));
        }
        if (ORDER != 2) rv = fma(dz, dvz, fma(dy, dvy, dx * dvx));

        // y = s^(-1/2): hardware seed + one third-order step  y <- y (1 + e/2 + 3 e^2 / 8), e = 1 - s y^2
        const double y0 = rsqrt_seed(s);
        const double e = fma(-(s * y0), y0, 1.0);
        // y0 (1 + e p) rather than fma(p, y0 e, y0): same count, but no DFMA with three distinct register
        // operands (those occupy the FP64 operand path for 3 cycles instead of 2)
        double y = y0 * fma(fma(0.375, e, 0.5), e, 1.0);
        y = skip ? 0.0 : y;

        const double y2 = y * y;
        const double my = p1.y * y;
        const double q = my * y2;
        A.pot -= my;
        if (ORDER == 2) {   // GRAPE-5 style: acceleration and potential only
            A.ax = fma(q, dx, A.ax); A.ay = fma(q, dy, A.ay); A.az = fma(q, dz, A.az);
            return;
        }
        const double alpha = rv * y2;
        const double a3 = -3.0 * alpha;
        const double tx = fma(a3, dx, dvx), ty = fma(a3, dy, dvy), tz = fma(a3, dz, dvz);
        A.ax = fma(q, dx, A.ax); A.ay = fma(q, dy, A.ay); A.az = fma(q, dz, A.az);
        A.jx = fma(q, tx, A.jx); A.jy = fma(q, ty, A.jy); A.jz = fma(q, tz, A.jz);
        if (ORDER == 6) {
            const double2 p4 = J.p4, p5 = J.p5;
            const double dax = p4.x - I.ax, day = p4.y - I.ay, daz = p5.x - I.az;
            const double w = fma(dvx, dvx, fma(dvy, dvy, fma(dvz, dvz, fma(dx, dax, fma(dy, day, dz * daz)))));
            const double b3 = -3.0 * fma(w, y2, alpha * alpha);
            const double a6 = a3 + a3;
            const double ux = fma(a6, tx, fma(b3, dx, dax));
            const double uy = fma(a6, ty, fma(b3, dy, day));
            const double uz = fma(a6, tz, fma(b3, dz, daz));
            A.sx = fma(q, ux, A.sx); A.sy = fma(q, uy, A.sy); A.sz = fma(q, uz, A.sz);
        }
    }
};

#ifndef S2_BANK_ONLY
cudaError_t dispatch_force_fp64(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                                cudaStream_t st, bool query, int *ctas_per_sm)
{
    const bool ngb = flags & S2_WANT_NGB, nn = (flags & S2_WANT_NN) || ngb;
    if (order == 2) {
        if (ngb) return launch_L<PolicyF64<2, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyF64<2, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyF64<2, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (order == 4) {
        if (ngb) return launch_L<PolicyF64<4, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyF64<4, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyF64<4, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (ngb) return launch_L<PolicyF64<6, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
    if (nn) return launch_L<PolicyF64<6, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    return launch_L<PolicyF64<6, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
}

// ---- fp32 fix-up (reading R-F32) -----------------------------------------------------------------
// The fp32 sweep flags the few i-particles whose jerk is a strongly cancelling sum (fp32_flag_kernel, s2_results.cu);
// they are re-evaluated here with the fp64 pair arithmetic above.  The flagged list is short (0.3-0.8 % of the i-list)
// and its length is known only on the device, so the work is cut into items (pair of flagged i, j-slice of <= 256
// particles) that the warps of a fixed grid take in turn: a single flagged particle is spread over N / 256 warps
// (2.5 us at N = 65536) instead of being swept by one warp alone (300 us).  No shared memory and no barrier: lanes
// read their own j from the L2-resident planes (coalesced 16-byte loads), each j feeds the two i of the item.
// Sums: lanes combine by the xor-butterfly; the slices of a group are added by the last warp to finish one of them, in
// a fixed order (below) -- deterministic.  Launched with programmatic stream serialisation behind the flagging kernel.
constexpr int kFixG = 2;          // flagged i-particles per item
template <class P>
__global__ void __launch_bounds__(128, P::ORDER == 6 ? 3 : 4) fp32_fix_sweep_kernel(const ForceArgs a)
{
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    asm volatile("griddepcontrol.wait;" ::: "memory");
    constexpr int NC = P::ORDER == 6 ? 10 : 7;
    __shared__ double s_V[kFixG * NC][128];
    const int count = *a.ni_dev;
    // groups below the capacity of the partial-row buffer are cut into a.S j-slices, one item each; the (unexpected)
    // rest takes one item per group that walks the same slices itself and adds them in the combine's order, so that a
    // particle gets the same bits whichever way it is handled and however many particles were flagged
    const int ngroups = (count + kFixG - 1) / kFixG, gcap = a.fix_kcap / kFixG;
    const int nsliced = a.S > 1 ? min(ngroups, gcap) : 0;
    const long long items_sliced = (long long)nsliced * a.S, items = items_sliced + (ngroups - nsliced);
    const int lane = threadIdx.x & 31;
    const long long nw = ((long long)gridDim.x * blockDim.x) >> 5;
    Decomp d{};
    Dec D{};
    for (long long it = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5; it < items; it += nw) {
        const bool sliced = it < items_sliced;
        const int g = sliced ? (int)(it / a.S) : nsliced + (int)(it - items_sliced);   // neighbouring warps: same i, next slice
        const int s_begin = sliced ? (int)(it % a.S) : 0, s_end = sliced ? s_begin + 1 : a.S;
        typename P::IState I[kFixG];
        int pos[kFixG];
#pragma unroll
        for (int u = 0; u < kFixG; ++u) {
            pos[u] = a.pos_list[min(g * kFixG + u, count - 1)];   // an odd tail recomputes the last entry, never written
            P::load_i(a, pos[u], I[u]);
        }
        // unsliced (rare): lane l holds the sum of slices l, l + 32, ... -- in shared memory, so that the common path
        // does not carry 2 x NC live doubles through the j loop
        if (!sliced) {
#pragma unroll
            for (int c = 0; c < kFixG * NC; ++c) s_V[c][threadIdx.x] = 0.0;
        }
        for (int s = s_begin; s < s_end; ++s) {
            typename P::Acc A[kFixG];
#pragma unroll
            for (int u = 0; u < kFixG; ++u) A[u].zero();
            const int j0 = a.j_first + s * a.slice_len, j1 = min(a.j_first + a.nj, j0 + a.slice_len);
#pragma unroll 4
            for (int jb = j0; jb < j1; jb += 32) {
                const bool valid = jb + lane < j1;
                const int j = valid ? jb + lane : j1 - 1;
                typename P::JData J;
                J.p0 = static_cast<const double2 *>(a.jp[0])[j]; J.p1 = static_cast<const double2 *>(a.jp[1])[j];
                J.p2 = static_cast<const double2 *>(a.jp[2])[j]; J.p3 = static_cast<const double2 *>(a.jp[3])[j];
                if (P::ORDER == 6) { J.p4 = static_cast<const double2 *>(a.jp[4])[j]; J.p5 = static_cast<const double2 *>(a.jp[5])[j]; }
#pragma unroll
                for (int u = 0; u < kFixG; ++u) P::template interact<1, true>(J, valid, j, I[u], A[u], D, d, nullptr, 0);
            }
#pragma unroll
            for (int m = 1; m < 32; m <<= 1) {
#pragma unroll
                for (int u = 0; u < kFixG; ++u) A[u].shfl_add(m);      // every lane ends with the same slice sums
            }
#pragma unroll
            for (int u = 0; u < kFixG; ++u) {
                double out[10];
                A[u].to_f64(out);
                const int k = g * kFixG + u;
                if (sliced) {
                    if (lane == 0 && k < count) {
                        double *r = a.fix_part + ((size_t)s * a.fix_kcap + k) * NC;
#pragma unroll
                        for (int c = 0; c < NC; ++c) r[c] = out[c];
                    }
                } else if (lane == (s & 31)) {
#pragma unroll
                    for (int c = 0; c < NC; ++c) s_V[u * NC + c][threadIdx.x] += out[c];
                }
            }
        }
        bool add_up = !sliced;
        double V[kFixG][NC];
#pragma unroll
        for (int u = 0; u < kFixG; ++u)
#pragma unroll
            for (int c = 0; c < NC; ++c) V[u][c] = sliced ? 0.0 : s_V[u * NC + c][threadIdx.x];
        if (sliced) {
            // the last warp to finish a slice of this group adds the group's rows: lane l takes slices l, l + 32, ... in
            // that order, then the xor-butterfly -- the same sums whoever arrives last.  No floating-point atomics.
            unsigned prev = 0;
            if (lane == 0) {
                __threadfence();
                prev = atomicAdd(a.fix_arrive + g, 1u);
            }
            prev = __shfl_sync(0xffffffffu, prev, 0);
            add_up = prev == (unsigned)a.S - 1u;
            if (add_up) {
                __threadfence();
#pragma unroll
                for (int u = 0; u < kFixG; ++u) {
                    const int k = min(g * kFixG + u, count - 1);
                    for (int sl = lane; sl < a.S; sl += 32) {
                        const double *r = a.fix_part + ((size_t)sl * a.fix_kcap + k) * NC;
#pragma unroll
                        for (int c = 0; c < NC; ++c) V[u][c] += __ldcg(r + c);
                    }
                }
                if (lane == 0) a.fix_arrive[g] = 0u;     // ready for the next call
            }
        }
        if (add_up) {                                    // warp-uniform
#pragma unroll
            for (int m = 1; m < 32; m <<= 1) {
#pragma unroll
                for (int u = 0; u < kFixG; ++u)
#pragma unroll
                    for (int c = 0; c < NC; ++c) V[u][c] += shfl_xor_d(V[u][c], m);
            }
            if (lane == 0) {
#pragma unroll
                for (int u = 0; u < kFixG; ++u) {
                    if (g * kFixG + u >= count) continue;
                    double *r = a.rec + (size_t)pos[u] * REC;
#pragma unroll
                    for (int c = 0; c < 7; ++c) r[c] = V[u][c];
                    if (P::ORDER == 6) { r[9] = V[u][7]; r[10] = V[u][8]; r[11] = V[u][9]; }
                }
            }
        }
    }
}

template <class K>
static cudaError_t launch_pdl_fix(K kern, int grid, const ForceArgs &a, cudaStream_t st)
{
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(grid); cfg.blockDim = dim3(128); cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, a);
}

// a.S j-slices of a.slice_len; a.ni = length of the whole i-list (bound of the flagged count); sm_count for the grid
cudaError_t launch_fp32_fix(const ForceArgs &a, int sm_count, cudaStream_t st)
{
    const long long worst = (long long)(a.fix_kcap / kFixG) * a.S + a.ni / kFixG + 1;   // items if every i were flagged
    const int grid = (int)std::min<long long>((worst + 3) / 4, (long long)4 * sm_count);
    cudaError_t e = a.order == 6 ? launch_pdl_fix(fp32_fix_sweep_kernel<PolicyF64<6, false, false>>, grid, a, st)
                                 : launch_pdl_fix(fp32_fix_sweep_kernel<PolicyF64<4, false, false>>, grid, a, st);
    return e;
}


// ---- small block steps of the integrator, many per launch (s2_bts.cu; sec 3.7) ---------------
// In a block-step run most steps move a handful of particles (median 4-10 of 16384): three dependent launches and a host
// synchronisation per step cost 30 us for 1 us of arithmetic.  This kernel runs such steps back to back WITHOUT leaving
// the GPU: one CTA of 512 threads per SM (cooperative launch: all co-resident).  CTA c OWNS the particles
// [c pc, (c+1) pc), one per thread, and keeps their base state, their step and their predicted j-planes in shared
// memory for the whole launch; global memory is read only where another CTA has changed it, and the predicted planes
// go back to it once, on the way out.  One block step:
//   exchange  every owner has published the active particles of its range for this step: a header {count} and one
//             record {address, id, predicted state} each.  Every CTA polls the headers, scans them (the active list is
//             ascending by owner and address) and knows n;
//   phase 1   sweep: the records are polled into shared memory (one thread each); one lane per active particle (32 to
//             a warp), the CTA's own j-range read from shared memory, cut into as many splits as there are warps to spare; the
//             splits are added in order and the CTA writes one partial row per active particle;
//   phase 2   combine + corrector: active particle k belongs to CTA k mod G, which polls the rows of all owners (a warp
//             per component: lane l takes rows l, l + 32, ... in that order, then the xor-butterfly) while the particle's
//             old state is already on its way from L2, then one thread per particle applies the Hermite corrector and
//             the time-step rule (bts_correct_from), writes the new state and keeps the step-level histogram;
//   barrier   the one grid barrier of a step: corrections and histogram are complete;
//   phase 3   next block time from the histogram; an owner whose particle was just corrected reloads it; every owner
//             predicts its particle to the new time (shared planes + global planes) and the owners publish the next
//             active set.
// Rows, records and headers are exchanged as 64-bit words {32 bits of payload, 32-bit sequence tag}: the reader polls
// until the words carry the tag of the step, so the data is its own flag and neither side needs a fence; the barrier
// after phase 2 keeps any CTA from running more than one exchange ahead of a reader (buffers are reused every step).
// The loop ends at the first step with more than b.spec_cap active particles or past b.t_end, or after b.max_steps; the
// control block, the global list, the base store and the predicted planes are then exactly what an ordinary step of
// s2_bts_run expects.  Every sum is taken in a fixed order: the run is bit-reproducible.
// Pair arithmetic: PolicyF64::interact above.
constexpr int kSmallThreads = 512, kSmallWarps = kSmallThreads / 32;
constexpr int kSmallCapMax = 1024;    // largest spec_cap (the address list in shared memory)
constexpr int kSmallMaxCtas = 256;    // the header scan takes one CTA per thread; rows per lane in the combine = 256 / 32
constexpr int kSmallPer = 8;          // particles a CTA combines per round
constexpr unsigned kSmallPolls = 1u << 22;   // a wait gives up after this many polls (seconds; a phase takes microseconds)

template <int ORDER>
struct SmallLayout {                  // dynamic shared memory of bts_small_steps_kernel
    static constexpr int NFB = ORDER == 6 ? 20 : 14;              // base fields (+ the step as field NFB)
    static constexpr int NPL = ORDER == 6 ? 6 : 4;                // predicted planes
    static constexpr int NC = ORDER == 6 ? 10 : 7;                // sums per particle
    static constexpr int NS = ORDER == 6 ? 9 : 6;                 // doubles of a predicted i-state
    static constexpr int RW = 2 + 2 * NS;                         // words of a record: address, id, state
    static constexpr size_t base_off = 0;
    static constexpr size_t j_off = base_off + (size_t)(NFB + 1) * kSmallThreads * 8;
    static constexpr size_t part_off = j_off + (size_t)NPL * kSmallThreads * 16;
    static constexpr size_t own_off = part_off + (size_t)NC * kSmallThreads * 8;
    static constexpr size_t list_off = own_off + (size_t)kSmallThreads * 4;
    static constexpr size_t off_off = list_off + (size_t)kSmallCapMax * 4;
    static constexpr int kRound = ORDER == 6 ? 256 : 512;         // active particles swept per round (their states in shared memory)
    static constexpr size_t is_off = (off_off + (size_t)(kSmallMaxCtas + 1) * 4 + 15) & ~(size_t)15;
    static constexpr size_t iid_off = is_off + (size_t)NS * kRound * 8;
    static constexpr size_t bytes = iid_off + (size_t)kRound * 4;
};

__device__ __forceinline__ unsigned long long ll_word(unsigned payload, unsigned tag) { return (unsigned long long)payload | ((unsigned long long)tag << 32); }
__device__ __forceinline__ void ll_store2(unsigned long long *p, unsigned lo, unsigned hi, unsigned tag)   // 16-byte aligned
{
    asm volatile("st.relaxed.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(ll_word(lo, tag)), "l"(ll_word(hi, tag)) : "memory");
}
__device__ __forceinline__ void ll_store_double(unsigned long long *p, double v, unsigned tag)
{
    ll_store2(p, (unsigned)__double2loint(v), (unsigned)__double2hiint(v), tag);
}
__device__ __forceinline__ void ll_load2(const unsigned long long *p, unsigned long long &x, unsigned long long &y)
{
    asm volatile("ld.relaxed.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(x), "=l"(y) : "l"(p) : "memory");
}
__device__ __forceinline__ bool ll_ok(unsigned long long x, unsigned long long y, unsigned tag)
{
    return (unsigned)(x >> 32) == tag && (unsigned)(y >> 32) == tag;
}
__device__ __forceinline__ double ll_double(unsigned long long x, unsigned long long y) { return __hiloint2double((int)(unsigned)y, (int)(unsigned)x); }

// Barrier over the whole (co-resident) grid.  Arrival is a release-add (this CTA's writes of the phase are visible
// before it counts), the wait polls with relaxed loads and ends with one acquire fence (which also drops the SM's L1
// lines: what other CTAs wrote is then read from L2).  The counter only grows during a launch (target = barriers so
// far x CTAs).
__device__ __forceinline__ bool grid_barrier(unsigned *bar, unsigned target, int *s_flag)
{
    __syncthreads();
    if (threadIdx.x == 0) {
        asm volatile("red.release.gpu.global.add.u32 [%0], %1;" ::"l"(bar), "r"(1u) : "memory");
        unsigned spins = 0, v;
        int ok = 1;
        for (;;) {
            asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(bar) : "memory");
            if (v >= target) break;
            if (++spins > kSmallPolls) { ok = 0; break; }
        }
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        *s_flag = ok;
    }
    __syncthreads();
    return *s_flag != 0;
}

template <int ORDER>
__global__ void __launch_bounds__(kSmallThreads, 1) bts_small_steps_kernel(const ForceArgs a, const BtsArgs b, const PredictArgs pa)
{
    using P = PolicyF64<ORDER, false, false>;
    using L = SmallLayout<ORDER>;
    constexpr int NC = L::NC, NFB = L::NFB, NPL = L::NPL, NS = L::NS, RW = L::RW;
    extern __shared__ __align__(16) unsigned char s_raw[];
    double (*s_base)[kSmallThreads] = reinterpret_cast<double (*)[kSmallThreads]>(s_raw + L::base_off);
    double2 (*s_J)[kSmallThreads] = reinterpret_cast<double2 (*)[kSmallThreads]>(s_raw + L::j_off);
    double (*s_part)[kSmallThreads] = reinterpret_cast<double (*)[kSmallThreads]>(s_raw + L::part_off);
    int *s_own = reinterpret_cast<int *>(s_raw + L::own_off);     // own active particles (thread numbers), ascending
    int *s_list = reinterpret_cast<int *>(s_raw + L::list_off);   // addresses of all active particles of the step
    int *s_off = reinterpret_cast<int *>(s_raw + L::off_off);     // exclusive scan of the owners' counts
    double (*s_I)[L::kRound] = reinterpret_cast<double (*)[L::kRound]>(s_raw + L::is_off);   // predicted states of a round's particles
    int *s_Iid = reinterpret_cast<int *>(s_raw + L::iid_off);
    __shared__ int s_w[kSmallWarps];
    __shared__ unsigned s_hist[2];
    __shared__ int s_flag, s_bad;
    __shared__ double s_r[kSmallPer][12];
    __shared__ long long s_ph[9];                                 // profile (b.prof): cycles of one CTA per part of a step
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int cta = blockIdx.x, G = gridDim.x;
    const int N = b.n, cap = b.spec_cap;
    const int pc = (((N + G - 1) / G) + 31) & ~31;                // particles per owner (<= kSmallThreads: the launcher checks)
    const int Gj = (N + pc - 1) / pc;                             // CTAs that own particles
    const int pbeg = min(N, cta * pc), np = min(N, pbeg + pc) - pbeg;
    const int i_own = pbeg + tid;
    const bool have = tid < np;
    Decomp d{};
    Dec D{};

    double t_cur = b.ctl->t_next, t_done = b.ctl->t_done;
    unsigned seq = (unsigned)b.ctl->tag + 1u;                      // tag of the step about to run
    int step = 0, n = 0;
    unsigned target = 0;
    bool ok = true;
    if (tid == 0) s_bad = 0;
    const bool prof = b.prof != nullptr && cta == b.prof_cta && tid == 0;
    long long pc0 = 0;
    if (prof) {
        for (int q = 0; q < 9; ++q) s_ph[q] = 0;
        pc0 = clock64();
    }
#define S2_PH(i)                     \
    if (prof) {                      \
        const long long c1 = clock64(); \
        s_ph[i] += c1 - pc0;         \
        pc0 = c1;                    \
    }

    // compaction of the own active particles (ascending), their records and the header, all tagged `tag`
    auto publish = [&](bool act, const double *xp, const double *vp, const double *ap, int id, unsigned tag) -> int {
        const unsigned bal = __ballot_sync(0xffffffffu, act);
        if (lane == 0) s_w[warp] = __popc(bal);
        __syncthreads();
        int pos = __popc(bal & ((1u << lane) - 1u)), total = 0;
#pragma unroll
        for (int w = 0; w < kSmallWarps; ++w) {
            if (w < warp) pos += s_w[w];
            total += s_w[w];
        }
        if (act) {
            s_own[pos] = tid;
            if (total <= cap) {                                   // (more than that here alone: the step is not a small one)
                unsigned long long *r = b.xrec + (size_t)(pbeg + pos) * RW;
                ll_store2(r, (unsigned)i_own, (unsigned)id, tag);
#pragma unroll
                for (int c = 0; c < 3; ++c) {
                    ll_store_double(r + 2 + 2 * c, xp[c], tag);
                    ll_store_double(r + 8 + 2 * c, vp[c], tag);
                    if (ORDER == 6) ll_store_double(r + 14 + 2 * c, ap[c], tag);
                }
            }
        }
        if (tid < G) {                                            // one copy per reader: no line is polled by more than one CTA
            const unsigned long long h = ll_word((unsigned)total, tag);
            asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(b.xhdr + (size_t)tid * G + cta), "l"(h) : "memory");
        }
        __syncthreads();
        return total;
    };

    // ---- entry: resident copies of the own particle, the own active particles of the first step ---------------------
    int my_id = 0, cnt = 0;
    bool act = false;
    {
        double xp[3] = {0, 0, 0}, vp[3] = {0, 0, 0}, ap[3] = {0, 0, 0};
        if (have) {
#pragma unroll
            for (int k = 0; k < NFB; ++k) s_base[k][tid] = __ldcg(pa.f[k] + i_own);
            s_base[NFB][tid] = __ldcg(b.dt + i_own);
            my_id = __ldcg(pa.id + i_own);
            double2 q[6];
#pragma unroll
            for (int p = 0; p < NPL; ++p) s_J[p][tid] = q[p] = __ldcg(pa.p[p] + i_own);   // (already predicted to t_cur)
            xp[0] = q[0].x; xp[1] = q[0].y; xp[2] = q[1].x; vp[0] = q[2].x; vp[1] = q[2].y; vp[2] = q[3].x;
            if (ORDER == 6) { ap[0] = q[4].x; ap[1] = q[4].y; ap[2] = q[5].x; }
            const double x = t_cur / s_base[NFB][tid];            // exact: the step is a power of two
            act = x == floor(x);
        }
        cnt = publish(act, xp, vp, ap, my_id, seq);
    }

    if (prof) pc0 = clock64();
    for (;;) {
        // ---- exchange: the owners' counts of this step -> scan, n ---------------------------------------------------
        {
            int c = 0;
            if (tid < Gj) {
                unsigned long long h = 0;
                unsigned spins = 0;
                for (;;) {
                    asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(h) : "l"(b.xhdr + (size_t)cta * G + tid) : "memory");
                    if ((unsigned)(h >> 32) == seq) break;
                    if (++spins > kSmallPolls) { s_bad = 1; break; }
                }
                c = (int)(unsigned)h;
            }
            int incl = c;
#pragma unroll
            for (int q = 1; q < 32; q <<= 1) {
                const int o = __shfl_up_sync(0xffffffffu, incl, q);
                if (lane >= q) incl += o;
            }
            if (lane == 31) s_w[warp] = incl;
            __syncthreads();
            int wb = 0;
            for (int w = 0; w < warp; ++w) wb += s_w[w];
            if (tid < Gj) s_off[tid] = wb + incl - c;
            if (tid == Gj - 1) s_off[Gj] = wb + incl;
            __syncthreads();
        }
        n = s_off[Gj];
        if (s_bad) { ok = false; break; }
        if (!(n >= 1 && n <= cap && t_cur <= b.t_end && step < b.max_steps)) break;
        S2_PH(0)

        // ---- phase 1: sweep -------------------------------------------------------------------------------------
        for (int k0 = 0; k0 < n; k0 += L::kRound) {               // (one round unless n > 512 | 256)
            const int nk = min(L::kRound, n - k0);                // particles of this round
            // their records, one thread each (polled until they carry this step's tag) -> shared memory
            for (int kl = tid; kl < nk; kl += kSmallThreads) {
                const int k = k0 + kl;
                int lo = 0, hi = Gj - 1;                          // owner of particle k: last c with s_off[c] <= k
                while (lo < hi) {
                    const int mid = (lo + hi + 1) >> 1;
                    if (s_off[mid] <= k) lo = mid; else hi = mid - 1;
                }
                const unsigned long long *r = b.xrec + ((size_t)lo * pc + (k - s_off[lo])) * RW;
                unsigned long long w[RW];
                for (unsigned spins = 0;; ++spins) {
                    bool all = true;
#pragma unroll
                    for (int u = 0; u < RW / 2; ++u) {
                        ll_load2(r + 2 * u, w[2 * u], w[2 * u + 1]);
                        all = all && ll_ok(w[2 * u], w[2 * u + 1], seq);
                    }
                    if (all) break;
                    if (spins > kSmallPolls) { s_bad = 1; break; }
                }
                s_list[k] = (int)(unsigned)w[0];
                s_Iid[kl] = (int)(unsigned)w[1];
#pragma unroll
                for (int q = 0; q < NS; ++q) s_I[q][kl] = ll_double(w[2 + 2 * q], w[3 + 2 * q]);
            }
            __syncthreads();
            S2_PH(1)
            const int ngr = (nk + 31) >> 5;                       // groups of 32 particles
            const int js = kSmallWarps / ngr;                     // splits of the own j-range: every warp gets an item
            // up to 32 particles: the lanes of a warp split its j as well (P2 lanes take the particles, 32 / P2 lane groups
            // take interleaved j), so that a handful of particles is a handful of pairs per lane, not per warp
            const int P2 = ngr > 1 ? 32 : (nk <= 1 ? 1 : 1 << (32 - __clz(nk - 1)));
            if (warp < ngr * js) {
                const int gl = warp / js, sp = warp - gl * js;    // neighbouring warps: same particles, next split
                const int ls = lane / P2, sub = 32 / P2;
                const int kl = min(gl * 32 + (lane & (P2 - 1)), nk - 1);   // (idle lanes recompute the last particle)
                typename P::IState I;
                I.x = s_I[0][kl]; I.y = s_I[1][kl]; I.z = s_I[2][kl]; I.vx = s_I[3][kl]; I.vy = s_I[4][kl]; I.vz = s_I[5][kl];
                I.ax = I.ay = I.az = 0.0;
                if (ORDER == 6) { I.ax = s_I[6][kl]; I.ay = s_I[7][kl]; I.az = s_I[8][kl]; }
                I.id = s_Iid[kl];
                I.h2 = 0.0;
                I.eps2 = a.eps2;
                typename P::Acc A;
                A.zero();
                const int len = (np + js - 1) / js;
                const int j0 = sp * len, j1 = min(np, j0 + len);
#pragma unroll 2
                for (int jj = j0 + ls; jj < j1; jj += sub) {      // the same j in the lanes of a group: broadcast reads of shared memory
                    typename P::JData J;
                    J.p0 = s_J[0][jj]; J.p1 = s_J[1][jj]; J.p2 = s_J[2][jj]; J.p3 = s_J[3][jj];
                    if (ORDER == 6) { J.p4 = s_J[4][jj]; J.p5 = s_J[5][jj]; }
                    P::template interact<1, false>(J, true, pbeg + jj, I, A, D, d, nullptr, 0);
                }
                for (int m = P2; m < 32; m <<= 1) A.shfl_add(m);  // the lane groups of a particle, fixed order
                if (ls == 0) {
                    double out[10];
                    A.to_f64(out);
                    const int row = (sp * ngr + gl) * 32 + lane;
#pragma unroll
                    for (int c = 0; c < NC; ++c) s_part[c][row] = out[c];
                }
            }
            __syncthreads();
            S2_PH(2)
            if (cta < Gj) {
                for (int e = tid; e < nk * NC; e += kSmallThreads) {   // this owner's row of each: the splits in order
                    const int c = e / nk, kl = e - c * nk;
                    double v = 0.0;
                    for (int sp = 0; sp < js; ++sp) v += s_part[c][sp * ngr * 32 + kl];
                    ll_store_double(b.xrows + (((size_t)cta * cap + k0 + kl) * NC + c) * 2, v, seq);
                }
            }
            __syncthreads();
        }

        S2_PH(3)
        // ---- phase 2: combine + corrector ----------------------------------------------------------------------
        const int mine = n > cta ? (n - cta + G - 1) / G : 0;     // this CTA's particles: k = cta + m G
        for (int m0 = 0; m0 < mine; m0 += kSmallPer) {
            const int mr = min(kSmallPer, mine - m0);
            BtsOld old;
            int i_m = 0;
            if (tid < mr) {                                       // old state: on its way while the rows are polled
                i_m = s_list[cta + (m0 + tid) * G];
                bts_load_old(b, i_m, old);
            }
            for (int it = warp; it < mr * NC; it += kSmallWarps) {
                const int m = it / NC, c = it - m * NC, k = cta + (m0 + m) * G;
                unsigned long long x[kSmallMaxCtas / 32], y[kSmallMaxCtas / 32];
                for (unsigned spins = 0;; ++spins) {
                    bool all = true;
#pragma unroll
                    for (int u = 0; u < kSmallMaxCtas / 32; ++u) {
                        const int row = lane + 32 * u;
                        if (row < Gj) {
                            ll_load2(b.xrows + (((size_t)row * cap + k) * NC + c) * 2, x[u], y[u]);
                            all = all && ll_ok(x[u], y[u], seq);
                        }
                    }
                    if (all) break;
                    if (spins > kSmallPolls) { s_bad = 1; break; }
                }
                double v = 0.0;
#pragma unroll
                for (int u = 0; u < kSmallMaxCtas / 32; ++u)      // added in row order
                    if (lane + 32 * u < Gj) v += ll_double(x[u], y[u]);
#pragma unroll
                for (int q = 1; q < 32; q <<= 1) v += shfl_xor_d(v, q);
                if (lane == 0) s_r[m][c < 7 ? c : c + 2] = v;     // record layout: acc, jerk, pot at 0..6, snap at 9..11
            }
            __syncthreads();
            S2_PH(4)
            if (tid < mr) bts_correct_from(b, i_m, t_cur, old, s_r[tid]);
            __syncthreads();
            S2_PH(5)
        }
        if (!(ok = grid_barrier(b.bar, target += G, &s_flag)) || s_bad) { ok = false; break; }
        S2_PH(6)

        // ---- phase 3: next block time, reload of a corrected particle, prediction, the next active set -------------------
        if (tid < 64) {
            const unsigned bal = __ballot_sync(0xffffffffu, __ldcg(b.hist + tid) > 0);
            if (lane == 0) s_hist[warp] = bal;
        }
        if (have && act) {                                        // corrected in this step (by CTA k mod G): new state from L2
#pragma unroll
            for (int k = 0; k < NFB; ++k) s_base[k][tid] = __ldcg(pa.f[k] + i_own);
            s_base[NFB][tid] = __ldcg(b.dt + i_own);
        }
        __syncthreads();
        const int lev = s_hist[1] ? 63 - __clz(s_hist[1]) : 31 - __clz(s_hist[0] | 1u);   // highest occupied level = smallest step
        const double t_next = t_cur + scalbn(1.0, -lev);
        {
            double xp[3] = {0, 0, 0}, vp[3] = {0, 0, 0}, ap[3] = {0, 0, 0};
            act = false;
            if (have) {
                const double x = t_next / s_base[NFB][tid];       // exact: the step is a power of two
                act = x == floor(x);
                predict_state<ORDER>([&](int k) { return s_base[k][tid]; }, t_next, xp, vp, ap);
                double2 q[6];
                q[0] = make_double2(xp[0], xp[1]); q[1] = make_double2(xp[2], s_base[1][tid]);
                q[2] = make_double2(vp[0], vp[1]); q[3] = make_double2(vp[2], __hiloint2double(0, my_id));
                q[4] = make_double2(ap[0], ap[1]); q[5] = make_double2(ap[2], 0.0);
#pragma unroll
                for (int p = 0; p < NPL; ++p) s_J[p][tid] = q[p];  // (the global planes are written once, on the way out)
            }
            S2_PH(7)
            cnt = publish(act, xp, vp, ap, my_id, seq + 1u);
        }
        S2_PH(8)
        if (cta == 0 && tid == 0) b.h_log[step] = n;
        t_done = t_cur;
        t_cur = t_next;
        ++step;
        ++seq;
    }

    // what the kernel leaves behind for whoever runs the pending step: the predicted planes of the own particles and the
    // own segment of the active list (s_off is that step's scan)
    if (ok) {
        if (have) {
#pragma unroll
            for (int p = 0; p < NPL; ++p) pa.p[p][i_own] = s_J[p][tid];
        }
        for (int q = tid; q < cnt; q += kSmallThreads) b.ilist[s_off[cta] + q] = pbeg + s_own[q];
    }
    if (prof) {
        for (int q = 0; q < 9; ++q) b.prof[q] += s_ph[q];
        b.prof[9] += step;
    }
#undef S2_PH
    if (cta == 0 && tid == 0) {
        BtsCtl c = *b.ctl;
        c.t_next = t_cur; c.n_next = n; c.steps += step; c.t_done = t_done; c.tag = (long long)seq;
        if (!ok) c.error = 1;
        *b.ctl = c;
        *b.h_ctl = c;
    }
    if (ok) {                                                     // the last CTA out leaves the counters at zero for the next launch
        __syncthreads();
        if (tid == 0 && atomicAdd(b.bar + 1, 1u) == (unsigned)G - 1u) {
            b.bar[0] = 0u;
            b.bar[1] = 0u;
        }
    }
}

// Launch of the above on the whole chip; b.spec_cap <= kSmallCapMax; b.xrows holds sm_count * spec_cap * (7 | 10) * 2 words,
// b.xrec n * (14 | 20) words, b.xhdr sm_count^2 words, all zero before the first launch after s2_bts_init.  Returns
// cudaErrorNotSupported when the device or the problem cannot run it (no cooperative launch, more SMs than the header scan
// takes, more than 512 particles per SM): the caller then steps the ordinary way.
cudaError_t launch_bts_small_steps(const ForceArgs &a, const BtsArgs &b, const PredictArgs &pa, int device, int sm_count, cudaStream_t st)
{
    static int supported[64] = {};                                // per device: 0 unknown, 1 yes, -1 no
    if (device < 0 || device >= 64 || b.spec_cap < 1 || b.spec_cap > kSmallCapMax || sm_count > kSmallMaxCtas) return cudaErrorNotSupported;
    if ((((b.n + sm_count - 1) / sm_count + 31) & ~31) > kSmallThreads) return cudaErrorNotSupported;
    const void *kern = a.order == 6 ? (const void *)bts_small_steps_kernel<6> : (const void *)bts_small_steps_kernel<4>;
    const size_t smem = a.order == 6 ? SmallLayout<6>::bytes : SmallLayout<4>::bytes;
    if (supported[device] == 0) {
        int coop = 0, per_sm = 0;
        cudaError_t e = cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, device);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(bts_small_steps_kernel<4>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SmallLayout<4>::bytes);
        if (e == cudaSuccess) e = cudaFuncSetAttribute(bts_small_steps_kernel<6>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)SmallLayout<6>::bytes);
        if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, bts_small_steps_kernel<6>, kSmallThreads, SmallLayout<6>::bytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            supported[device] = -1;
            return cudaErrorNotSupported;
        }
        supported[device] = (coop && per_sm >= 1) ? 1 : -1;
    }
    if (supported[device] < 0) return cudaErrorNotSupported;
    void *args[3] = {(void *)&a, (void *)&b, (void *)&pa};
    return cudaLaunchCooperativeKernel(kern, dim3(sm_count), dim3(kSmallThreads), args, smem, st);
}

#endif   // S2_BANK_ONLY

// ---- uniform-operand sweep (a4 at the largest n_i) ------------------------------------------------------------
// Every lane of a warp reads the same j-particle, so j is warp-uniform data.  Here it is not staged through
// shared memory at all: a chunk of the predicted j-store is copied into the module's constant bank between
// launches, the kernel reads it with uniform loads (LDCU) and the FP64 instructions take it as uniform-register
// operands (DADD R, -R, UR).  That removes the LDS.128 write-backs that cost the FP64 operand path ~2.75 cycles
// each and every barrier: warps are fully independent, one i-particle per lane, eight pairs in
// flight per thread.  The price is one launch per chunk (1024 j at 4th order), with the running sums carried
// through an SoA state buffer; sums are added in address order chunk by chunk, so results are bit-reproducible.
constexpr int kBankLooks = 15;   // later looks at the next chunk's ticket inside a chunk (0: only at the start);
                                            // measured at n_i = 65536 / 81920 / 2^18: 0: 421 / 480 / 513, 3: 494 / - / 518, 7: 501 / 503 / 518,
                                            // 15: 506 / 510 / 518, 31: 507 / 511 / 518, 63: 501 / 504 / 512 Gpairs/s
template <class P, int BANK, int THREADS>   // BANK only makes the kernels of the two translation units distinct symbols
__global__ void __launch_bounds__(THREADS, P::kMinBlocksBank * P::kBankThreads / THREADS) force_sweep_bank_kernel(const ForceArgs a)
{
    constexpr int NC = P::ORDER == 6 ? 10 : 7;   // running sums carried per i
    Decomp d;
    d.lane = threadIdx.x & 31;
    d.il = d.lane; d.jl = 0; d.wi = threadIdx.x >> 5; d.wj = 0; d.slice = 0;
    d.i = blockIdx.x * THREADS + threadIdx.x;   // 256 threads (2 CTAs per SM) or 128 (4 per SM: finer fill of shared rounds)
    d.i_valid = d.i < a.ni;
    if (!d.i_valid) d.i = a.ni - 1;   // padding lanes recompute the last i and never write
    // Overlap of consecutive chunk launches (programmatic dependent launch) and hand-over of the two banks:
    //   * the launch of chunk c reads bank c & 1; when its last CTA is through the loop, that CTA copies chunk c + 2
    //     into the same bank and publishes ready[bank] = ticket(c + 2);
    //   * a CTA lets the next launch start (launch_dependents) only once it has SEEN the next chunk ready -- so the
    //     next launch, and the constant-cache invalidation that comes with it, happens after the bank was rewritten
    //     and after its previous readers were through; CTAs that start too early for that trigger by exiting;
    //   * everything a CTA reads from the previous launch (running totals, decisions) sits behind griddepcontrol.wait.
    __shared__ int s_next_ready, s_last;
    if (a.bank_wait_early) asm volatile("griddepcontrol.wait;" ::: "memory");
    if (a.bank_flags) {
        if (threadIdx.x == 0) {
            unsigned r;
            if (a.bank_spin) {   // never spins in practice (see above); a guard, not a synchronisation point
                do {
                    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(a.bank_flags + a.bank_id) : "memory");
                    if ((int)(r - a.bank_ticket) < 0) __nanosleep(200);
                } while ((int)(r - a.bank_ticket) < 0);
            }
            int nr = a.bank_next_known;
            if (!nr) {
                asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(a.bank_flags + (a.bank_id ^ 1)) : "memory");
                nr = (int)(r - (a.bank_ticket + 1u)) >= 0;
            }
            s_next_ready = nr;
        }
        __syncthreads();
        if (s_next_ready) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
    }
    const size_t ni = (size_t)a.ni;
    double *st = a.bank_state + d.i;   // SoA: component c of particle i at bank_state[c * ni + i]
    double *ist = st + REC * ni;       // parked i-state behind the REC running components
    typename P::IState I;
    if (a.bank_first) {
        P::load_i(a, d.i, I);
        if (d.i_valid && !a.bank_last) P::park_i(ist, ni, I);
    } else {
        P::unpark_i(a, ist, ni, d.i, I);
    }

    // The running totals are NOT live during the loop (they would cost 14-20 registers and a worse schedule:
    // 482 -> 502 Gpairs/s measured): the chunk is summed from zero and added to the parked totals afterwards,
    // which is also the two-level accumulation of the tiled sweeps (per-chunk partial sums, then the total).
    typename P::Acc tot;
    typename P::Part part;
    Dec D;
    if (a.bank_first) {
        D.template init<P::NN, P::NGB>(I.h2);
    } else {
        D.nn_d2 = CUDART_INF; D.nn_j = -1; D.cnt = 0;
        if (P::NN || P::NGB) {
            D.nn_d2 = st[10 * ni];
            const double pk = st[11 * ni];
            D.nn_j = __double2loint(pk);
            D.cnt = __double2hiint(pk);
        }
        D.template set_thr<P::NN, P::NGB>(I.h2);
    }
    part.zero();
    int *seg = P::NGB ? a.seg + (size_t)d.i * a.segcap : nullptr;

    const int cnt = a.bank_cnt, j0 = a.bank_j0;
    // A CTA that started before the next chunk was published (every CTA of a launch of one residency round or less:
    // they start while the last CTA of the previous launch is still refilling) looks again a few times on its way
    // through the chunk -- warp by warp, no barrier -- so that the next launch can move into the free CTA slots
    // instead of waiting for this CTA to exit.  Same condition as at the start, only observed later.
    // (a launch that waits for its predecessor right at its start gains nothing from being launched earlier)
    bool trig = a.bank_flags == nullptr || a.bank_wait_early || __ballot_sync(0xffffffffu, s_next_ready != 0) != 0u;   // warp-uniform
    constexpr int kLooks = (P::NN || P::NGB) ? 0 : kBankLooks;   // decision launches wait at their start: no looks compiled in
    constexpr int kLookEvery = P::kChunk / (kLooks + 1) / 8 * 8;
#pragma unroll P::kUnrollBank
    for (int k = 0; k < cnt; ++k) {
        if (kLooks > 0 && k > 0 && k % kLookEvery == 0 && !trig) {
            unsigned r;
            asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(r) : "l"(a.bank_flags + (a.bank_id ^ 1)) : "memory");
            if (__ballot_sync(0xffffffffu, (int)(r - (a.bank_ticket + 1u)) >= 0) != 0u) {
                trig = true;
                asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
            }
        }
        typename P::JData J;
        P::load_j_bank(k, J);
        P::template interact<1, false>(J, true, j0 + k, I, part, D, d, seg, a.segcap);
    }
    if (a.bank_flags) {
        // the last CTA through its loop refills this bank with the chunk after next (through the bank's address in
        // global memory) and publishes it
        __syncthreads();
        if (threadIdx.x == 0) {
            const unsigned prev = atomicAdd(a.bank_flags + 4 + a.bank_id, 1u);
            s_last = prev == gridDim.x - 1;
            if (s_last) a.bank_flags[4 + a.bank_id] = 0u;
        }
        __syncthreads();
        if (s_last && a.bank_next_cnt > 0) {
            double2 *dst = a.bank_self;
#pragma unroll
            for (int p = 0; p < P::NPL; ++p) {
                const double2 *src = static_cast<const double2 *>(a.jp[p]) + a.bank_next_j0;
                for (int k = threadIdx.x; k < a.bank_next_cnt; k += THREADS) dst[p * P::kChunk + k] = __ldcg(src + k);
            }
            __threadfence();
            __syncthreads();
            if (threadIdx.x == 0)
                asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(a.bank_flags + a.bank_id), "r"(a.bank_ticket + 2u) : "memory");
        }
        // CTAs that did not see the next chunk ready at their start let the next launch go by exiting: that is behind
        // their griddepcontrol.wait, i.e. after the previous launch (whose last CTA refills the next bank) has completed
    }
    if (a.bank_first) {
        tot.zero();
    } else {
        if (!a.bank_wait_early) asm volatile("griddepcontrol.wait;" ::: "memory");   // the previous chunk's totals
        double o[10];
#pragma unroll
        for (int c = 0; c < NC; ++c) o[c] = st[c * ni];
        tot.from_f64(o);
    }
    tot.add(part);
    if (!d.i_valid) return;

    double out[10];
    tot.to_f64(out);
    if (!a.bank_last) {
#pragma unroll
        for (int c = 0; c < NC; ++c) st[c * ni] = out[c];
        if (P::NN || P::NGB) {
            st[10 * ni] = D.nn_d2;
            st[11 * ni] = __hiloint2double(D.cnt, D.nn_j);
        }
        return;
    }
    int nn = D.nn_j;
    if (P::NN && nn >= 0) nn = __double2loint(a.jid_plane[nn].y);
    if (P::NGB && D.cnt > a.ngb_cap) *a.overflow_flag = 1;
    double2 *r2 = reinterpret_cast<double2 *>(a.rec + (size_t)d.i * REC);
    r2[0] = make_double2(out[0], out[1]);
    r2[1] = make_double2(out[2], out[3]);
    r2[2] = make_double2(out[4], out[5]);
    r2[3] = make_double2(out[6], D.nn_d2);
    r2[4] = make_double2(__hiloint2double(D.cnt, nn), out[7]);
    r2[5] = make_double2(out[8], out[9]);
}

template <class P>
static cudaError_t launch_bank(const ForceArgs &a, cudaStream_t st, int *geom)
{
    if (geom) { geom[0] = P::kChunk; geom[1] = P::kBankThreads; geom[2] = P::kMinBlocksBank; return cudaSuccess; }
    cudaLaunchConfig_t cfg = {};
    // the 128-thread instance exists for the plain 4th-order sweep only (s2_api.cu asks for it at mid-sized i-lists)
    constexpr bool kHasSmall = P::ORDER == 4 && !P::NN && !P::NGB && P::kBankThreads == 256;
    const int threads = (kHasSmall && a.bank_threads == 128) ? 128 : P::kBankThreads;
    cfg.gridDim = dim3((a.ni + threads - 1) / threads);
    cfg.blockDim = dim3(threads);
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = a.bank_pdl ? 1 : 0;
    if constexpr (kHasSmall)
        if (threads == 128) return cudaLaunchKernelEx(&cfg, force_sweep_bank_kernel<P, S2_BANK_ID, 128>, a);
    return cudaLaunchKernelEx(&cfg, force_sweep_bank_kernel<P, S2_BANK_ID, P::kBankThreads>, a);
}

// geom != nullptr: only report {chunk length of this order's bank layout, threads per CTA, CTAs per SM aimed at}
cudaError_t S2_CAT(dispatch_force_fp64_bank, S2_BANK_ID)(int order, unsigned flags, const ForceArgs &a, cudaStream_t st, int *geom)
{
    const bool ngb = flags & S2_WANT_NGB, nn = (flags & S2_WANT_NN) || ngb;
    if (order == 2) {
        if (ngb) return launch_bank<PolicyF64<2, true, true>>(a, st, geom);
        if (nn) return launch_bank<PolicyF64<2, true, false>>(a, st, geom);
        return launch_bank<PolicyF64<2, false, false>>(a, st, geom);
    }
    if (order == 4) {
        if (ngb) return launch_bank<PolicyF64<4, true, true>>(a, st, geom);
        if (nn) return launch_bank<PolicyF64<4, true, false>>(a, st, geom);
        return launch_bank<PolicyF64<4, false, false>>(a, st, geom);
    }
    if (ngb) return launch_bank<PolicyF64<6, true, true>>(a, st, geom);
    if (nn) return launch_bank<PolicyF64<6, true, false>>(a, st, geom);
    return launch_bank<PolicyF64<6, false, false>>(a, st, geom);
}

// device address of the constant bank (target of the per-chunk device-to-device copies)
cudaError_t S2_CAT(force_bank_address, S2_BANK_ID)(void **p) { return cudaGetSymbolAddress(p, c_jbank); }

}  // namespace s2
