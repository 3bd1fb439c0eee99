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
#include "s2_force_sweep.cuh"

namespace s2 {

__device__ __forceinline__ double rsqrt_seed(double s)
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(s));
    return y;
}

template <int ORDER_, bool NN_, bool NGB_>
struct PolicyF64 {
    static constexpr int ORDER = ORDER_;
    static constexpr bool NN = NN_, NGB = NGB_;
    // planes staged per tile: P0 P1 P2 P3 [P4 P5]; 2nd order (acc + pot only, GRAPE-5 style L34) needs no velocities:
    // P0 P1 P3 (P3 carries the id)
    static constexpr int NPL = ORDER == 6 ? 6 : (ORDER == 2 ? 3 : 4);
    static constexpr int kIdPlane = ORDER == 2 ? 2 : 3;
#ifndef S2_F64_MINBLOCKS
#define S2_F64_MINBLOCKS 2
#endif
#ifndef S2_F64_UNROLL
#define S2_F64_UNROLL 4
#endif
    static constexpr int kMinBlocks = S2_F64_MINBLOCKS;
    static constexpr int kUnroll = S2_F64_UNROLL;   // pairs in flight per thread in the one-lane-per-i loop
#ifndef S2_F64_UNROLL_TILED
#define S2_F64_UNROLL_TILED 4
#endif
#ifndef S2_F64_MINBLOCKS_TILED
#define S2_F64_MINBLOCKS_TILED 2
#endif
#ifndef S2_F64_MINBLOCKS_TILED6
#define S2_F64_MINBLOCKS_TILED6 1
#endif
#ifndef S2_F64_UNROLL_TILED6
#define S2_F64_UNROLL_TILED6 4
#endif
    static constexpr int kMinBlocksTiled = ORDER == 6 ? S2_F64_MINBLOCKS_TILED6 : S2_F64_MINBLOCKS_TILED;
    static constexpr int kIPT = kIptF64;                        // i-particles per thread in the register-tiled sweep
    // j per unrolled step there (x kIPT pairs in flight).  The 6th-order pair holds 18 more live doubles: with
    // 128 registers the totals spill inside the loop, so that variant runs one CTA per SM with 208 registers
    // (measured 290 vs 277 Gpairs/s)
    static constexpr int kUnrollTiled = ORDER == 6 ? S2_F64_UNROLL_TILED6 : S2_F64_UNROLL_TILED;

    struct IState {
        double x, y, z, vx, vy, vz, ax, ay, az, h2, eps2;
        int id;
    };

    struct Acc {
        double ax, ay, az, jx, jy, jz, pot, sx, sy, sz;
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

}  // namespace s2
