// s2_force_fp32.cu -- single-precision pair arithmetic for the force sweep (j-particles
// "converted to either float or double-single" on the device; L128-L132).
//
// Reading P10: "plain fp32" keeps every pair operation in fp32, but
//   (a) positions are held as (hi, lo) float pairs and r is formed as (hi_j - hi_i) + (lo_j - lo_i), so the
//       separation of a close pair does not inherit the 6e-8 |x| rounding of a float coordinate;
//   (b) a thread sums in fp32 only over one j tile (<= 256 terms); tile sums are added to fp64 totals;
//   (c) (reading R-F32) each pair term is good to ~4e-7, so the error of a sum is ~4e-7 sqrt(sum_j |term_j|^2) whatever
//       the total is; where a particle's jerk is a strongly cancelling sum no fp32 pair arithmetic reaches 1e-5 of the
//       total (tests/test_fp32_conditioning.py).  The sweep therefore also accumulates sum_j q_j^2 per i (one FFMA2 per
//       two pairs), and i-particles whose estimate sqrt(sum q^2) (|v_i| + v_esc) exceeds 8 |jerk_i| -- 0.3-0.8 % of a
//       Plummer sphere -- are re-evaluated by the fp64 sweep (s2_api.cu "fp32 fix-up").
// The two integer decisions (nearest neighbour, neighbour test) use the fp64 squared distance formed from
// the fp64 predicted positions (planes P0, P1 staged next to the float planes) in every precision mode.
//
// j planes (float4 per particle): F0 (x_hi, y_hi, z_hi, m)  F1 (x_lo, y_lo, z_lo, id bits)  F2 (vx, vy, vz, 0)
//                                 [6th order: F3 (ax, ay, az, 0)]  [NN/NGB: P0 (x, y) P1 (z, m) as double2]
#include "s2_force_sweep.cuh"

namespace s2 {

__device__ __forceinline__ float rsqrt_f32(float s)
{
    float y;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(s));   // MUFU.RSQ, <= 2^-22.4 relative
    return y;
}

// Packed fp32 pairs (sm_100a: FADD2 / FMUL2 / FFMA2, PTX add/mul/fma.rn.f32x2): one issue slot carries the same IEEE
// operation for two i-particles of a thread.  The FP32 pipe does not get wider (a packed instruction occupies it for
// two cycles), but the sweep is ISSUE-bound (33 FP32 + ~6 other slots per pair, FP32 pipe width = issue width), so
// halving the FP32 issue slots frees the scheduler for the loads, MUFU and selects.  Each element is rounded exactly
// like the scalar instruction, so the results keep the bits of the scalar sweeps.  A scalar operand that is the same
// for both halves (the j-particle) is written as a (v, v) pack, which ptxas turns into a broadcast operand (R.F32).
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pk2(float lo, float hi)
{
    f32x2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk2(f32x2 v, float &lo, float &hi) { asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ f32x2 bc2(float v) { return pk2(v, v); }
__device__ __forceinline__ f32x2 add2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b)
{
    f32x2 d;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b));
    return d;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c)
{
    f32x2 d;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c));
    return d;
}

template <int ORDER_, bool NN_, bool NGB_>
struct PolicyF32 {
    static constexpr int ORDER = ORDER_;
    static constexpr bool NN = NN_, NGB = NGB_;
    static constexpr bool DEC = NN || NGB;
    static constexpr int NQ = ORDER == 6 ? 4 : (ORDER == 2 ? 2 : 3);     // float planes (2nd order: F0, F1 only)
    static constexpr int NPL = NQ + (DEC ? 2 : 0);    // + fp64 position planes for the decisions
    static constexpr int kMinBlocks = 2;
    static constexpr int kUnroll = 4;
    static constexpr int kIPT = kIptF32;          // i-particles per thread in the register-tiled sweep
    static constexpr int kUnrollTiled = 4;
    static constexpr int kMinBlocksTiled = 2;

    struct IState {
        float xh, yh, zh, xl, yl, zl, vx, vy, vz, ax, ay, az, eps2;
        double x, y, z, h2;   // fp64 position for the decisions
        int id;
    };

    static constexpr bool kTrackW = ORDER != 2;   // sum of q^2 per i: conditioning estimate of the jerk sum (R-F32)
    struct Part {   // fp32 sums over one tile
        float ax, ay, az, jx, jy, jz, pot, sx, sy, sz;
        float w;    // sum of q^2 over the tile
        __device__ __forceinline__ void zero()
        {
            ax = ay = az = jx = jy = jz = pot = 0.f;
            w = 0.f;
            if (ORDER == 6) sx = sy = sz = 0.f;
        }
    };

    struct Acc {    // fp64 totals
        double ax, ay, az, jx, jy, jz, pot, sx, sy, sz;
        double w;
        __device__ __forceinline__ void zero()
        {
            ax = ay = az = jx = jy = jz = pot = 0.0;
            w = 0.0;
            if (ORDER == 6) sx = sy = sz = 0.0;
        }
        __device__ __forceinline__ void add(const Part &o)
        {
            ax += (double)o.ax; ay += (double)o.ay; az += (double)o.az;
            jx += (double)o.jx; jy += (double)o.jy; jz += (double)o.jz;
            pot += (double)o.pot;
            if (kTrackW) w += (double)o.w;
            if (ORDER == 6) { sx += (double)o.sx; sy += (double)o.sy; sz += (double)o.sz; }
        }
        __device__ __forceinline__ double wq() const { return w; }
        __device__ __forceinline__ void shfl_add(int m)
        {
            if (kTrackW) w += shfl_xor_d(w, m);
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

    static __device__ __forceinline__ void load_i(const ForceArgs &a, int i, IState &I)
    {
        const int ia = a.i_addr ? a.i_addr[i] : i;
        const float4 f0 = static_cast<const float4 *>(a.ip[0])[ia];
        const float4 f1 = static_cast<const float4 *>(a.ip[1])[ia];
        I.xh = f0.x; I.yh = f0.y; I.zh = f0.z;
        I.xl = f1.x; I.yl = f1.y; I.zl = f1.z;
        I.id = __float_as_int(f1.w);
        if (ORDER != 2) {
            const float4 f2 = static_cast<const float4 *>(a.ip[2])[ia];
            I.vx = f2.x; I.vy = f2.y; I.vz = f2.z;
        }
        if (ORDER == 6) {
            const float4 f3 = static_cast<const float4 *>(a.ip[3])[ia];
            I.ax = f3.x; I.ay = f3.y; I.az = f3.z;
        }
        if (DEC) {
            const double2 p0 = static_cast<const double2 *>(a.ip[NQ])[ia];
            const double2 p1 = static_cast<const double2 *>(a.ip[NQ + 1])[ia];
            I.x = p0.x; I.y = p0.y; I.z = p1.x;
        }
        I.h2 = (NGB && a.h2) ? a.h2[i] : 0.0;
        I.eps2 = (float)a.eps2;
    }

    struct JData {
        float4 f0, f1, f2, f3;
        double2 p0, p1;
    };
    static __device__ __forceinline__ void load_j(const unsigned char *stage, int tile, int k, JData &J)
    {
        const float4 *pl = reinterpret_cast<const float4 *>(stage);
        J.f0 = pl[k]; J.f1 = pl[tile + k];
        if (ORDER != 2) J.f2 = pl[2 * tile + k];
        if (ORDER == 6) J.f3 = pl[3 * tile + k];
        if (DEC) {
            const double2 *pd = reinterpret_cast<const double2 *>(stage);
            J.p0 = pd[NQ * tile + k]; J.p1 = pd[(NQ + 1) * tile + k];
        }
    }

    template <int L, bool MASKED>
    static __device__ __forceinline__ void pair(const unsigned char *stage, int tile, int k, bool valid, int jaddr,
                                                const IState &I, Part &A, Dec &D, const Decomp &d, int *seg,
                                                int segcap)
    {
        JData J;
        load_j(stage, tile, k, J);
        interact<L, MASKED>(J, valid, jaddr, I, A, D, d, seg, segcap);
    }

    template <int L, bool MASKED>
    static __device__ __forceinline__ void interact(const JData &J, bool valid, int jaddr, const IState &I, Part &A,
                                                    Dec &D, const Decomp &d, int *seg, int segcap)
    {
        const float4 f0 = J.f0, f1 = J.f1, f2 = J.f2;
        const bool skip = (__float_as_int(f1.w) == I.id) || (MASKED && !valid);

        const float dx = (f0.x - I.xh) + (f1.x - I.xl);
        const float dy = (f0.y - I.yh) + (f1.y - I.yl);
        const float dz = (f0.z - I.zh) + (f1.z - I.zl);
        float s;
        if (DEC) {
            // the decisions are taken on the fp64 d2 (reading P13), but only for pairs whose fp32 estimate comes
            // within the guard band of the rejection threshold (one-lane-per-i paths; L > 1 lanes vote together)
            const float d2f = fmaf(dz, dz, fmaf(dy, dy, dx * dx));
            s = d2f + I.eps2;
            if (L > 1 || d2f < D.thrf) {
                const double2 p0 = J.p0, p1 = J.p1;
                const double ex = p0.x - I.x, ey = p0.y - I.y, ez = p1.x - I.z;
                const double d2 = __fma_rn(ez, ez, __fma_rn(ey, ey, __dmul_rn(ex, ex)));
                decide<L, NN, NGB>(d2, jaddr, skip, I.h2, D, d, seg, segcap);
            }
        } else {
            s = fmaf(dz, dz, fmaf(dy, dy, fmaf(dx, dx, I.eps2)));
        }
        float y = rsqrt_f32(s);
        y = skip ? 0.f : y;
        const float y2 = y * y;
        const float my = f0.w * y;
        const float q = my * y2;
        A.pot -= my;
        A.ax = fmaf(q, dx, A.ax); A.ay = fmaf(q, dy, A.ay); A.az = fmaf(q, dz, A.az);
        if (ORDER == 2) return;
        A.w = fmaf(q, q, A.w);
        const float dvx = f2.x - I.vx, dvy = f2.y - I.vy, dvz = f2.z - I.vz;
        const float rv = fmaf(dz, dvz, fmaf(dy, dvy, dx * dvx));
        const float alpha = rv * y2;
        const float a3 = -3.f * alpha;
        const float tx = fmaf(a3, dx, dvx), ty = fmaf(a3, dy, dvy), tz = fmaf(a3, dz, dvz);
        A.jx = fmaf(q, tx, A.jx); A.jy = fmaf(q, ty, A.jy); A.jz = fmaf(q, tz, A.jz);
        if (ORDER == 6) {
            const float4 f3 = J.f3;
            const float dax = f3.x - I.ax, day = f3.y - I.ay, daz = f3.z - I.az;
            const float w = fmaf(dvx, dvx, fmaf(dvy, dvy, fmaf(dvz, dvz, fmaf(dx, dax, fmaf(dy, day, dz * daz)))));
            const float b3 = -3.f * fmaf(w, y2, alpha * alpha);
            const float a6 = a3 + a3;
            const float ux = fmaf(a6, tx, fmaf(b3, dx, dax));
            const float uy = fmaf(a6, ty, fmaf(b3, dy, day));
            const float uz = fmaf(a6, tz, fmaf(b3, dz, daz));
            A.sx = fmaf(q, ux, A.sx); A.sy = fmaf(q, uy, A.sy); A.sz = fmaf(q, uz, A.sz);
        }
    }

    // Two i-particles of one thread against the same j, every FP32 operation packed (see f32x2 above).  Same
    // operations in the same order as interact<1, false> for each half.
    static constexpr bool kPacked2 = true;
    static __device__ __forceinline__ void interact2(const JData &J, bool jvalid, int jaddr, const IState *I, Part *A, Dec *D,
                                                     const Decomp *d, int *const *seg, int segcap)
    {
        const float4 f0 = J.f0, f1 = J.f1, f2 = J.f2;
        const int jid = __float_as_int(f1.w);
        const bool skip0 = jid == I[0].id || !jvalid, skip1 = jid == I[1].id || !jvalid;   // jvalid: false on a masked tail lane

        const f32x2 dx = add2(sub2(bc2(f0.x), pk2(I[0].xh, I[1].xh)), sub2(bc2(f1.x), pk2(I[0].xl, I[1].xl)));
        const f32x2 dy = add2(sub2(bc2(f0.y), pk2(I[0].yh, I[1].yh)), sub2(bc2(f1.y), pk2(I[0].yl, I[1].yl)));
        const f32x2 dz = add2(sub2(bc2(f0.z), pk2(I[0].zh, I[1].zh)), sub2(bc2(f1.z), pk2(I[0].zl, I[1].zl)));
        f32x2 s;
        if (DEC) {
            const f32x2 d2f = fma2(dz, dz, fma2(dy, dy, mul2(dx, dx)));
            s = add2(d2f, bc2(I[0].eps2));
            float e0, e1;
            upk2(d2f, e0, e1);
            if (e0 < D[0].thrf || e1 < D[1].thrf) {
                const double2 p0 = J.p0, p1 = J.p1;
#pragma unroll
                for (int u = 0; u < 2; ++u) {
                    if ((u ? e1 : e0) < D[u].thrf) {
                        const double ex = p0.x - I[u].x, ey = p0.y - I[u].y, ez = p1.x - I[u].z;
                        const double d2 = __fma_rn(ez, ez, __fma_rn(ey, ey, __dmul_rn(ex, ex)));
                        decide<1, NN, NGB>(d2, jaddr, u ? skip1 : skip0, I[u].h2, D[u], d[u], seg[u], segcap);
                    }
                }
            }
        } else {
            s = fma2(dz, dz, fma2(dy, dy, fma2(dx, dx, bc2(I[0].eps2))));
        }
        float s0, s1;
        upk2(s, s0, s1);
        float y0 = rsqrt_f32(s0), y1 = rsqrt_f32(s1);
        y0 = skip0 ? 0.f : y0;
        y1 = skip1 ? 0.f : y1;
        const f32x2 y = pk2(y0, y1);
        const f32x2 y2 = mul2(y, y);
        const f32x2 my = mul2(bc2(f0.w), y);
        const f32x2 q = mul2(my, y2);
        f32x2 apot = pk2(A[0].pot, A[1].pot), aax = pk2(A[0].ax, A[1].ax), aay = pk2(A[0].ay, A[1].ay), aaz = pk2(A[0].az, A[1].az);
        apot = sub2(apot, my);
        aax = fma2(q, dx, aax); aay = fma2(q, dy, aay); aaz = fma2(q, dz, aaz);
        upk2(apot, A[0].pot, A[1].pot);
        upk2(aax, A[0].ax, A[1].ax); upk2(aay, A[0].ay, A[1].ay); upk2(aaz, A[0].az, A[1].az);
        if (ORDER == 2) return;
        {
            f32x2 aw = pk2(A[0].w, A[1].w);
            aw = fma2(q, q, aw);
            upk2(aw, A[0].w, A[1].w);
        }
        const f32x2 dvx = sub2(bc2(f2.x), pk2(I[0].vx, I[1].vx));
        const f32x2 dvy = sub2(bc2(f2.y), pk2(I[0].vy, I[1].vy));
        const f32x2 dvz = sub2(bc2(f2.z), pk2(I[0].vz, I[1].vz));
        const f32x2 rv = fma2(dz, dvz, fma2(dy, dvy, mul2(dx, dvx)));
        const f32x2 alpha = mul2(rv, y2);
        const f32x2 a3 = mul2(bc2(-3.f), alpha);
        const f32x2 tx = fma2(a3, dx, dvx), ty = fma2(a3, dy, dvy), tz = fma2(a3, dz, dvz);
        f32x2 ajx = pk2(A[0].jx, A[1].jx), ajy = pk2(A[0].jy, A[1].jy), ajz = pk2(A[0].jz, A[1].jz);
        ajx = fma2(q, tx, ajx); ajy = fma2(q, ty, ajy); ajz = fma2(q, tz, ajz);
        upk2(ajx, A[0].jx, A[1].jx); upk2(ajy, A[0].jy, A[1].jy); upk2(ajz, A[0].jz, A[1].jz);
        if (ORDER == 6) {
            const float4 f3 = J.f3;
            const f32x2 dax = sub2(bc2(f3.x), pk2(I[0].ax, I[1].ax));
            const f32x2 day = sub2(bc2(f3.y), pk2(I[0].ay, I[1].ay));
            const f32x2 daz = sub2(bc2(f3.z), pk2(I[0].az, I[1].az));
            const f32x2 w = fma2(dvx, dvx, fma2(dvy, dvy, fma2(dvz, dvz, fma2(dx, dax, fma2(dy, day, mul2(dz, daz))))));
            const f32x2 b3 = mul2(bc2(-3.f), fma2(w, y2, mul2(alpha, alpha)));
            const f32x2 a6 = add2(a3, a3);
            const f32x2 ux = fma2(a6, tx, fma2(b3, dx, dax));
            const f32x2 uy = fma2(a6, ty, fma2(b3, dy, day));
            const f32x2 uz = fma2(a6, tz, fma2(b3, dz, daz));
            f32x2 asx = pk2(A[0].sx, A[1].sx), asy = pk2(A[0].sy, A[1].sy), asz = pk2(A[0].sz, A[1].sz);
            asx = fma2(q, ux, asx); asy = fma2(q, uy, asy); asz = fma2(q, uz, asz);
            upk2(asx, A[0].sx, A[1].sx); upk2(asy, A[0].sy, A[1].sy); upk2(asz, A[0].sz, A[1].sz);
        }
    }
};

cudaError_t dispatch_force_fp32(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                                cudaStream_t st, bool query, int *ctas_per_sm)
{
    const bool ngb = flags & S2_WANT_NGB, nn = (flags & S2_WANT_NN) || ngb;
    if (order == 2) {
        if (ngb) return launch_L<PolicyF32<2, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyF32<2, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyF32<2, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (order == 4) {
        if (ngb) return launch_L<PolicyF32<4, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyF32<4, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyF32<4, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (ngb) return launch_L<PolicyF32<6, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
    if (nn) return launch_L<PolicyF32<6, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    return launch_L<PolicyF32<6, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
}

}  // namespace s2
