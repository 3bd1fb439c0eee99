// s2_force_ds.cu -- double-single pair arithmetic for the force sweep ("converted to ...
// double-single"; footnote 1 L198: two single-precision numbers giving ~14 significant digits; L132: the
// reciprocal square root starts from the special-function unit).
//
// Reading P11: a value is hi + lo with two floats (~48 bits).  To hold 1e-10 as a maximum over
// particles the WHOLE pair evaluation -- differences, s, the rsqrt refinement, every product -- and the
// accumulators run in double-single arithmetic built from error-free transformations (two-sum,
// fast-two-sum, FMA-based two-product).  Every operation below is an FP32-pipe instruction; nothing is
// evaluated in fp64 except the nearest-neighbour / neighbour decisions, which use the fp64 squared distance
// in every precision mode (planes P0, P1).
//
// j planes (float4 per particle): D0 (x_hi, x_lo, y_hi, y_lo)  D1 (z_hi, z_lo, m_hi, m_lo)
//   D2 (vx_hi, vx_lo, vy_hi, vy_lo)  D3 (vz_hi, vz_lo, id bits, 0)  [6th: D4 (ax_hi, ax_lo, ay_hi, ay_lo)
//   D5 (az_hi, az_lo, 0, 0)]  [NN/NGB: P0 (x, y)  P1 (z, m) as double2]
#include "s2_force_sweep.cuh"

namespace s2 {

struct ds {
    float hi, lo;
};

// The intrinsics (__fadd_rn, __fmul_rn, __fmaf_rn) are never contracted or re-associated by the compiler.
__device__ __forceinline__ ds two_sum(float a, float b)   // a + b = hi + lo exactly (6 ops)
{
    const float s = __fadd_rn(a, b);
    const float bb = __fsub_rn(s, a);
    const float e = __fadd_rn(__fsub_rn(a, __fsub_rn(s, bb)), __fsub_rn(b, bb));
    return {s, e};
}
__device__ __forceinline__ ds fast_two_sum(float a, float b)   // needs |a| >= |b| or a == 0 (3 ops)
{
    const float s = __fadd_rn(a, b);
    return {s, __fsub_rn(b, __fsub_rn(s, a))};
}
__device__ __forceinline__ ds ds_add(ds a, ds b)   // 11 ops
{
    ds s = two_sum(a.hi, b.hi);
    s.lo = __fadd_rn(s.lo, __fadd_rn(a.lo, b.lo));
    return fast_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ ds ds_neg(ds a) { return {-a.hi, -a.lo}; }
// a - b where the high parts may cancel almost completely (coordinate differences of a close pair): the
// renormalisation uses the full two-sum, so it stays exact when the low-part difference exceeds the high one
__device__ __forceinline__ ds ds_sub_cancel(ds a, ds b)   // 14 ops
{
    ds s = two_sum(a.hi, -b.hi);
    s.lo = __fadd_rn(s.lo, __fsub_rn(a.lo, b.lo));
    return two_sum(s.hi, s.lo);
}
__device__ __forceinline__ ds ds_mul(ds a, ds b)   // 7 ops
{
    const float p = __fmul_rn(a.hi, b.hi);
    float e = __fmaf_rn(a.hi, b.hi, -p);
    e = __fmaf_rn(a.hi, b.lo, e);
    e = __fmaf_rn(a.lo, b.hi, e);
    return fast_two_sum(p, e);
}
__device__ __forceinline__ ds ds_sqr(ds a)   // 7 ops
{
    const float p = __fmul_rn(a.hi, a.hi);
    float e = __fmaf_rn(a.hi, a.hi, -p);
    e = __fmaf_rn(__fadd_rn(a.hi, a.hi), a.lo, e);
    return fast_two_sum(p, e);
}
__device__ __forceinline__ ds ds_mul_f(ds a, float f)   // 6 ops
{
    const float p = __fmul_rn(a.hi, f);
    float e = __fmaf_rn(a.hi, f, -p);
    e = __fmaf_rn(a.lo, f, e);
    return fast_two_sum(p, e);
}
__device__ __forceinline__ ds ds_fma(ds a, ds b, ds c) { return ds_add(ds_mul(a, b), c); }   // a b + c
// c + a b for an accumulator c: the product (p, e) is added without being renormalised first (|e| <= a few ulp(p),
// which the low-part sum absorbs) -- 15 ops instead of 18
__device__ __forceinline__ ds ds_acc(ds c, ds a, ds b)
{
    const float p = __fmul_rn(a.hi, b.hi);
    float e = __fmaf_rn(a.hi, b.hi, -p);
    e = __fmaf_rn(a.hi, b.lo, e);
    e = __fmaf_rn(a.lo, b.hi, e);
    ds s = two_sum(c.hi, p);
    s.lo = __fadd_rn(s.lo, __fadd_rn(c.lo, e));
    return fast_two_sum(s.hi, s.lo);
}
__device__ __forceinline__ ds ds_from_double(double x)
{
    const float hi = __double2float_rn(x);
    return {hi, __double2float_rn(x - (double)hi)};
}
__device__ __forceinline__ ds ds_shfl_xor(ds a, int m)
{
    return {__shfl_xor_sync(0xffffffffu, a.hi, m), __shfl_xor_sync(0xffffffffu, a.lo, m)};
}

// s^(-1/2) in double-single: MUFU.RSQ seed y0 (<= 2^-22 relative), residual e = 1 - s y0^2 formed in
// double-single (y0^2 by an exact two-product), then y = y0 + y0 e (1/2 + 3 e / 8): relative error ~ e^3
// plus the 2^-46 rounding of the correction term.
__device__ __forceinline__ ds ds_rsqrt(ds s)
{
    float y0;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(y0) : "f"(s.hi));
    const float p = __fmul_rn(y0, y0);
    const ds y0sq = {p, __fmaf_rn(y0, y0, -p)};
    const ds t = ds_mul(s, y0sq);
    const float e = __fsub_rn(__fsub_rn(1.0f, t.hi), t.lo);   // 1 - t.hi is exact (t.hi in [1/2, 2])
    const float corr = __fmul_rn(__fmul_rn(y0, e), __fmaf_rn(0.375f, e, 0.5f));
    return fast_two_sum(y0, corr);
}

template <int ORDER_, bool NN_, bool NGB_>
struct PolicyDS {
    static constexpr int ORDER = ORDER_;
    static constexpr bool NN = NN_, NGB = NGB_;
    static constexpr bool DEC = NN || NGB;
    static constexpr int NQ = ORDER == 6 ? 6 : (ORDER == 2 ? 3 : 4);   // 2nd order stages D0, D1, D3 (D3 carries the id)
    static constexpr int kIdPlane = ORDER == 2 ? 2 : 3;
    static constexpr int NPL = NQ + (DEC ? 2 : 0);
    static constexpr int kMinBlocks = 2;
    static constexpr int kUnroll = 1;
    static constexpr int kIPT = kIptDS;          // no register tiling: a double-single pair is ~400 FP32 instructions
    static constexpr bool kPacked2 = false;

    struct IState {
        ds x, y, z, vx, vy, vz, ax, ay, az, eps2;
        double px, py, pz, h2;   // fp64 position for the decisions
        int id;
    };

    static constexpr bool kTrackW = false;
    struct Acc {
        ds ax, ay, az, jx, jy, jz, pot, sx, sy, sz;
        __device__ __forceinline__ double wq() const { return 0.0; }
        __device__ __forceinline__ void zero()
        {
            ax = ay = az = jx = jy = jz = pot = ds{0.f, 0.f};
            if (ORDER == 6) sx = sy = sz = ds{0.f, 0.f};
        }
        __device__ __forceinline__ void add(const Acc &o)
        {
            ax = ds_add(ax, o.ax); ay = ds_add(ay, o.ay); az = ds_add(az, o.az);
            jx = ds_add(jx, o.jx); jy = ds_add(jy, o.jy); jz = ds_add(jz, o.jz);
            pot = ds_add(pot, o.pot);
            if (ORDER == 6) { sx = ds_add(sx, o.sx); sy = ds_add(sy, o.sy); sz = ds_add(sz, o.sz); }
        }
        __device__ __forceinline__ void shfl_add(int m)
        {
            ax = ds_add(ax, ds_shfl_xor(ax, m)); ay = ds_add(ay, ds_shfl_xor(ay, m)); az = ds_add(az, ds_shfl_xor(az, m));
            jx = ds_add(jx, ds_shfl_xor(jx, m)); jy = ds_add(jy, ds_shfl_xor(jy, m)); jz = ds_add(jz, ds_shfl_xor(jz, m));
            pot = ds_add(pot, ds_shfl_xor(pot, m));
            if (ORDER == 6) {
                sx = ds_add(sx, ds_shfl_xor(sx, m)); sy = ds_add(sy, ds_shfl_xor(sy, m)); sz = ds_add(sz, ds_shfl_xor(sz, m));
            }
        }
        static __device__ __forceinline__ double val(ds a) { return (double)a.hi + (double)a.lo; }
        __device__ __forceinline__ void to_f64(double o[10]) const
        {
            o[0] = val(ax); o[1] = val(ay); o[2] = val(az); o[3] = val(jx); o[4] = val(jy); o[5] = val(jz);
            o[6] = val(pot);
            o[7] = ORDER == 6 ? val(sx) : 0.0; o[8] = ORDER == 6 ? val(sy) : 0.0; o[9] = ORDER == 6 ? val(sz) : 0.0;
        }
    };
    using Part = Acc;   // double-single per-tile sums, added to double-single totals

    static __device__ __forceinline__ void load_i(const ForceArgs &a, int i, IState &I)
    {
        const int ia = a.i_addr ? a.i_addr[i] : i;
        const float4 d0 = static_cast<const float4 *>(a.ip[0])[ia];
        const float4 d1 = static_cast<const float4 *>(a.ip[1])[ia];
        const float4 d3 = static_cast<const float4 *>(a.ip[kIdPlane])[ia];
        I.x = {d0.x, d0.y}; I.y = {d0.z, d0.w}; I.z = {d1.x, d1.y};
        if (ORDER != 2) {
            const float4 d2 = static_cast<const float4 *>(a.ip[2])[ia];
            I.vx = {d2.x, d2.y}; I.vy = {d2.z, d2.w}; I.vz = {d3.x, d3.y};
        }
        I.id = __float_as_int(d3.z);
        if (ORDER == 6) {
            const float4 d4 = static_cast<const float4 *>(a.ip[4])[ia];
            const float4 d5 = static_cast<const float4 *>(a.ip[5])[ia];
            I.ax = {d4.x, d4.y}; I.ay = {d4.z, d4.w}; I.az = {d5.x, d5.y};
        }
        if (DEC) {
            const double2 p0 = static_cast<const double2 *>(a.ip[NQ])[ia];
            const double2 p1 = static_cast<const double2 *>(a.ip[NQ + 1])[ia];
            I.px = p0.x; I.py = p0.y; I.pz = p1.x;
        }
        I.h2 = (NGB && a.h2) ? a.h2[i] : 0.0;
        I.eps2 = ds_from_double(a.eps2);
    }

    template <int L, bool MASKED>
    static __device__ __forceinline__ void pair(const unsigned char *stage, int tile, int k, bool valid, int jaddr,
                                                const IState &I, Part &A, Dec &D, const Decomp &d, int *seg,
                                                int segcap)
    {
        const float4 *pl = reinterpret_cast<const float4 *>(stage);
        const float4 d0 = pl[k], d1 = pl[tile + k], d2 = pl[2 * tile + k], d3 = ORDER == 2 ? d2 : pl[3 * tile + k];
        const bool skip = (__float_as_int(d3.z) == I.id) || (MASKED && !valid);

        const ds dx = ds_sub_cancel({d0.x, d0.y}, I.x), dy = ds_sub_cancel({d0.z, d0.w}, I.y),
                 dz = ds_sub_cancel({d1.x, d1.y}, I.z);
        if (DEC) {
            // fp64 decisions (reading P13), behind an fp32 prefilter on the one-lane-per-i path
            const float d2f = fmaf(dz.hi, dz.hi, fmaf(dy.hi, dy.hi, dx.hi * dx.hi));
            if (L > 1 || d2f < D.thrf) {
                const double2 *pd = reinterpret_cast<const double2 *>(stage);
                const double2 p0 = pd[NQ * tile + k], p1 = pd[(NQ + 1) * tile + k];
                const double ex = p0.x - I.px, ey = p0.y - I.py, ez = p1.x - I.pz;
                const double dd = __fma_rn(ez, ez, __fma_rn(ey, ey, __dmul_rn(ex, ex)));
                decide<L, NN, NGB>(dd, jaddr, skip, I.h2, D, d, seg, segcap);
            }
        }
        const ds m = {d1.z, d1.w};
        const ds s = ds_add(ds_add(ds_add(ds_sqr(dx), ds_sqr(dy)), ds_sqr(dz)), I.eps2);
        ds y = ds_rsqrt(s);
        if (skip) y = ds{0.f, 0.f};
        const ds y2 = ds_sqr(y);
        const ds my = ds_mul(m, y);
        const ds q = ds_mul(my, y2);
        A.pot = ds_add(A.pot, ds_neg(my));
        A.ax = ds_acc(A.ax, q, dx); A.ay = ds_acc(A.ay, q, dy); A.az = ds_acc(A.az, q, dz);
        if (ORDER == 2) return;
        const ds dvx = ds_sub_cancel({d2.x, d2.y}, I.vx), dvy = ds_sub_cancel({d2.z, d2.w}, I.vy),
                 dvz = ds_sub_cancel({d3.x, d3.y}, I.vz);
        const ds rv = ds_add(ds_add(ds_mul(dx, dvx), ds_mul(dy, dvy)), ds_mul(dz, dvz));
        const ds alpha = ds_mul(rv, y2);
        const ds a3 = ds_mul_f(alpha, -3.0f);
        const ds tx = ds_fma(a3, dx, dvx), ty = ds_fma(a3, dy, dvy), tz = ds_fma(a3, dz, dvz);
        A.jx = ds_acc(A.jx, q, tx); A.jy = ds_acc(A.jy, q, ty); A.jz = ds_acc(A.jz, q, tz);
        if (ORDER == 6) {
            const float4 d4 = pl[4 * tile + k], d5 = pl[5 * tile + k];
            const ds dax = ds_sub_cancel({d4.x, d4.y}, I.ax), day = ds_sub_cancel({d4.z, d4.w}, I.ay),
                     daz = ds_sub_cancel({d5.x, d5.y}, I.az);
            ds w = ds_add(ds_add(ds_sqr(dvx), ds_sqr(dvy)), ds_sqr(dvz));
            w = ds_add(w, ds_add(ds_add(ds_mul(dx, dax), ds_mul(dy, day)), ds_mul(dz, daz)));
            const ds b3 = ds_mul_f(ds_add(ds_mul(w, y2), ds_sqr(alpha)), -3.0f);
            const ds a6 = {a3.hi + a3.hi, a3.lo + a3.lo};   // exact doubling
            const ds ux = ds_add(ds_fma(a6, tx, ds_mul(b3, dx)), dax);
            const ds uy = ds_add(ds_fma(a6, ty, ds_mul(b3, dy)), day);
            const ds uz = ds_add(ds_fma(a6, tz, ds_mul(b3, dz)), daz);
            A.sx = ds_acc(A.sx, q, ux); A.sy = ds_acc(A.sy, q, uy); A.sz = ds_acc(A.sz, q, uz);
        }
    }
};

cudaError_t dispatch_force_ds(int order, unsigned flags, int L, dim3 grid, size_t smem, const ForceArgs &a,
                              cudaStream_t st, bool query, int *ctas_per_sm)
{
    const bool ngb = flags & S2_WANT_NGB, nn = (flags & S2_WANT_NN) || ngb;
    if (order == 2) {
        if (ngb) return launch_L<PolicyDS<2, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyDS<2, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyDS<2, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (order == 4) {
        if (ngb) return launch_L<PolicyDS<4, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
        if (nn) return launch_L<PolicyDS<4, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
        return launch_L<PolicyDS<4, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    }
    if (ngb) return launch_L<PolicyDS<6, true, true>>(L, grid, smem, a, st, query, ctas_per_sm);
    if (nn) return launch_L<PolicyDS<6, true, false>>(L, grid, smem, a, st, query, ctas_per_sm);
    return launch_L<PolicyDS<6, false, false>>(L, grid, smem, a, st, query, ctas_per_sm);
}

// Test hook (s2_test_ds_ops): every double-single primitive on n operand pairs, results as fp64.
__global__ void ds_ops_kernel(int n, const double *a, const double *b, double *out)
{
    const int k = blockIdx.x * blockDim.x + threadIdx.x;
    if (k >= n) return;
    const ds x = ds_from_double(a[k]), y = ds_from_double(b[k]);
    auto val = [](ds v) { return (double)v.hi + (double)v.lo; };
    double *o = out + (size_t)k * 8;
    o[0] = val(x);                              // fp64 -> DS -> fp64 round trip
    o[1] = val(ds_add(x, y));
    o[2] = val(ds_sub_cancel(x, y));
    o[3] = val(ds_mul(x, y));
    o[4] = val(ds_sqr(x));
    o[5] = val(ds_mul_f(x, -3.0f));
    o[6] = val(ds_rsqrt(ds{fabsf(x.hi), x.hi < 0.f ? -x.lo : x.lo}));   // of |a|
    o[7] = val(ds_acc(x, x, y));                // the accumulate form used by the sweep
}

cudaError_t run_ds_ops(int n, const double *d_a, const double *d_b, double *d_out, cudaStream_t st)
{
    if (n <= 0) return cudaSuccess;
    ds_ops_kernel<<<(n + 255) / 256, 256, 0, st>>>(n, d_a, d_b, d_out);
    return cudaGetLastError();
}

}  // namespace s2
