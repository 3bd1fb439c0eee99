// s2_predict.cuh -- the Taylor predictor of one j-particle (a2), shared by predict_kernel (s2_store.cu) and the
// block-step integrator's select kernel (s2_bts.cu), which predicts the j-store to the next block time in the same
// launch that finds that time.
// Predictor (reading P2), Horner form, fp64 FMA:
//   4th: x_p = x + dt (v + dt/2 (a + dt/3 j));                 v_p = v + dt (a + dt/2 j)
//   6th: x_p = x + dt (v + dt/2 (a + dt/3 (j + dt/4 (s + dt/5 c))))
//        v_p = v + dt (a + dt/2 (j + dt/3 (s + dt/4 c)));      a_p = a + dt (j + dt/2 (s + dt/3 c))
// One thread per j: 14 (20) coalesced 8-byte reads + id, 4 (6) coalesced 16-byte plane writes,
// plus the float / double-single planes when the context computes in those precisions.
#pragma once

#include "s2_internal.h"

namespace s2 {

__device__ __forceinline__ float2 split_ds(double x)
{
    float hi = __double2float_rn(x);
    float lo = __double2float_rn(x - (double)hi);
    return make_float2(hi, lo);
}

// the Taylor series alone; f(k) returns base field k of the particle (t, m, x[3], v[3], a[3], jerk[3] [, snap[3], crackle[3]])
template <int ORDER, class F>
__device__ __forceinline__ void predict_state(F f, double t, double xp[3], double vp[3], double ap[3])
{
    const double dt = t - f(0);
    const double h2 = 0.5 * dt, h3 = dt * (1.0 / 3.0);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        const double x = f(2 + c), v = f(5 + c), ac = f(8 + c), jk = f(11 + c);
        if (ORDER == 4) {
            xp[c] = fma(dt, fma(h2, fma(h3, jk, ac), v), x);
            vp[c] = fma(dt, fma(h2, jk, ac), v);
            ap[c] = ac;
        } else {
            const double s = f(14 + c), cr = f(17 + c);
            const double h4 = 0.25 * dt, h5 = 0.2 * dt;
            xp[c] = fma(dt, fma(h2, fma(h3, fma(h4, fma(h5, cr, s), jk), ac), v), x);
            vp[c] = fma(dt, fma(h2, fma(h3, fma(h4, cr, s), jk), ac), v);
            ap[c] = fma(dt, fma(h2, fma(h3, cr, s), jk), ac);
        }
    }
}

template <int ORDER>
__device__ __forceinline__ void predict_one(const PredictArgs &a, int j, double t)
{
    const double m = a.f[1][j];
    const int id = a.id[j];
    double xp[3], vp[3], ap[3];
    predict_state<ORDER>([&](int k) { return a.f[k][j]; }, t, xp, vp, ap);
    const double idbits = __hiloint2double(0, id);
    a.p[0][j] = make_double2(xp[0], xp[1]);
    a.p[1][j] = make_double2(xp[2], m);
    a.p[2][j] = make_double2(vp[0], vp[1]);
    a.p[3][j] = make_double2(vp[2], idbits);
    if (ORDER == 6) {
        a.p[4][j] = make_double2(ap[0], ap[1]);
        a.p[5][j] = make_double2(ap[2], 0.0);
    }
    if (a.precision == S2_FP32) {
        float2 X = split_ds(xp[0]), Y = split_ds(xp[1]), Z = split_ds(xp[2]);
        a.q[0][j] = make_float4(X.x, Y.x, Z.x, __double2float_rn(m));
        a.q[1][j] = make_float4(X.y, Y.y, Z.y, __int_as_float(id));
        a.q[2][j] = make_float4(__double2float_rn(vp[0]), __double2float_rn(vp[1]), __double2float_rn(vp[2]), 0.f);
        if (ORDER == 6)
            a.q[3][j] = make_float4(__double2float_rn(ap[0]), __double2float_rn(ap[1]), __double2float_rn(ap[2]), 0.f);
    } else if (a.precision == S2_DS) {
        float2 X = split_ds(xp[0]), Y = split_ds(xp[1]), Z = split_ds(xp[2]), M = split_ds(m);
        float2 U = split_ds(vp[0]), V = split_ds(vp[1]), W = split_ds(vp[2]);
        a.q[0][j] = make_float4(X.x, X.y, Y.x, Y.y);
        a.q[1][j] = make_float4(Z.x, Z.y, M.x, M.y);
        a.q[2][j] = make_float4(U.x, U.y, V.x, V.y);
        a.q[3][j] = make_float4(W.x, W.y, __int_as_float(id), 0.f);
        if (ORDER == 6) {
            float2 A = split_ds(ap[0]), B = split_ds(ap[1]), Cc = split_ds(ap[2]);
            a.q[4][j] = make_float4(A.x, A.y, B.x, B.y);
            a.q[5][j] = make_float4(Cc.x, Cc.y, 0.f, 0.f);
        }
    }
}

}  // namespace s2
