// s2_bts_correct.cuh -- corrector and time-step rule of the block-time-step integrator for ONE active particle
// (sec 3.7; the schemes the paper names: 4th-order Hermite ref [27], 6th-order ref [5]).  Called by
// bts_correct_kernel (s2_bts.cu), one thread per active particle, and by lane 0 of reduce_kernel (s2_reduce.cu) right after
// it has written the particle's final force record -- which saves the corrector's launch in the usual block step.
#pragma once

#include "s2_internal.h"

namespace s2 {

__device__ __forceinline__ double pow2_floor(double x)   // largest power of two <= x, x > 0 finite
{
    return __hiloint2double(__double2hiint(x) & 0xfff00000, 0);
}
__device__ __forceinline__ double pow2_inv(double p)     // 1 / p for p a (normal) power of two: exact, and no division
{
    return __hiloint2double(0x7fe00000 - __double2hiint(p), 0);
}
__device__ __forceinline__ int level_of(double dt)       // dt = 2^-level
{
    return 1023 - ((__double2hiint(dt) >> 20) & 0x7ff);
}
__device__ __forceinline__ double norm3(const double a[3]) { return sqrt(a[0] * a[0] + a[1] * a[1] + a[2] * a[2]); }

// new step from the raw criterion value: power of two, at most doubled, doubled only at an even block boundary
__device__ __forceinline__ double next_step(double raw, double old, double t_new, double dt_min, double dt_max)
{
    double nw = fmin(pow2_floor(fmax(raw, dt_min)), 2.0 * old);
    if (nw > old) {
        const double x = t_new * (0.5 * pow2_inv(old));  // t_new / (2 old), exact: the step is a power of two
        if (x != floor(x)) nw = old;
    }
    return fmin(fmax(nw, dt_min), dt_max);
}


// 4th order (ref [27]):  v1 = v0 + (a0 + a1) dt/2 + (j0 - j1) dt^2/12;  x1 = x0 + (v0 + v1) dt/2 + (a0 - a1) dt^2/12
//   s0 = (-6 (a0 - a1) - dt (4 j0 + 2 j1)) / dt^2,  c0 = (12 (a0 - a1) + 6 dt (j0 + j1)) / dt^3,  s1 = s0 + c0 dt
//   dt' = sqrt(eta (|a1| |s1| + |j1|^2) / (|j1| |c0| + |s1|^2))                                   (Aarseth criterion)
// 6th order (ref [5]), h = dt/2, A+- = a1 +- a0, J+- = h (j1 +- j0), S+- = h^2 (s1 +- s0):
//   v1 = v0 + h (A+ - 2/5 J- + 1/15 S+);  x1 = x0 + h (v1 + v0) - 2/5 h^2 A- + h^3/15 (j1 + j0)
//   F5 = (S- - 3 J+ + 3 A-)/16, F4 = (S+ - J-)/16, F3 = (5 J+ - 5 A- - S-)/8
//   a3 = 6 (F3 + 4 F4 + 10 F5)/h^3 (stored as crackle), a4 = 24 (F4 + 5 F5)/h^4, a5 = 120 F5/h^5
//   dt' = eta (A1 / A4)^(1/3),  A1 = sqrt(|a1||s1| + |j1|^2),  A4 = sqrt(|a3||a5| + |a4|^2)
// k: position in the active list (bts_correct_one); r: the final force record of that particle.  Reads the particle's old state from the
// base j-store, writes the corrected state, its time and its new step in place, and keeps the step-level histogram.
// a particle's state at the start of its step, as the corrector needs it
struct BtsOld {
    double dt, x0[3], v0[3], a0[3], j0[3], s0[3];
};
// (loads that bypass L1: the small-step kernel corrects particles that other SMs corrected steps before)
__device__ __forceinline__ void bts_load_old(const BtsArgs &a, int i, BtsOld &o)
{
    o.dt = __ldcg(a.dt + i);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        o.x0[c] = __ldcg(a.f[2 + c] + i); o.v0[c] = __ldcg(a.f[5 + c] + i); o.a0[c] = __ldcg(a.f[8 + c] + i); o.j0[c] = __ldcg(a.f[11 + c] + i);
        o.s0[c] = a.order == 6 ? __ldcg(a.f[14 + c] + i) : 0.0;
    }
}

// i: address of the particle; t_new: the block time it is corrected to; o: its old state; r: its final force record
__device__ __forceinline__ void bts_correct_from(const BtsArgs &a, int i, double t_new, const BtsOld &o, const double *r)
{
    const double dt = o.dt;
    double x0[3], v0[3], a0[3], j0[3], a1[3], j1[3], x1[3], v1[3];
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        x0[c] = o.x0[c]; v0[c] = o.v0[c]; a0[c] = o.a0[c]; j0[c] = o.j0[c];
        a1[c] = r[c]; j1[c] = r[3 + c];
    }
    double raw;
    if (a.order != 6) {
        double s1[3], c0[3];
        // (divisions by powers of the step are multiplications by exact reciprocals: same bits, a tenth of the latency)
        const double h = 0.5 * dt, d2 = dt * dt, idt = pow2_inv(dt), id2 = idt * idt, id3 = id2 * idt;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            v1[c] = v0[c] + (a0[c] + a1[c]) * h + (j0[c] - j1[c]) * (d2 / 12.0);
            x1[c] = x0[c] + (v0[c] + v1[c]) * h + (a0[c] - a1[c]) * (d2 / 12.0);
            const double s0 = (-6.0 * (a0[c] - a1[c]) - dt * (4.0 * j0[c] + 2.0 * j1[c])) * id2;
            c0[c] = (12.0 * (a0[c] - a1[c]) + 6.0 * dt * (j0[c] + j1[c])) * id3;
            s1[c] = s0 + c0[c] * dt;
        }
        const double an = norm3(a1), jn = norm3(j1), sn = norm3(s1), cn = norm3(c0);
        raw = sqrt(a.eta * (an * sn + jn * jn) / fmax(jn * cn + sn * sn, 1e-300));
    } else {
        double s1[3], c1[3], p1[3], q1[3];
        const double h = 0.5 * dt, h2 = h * h, h3 = h2 * h, ih = pow2_inv(h), ih2 = ih * ih, ih3 = ih2 * ih, ih4 = ih2 * ih2, ih5 = ih2 * ih3;
#pragma unroll
        for (int c = 0; c < 3; ++c) {
            const double s0 = o.s0[c];
            s1[c] = r[9 + c];
            const double Ap = a1[c] + a0[c], Am = a1[c] - a0[c];
            const double Jp = h * (j1[c] + j0[c]), Jm = h * (j1[c] - j0[c]);
            const double Sp = h2 * (s1[c] + s0), Sm = h2 * (s1[c] - s0);
            v1[c] = v0[c] + h * (Ap - 0.4 * Jm + Sp / 15.0);
            x1[c] = x0[c] + h * (v1[c] + v0[c]) - 0.4 * h2 * Am + (h3 / 15.0) * (j1[c] + j0[c]);
            const double F5 = (Sm - 3.0 * Jp + 3.0 * Am) / 16.0, F4 = (Sp - Jm) / 16.0, F3 = (5.0 * Jp - 5.0 * Am - Sm) / 8.0;
            c1[c] = 6.0 * (F3 + 4.0 * F4 + 10.0 * F5) * ih3;
            p1[c] = 24.0 * (F4 + 5.0 * F5) * ih4;
            q1[c] = 120.0 * F5 * ih5;
            a.f[14 + c][i] = s1[c];
            a.f[17 + c][i] = c1[c];
        }
        const double A1 = sqrt(norm3(a1) * norm3(s1) + norm3(j1) * norm3(j1));
        const double A4 = sqrt(norm3(c1) * norm3(q1) + norm3(p1) * norm3(p1));
        raw = a.eta * cbrt(A1 / fmax(A4, 1e-300));
        if (a.averaged) {
            // the generalised criterion "is unstable when the force computation is not accurate enough",
            // so the paper's runs take "the average of the Aarseth fourth order method and the sixth order extension"
            const double jn = norm3(j1), sn = norm3(s1), cn = norm3(c1);
            const double raw4 = sqrt(a.eta4 * (norm3(a1) * sn + jn * jn) / fmax(jn * cn + sn * sn, 1e-300));
            raw = 0.5 * (raw + raw4);
        }
    }
    const double nw = next_step(raw, dt, t_new, a.dt_min, a.dt_max);
#pragma unroll
    for (int c = 0; c < 3; ++c) {
        a.f[2 + c][i] = x1[c]; a.f[5 + c][i] = v1[c]; a.f[8 + c][i] = a1[c]; a.f[11 + c][i] = j1[c];
    }
    a.f[0][i] = t_new;
    a.pot[i] = r[6];
    if (nw != dt) {
        a.dt[i] = nw;
        atomicSub(&a.hist[level_of(dt)], 1);     // integer atomics: the histogram does not depend on their order
        atomicAdd(&a.hist[level_of(nw)], 1);
    }
}

__device__ __forceinline__ void bts_correct_particle(const BtsArgs &a, int i, double t_new, const double *r)
{
    BtsOld o;
    bts_load_old(a, i, o);
    bts_correct_from(a, i, t_new, o, r);
}

__device__ __forceinline__ void bts_correct_one(const BtsArgs &a, int k, const double *r)
{
    bts_correct_particle(a, a.ilist[k], a.ctl->t_next, r);
}

}  // namespace s2
