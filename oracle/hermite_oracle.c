/*
 * hermite_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU definition of what the hot path of
 * arXiv:1510.04068 (Sapporo2) computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may call this.  It shares
 * no code with the CUDA library (paper_1510_04068_b200/csrc) and neither
 * includes the other.
 *
 * What the paper fixes and what it does not:
 *   The paper prints no formula.  It names the operations:
 *     - "one kernel to predict the particles to the new time-step"      (sec 2.2.4)
 *     - 4th-order Hermite needs "the acceleration and the first time derivative
 *       of the acceleration (jerk)", "information of the nearest neighbouring
 *       particle", and "a list of particles within a given radius"     (L92, sec 3)
 *     - 6th-order Hermite (ref [5])                                     (L76, L140)
 *     - "nearest neighbours (particle-ID and distance)"                 (L174, sec 4.1)
 *   so this file writes out the textbook definitions those names refer to
 *   (readings P1-P18 are listed in DESIGN.md).
 *   The direct sum is exact (L28, L46): the oracle is the plain double loop,
 *   in long double (x87 80-bit, 64-bit significand), rounded to fp64 once.
 *
 * Parity pins (tests/test_oracle_pins.py): two-body closed form, circular-orbit
 * closed form, regular n-gon closed form, Newton's third law, finite-difference
 * jerk and snap along the predictor polynomials, exact rational evaluation of
 * the predictor, brute-force neighbour sets, integer-lattice ties; oracle_term_norms
 * on the circular two-body orbit, the rotating n-gon and a generic single pair.
 * Conventions P3-P9 versus the real Sapporo2 library: parity unpinned (the
 * library is not available and the paper does not state them).
 */
#include <float.h>
#include <math.h>
#include <stddef.h>
#include <stdlib.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#if LDBL_MANT_DIG < 64
#error "oracle needs an extended long double (>= 64-bit significand)"
#endif

typedef long double ld;

int oracle_ldbl_mant_dig(void) { return LDBL_MANT_DIG; }

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ---------------------------------------------------------------------------
 * O1 -- Taylor predictor ("predict"; reading P2).
 *   4th order:  x_p = x + dt (v + dt/2 (a + dt/3 j));      v_p = v + dt (a + dt/2 j)
 *   6th order:  x_p = x + dt (v + dt/2 (a + dt/3 (j + dt/4 (s + dt/5 c))))
 *               v_p = v + dt (a + dt/2 (j + dt/3 (s + dt/4 c)))
 *               a_p = a + dt (j + dt/2 (s + dt/3 c))
 * evaluated in long double, dt = t - t_j (any sign), rounded once to fp64.
 * Arrays are (n,3) row-major.  snap/crackle/ap may be NULL when order == 4.
 * ------------------------------------------------------------------------- */
void oracle_predict(int n, int order, double t, const double *tj,
                    const double *x, const double *v, const double *a, const double *jk,
                    const double *s, const double *c,
                    double *xp, double *vp, double *ap)
{
    for (int p = 0; p < n; ++p) {
        ld dt = (ld)t - (ld)tj[p];
        for (int k = 0; k < 3; ++k) {
            size_t q = (size_t)3 * p + k;
            if (order == 4) {
                ld X = (ld)x[q] + dt * ((ld)v[q] + dt / 2 * ((ld)a[q] + dt / 3 * (ld)jk[q]));
                ld V = (ld)v[q] + dt * ((ld)a[q] + dt / 2 * (ld)jk[q]);
                xp[q] = (double)X;
                vp[q] = (double)V;
                if (ap) ap[q] = a[q];
            } else {
                ld X = (ld)x[q] + dt * ((ld)v[q] + dt / 2 * ((ld)a[q] + dt / 3 * ((ld)jk[q]
                                  + dt / 4 * ((ld)s[q] + dt / 5 * (ld)c[q]))));
                ld V = (ld)v[q] + dt * ((ld)a[q] + dt / 2 * ((ld)jk[q] + dt / 3 * ((ld)s[q] + dt / 4 * (ld)c[q])));
                ld A = (ld)a[q] + dt * ((ld)jk[q] + dt / 2 * ((ld)s[q] + dt / 3 * (ld)c[q]));
                xp[q] = (double)X;
                vp[q] = (double)V;
                ap[q] = (double)A;
            }
        }
    }
}

/* ---------------------------------------------------------------------------
 * O3/O4 -- pair terms and per-i outputs.
 * For every j in address order 0..N-1 with id_j != id_i (self skipped by
 * identity for ALL outputs, reading P3):
 *     r = x_j - x_i ; v = v_j - v_i ; a = a_j - a_i (6th order)
 *     s     = r.r + eps2
 *     q     = m_j s^(-3/2)
 *     A0    = q r                                  acc  += A0
 *     alpha = (r.v)/s
 *     A1    = q v - 3 alpha A0                     jerk += A1
 *     beta  = (v.v + r.a)/s + alpha^2
 *     A2    = q a - 6 alpha A1 - 3 beta A0         snap += A2   (6th order)
 *     pot  -= m_j s^(-1/2)                          (P4, P5: softened, negative)
 *     d2    = r.r  (unsoftened, P4)
 *     nearest neighbour: strict <, first minimum in address order (P6)
 *     neighbour: d2 < h2_i, strict (P7)
 *
 * The two integer decisions (nearest neighbour, neighbour membership) are
 * taken on d2 evaluated in the CUDA path's decision precision (fp64):
 *     dx = fl(x_j - x_i) ...;  d2 = fma(dz, dz, fma(dy, dy, fl(dx*dx)))
 * (reading R-D2).  The decisions taken on the long-double d2 (the
 * oracle's own arithmetic, no formula shared with the kernels) are returned
 * as well: nn_addr_ld / nn_d2_ld (d2 rounded to fp64 once) and the neighbour
 * set ngb_count_ld / ngb_list_ld (rr < h2_i in long double).  The GPU parity
 * tests are judged against THESE, within north_star's band (nn: candidates
 * whose long-double d2 differ by <= 1e-12 relative; sets: pairs within 1e-12
 * relative of h2); equality with the fp64 decision is a secondary check.
 *
 * Inputs: (N,3) predicted arrays of the j-store; explicit i arrays (ni,3).
 * Outputs (any may be NULL): acc, jerk, snap (ni,3); pot, nn_d2 (ni);
 *   nn_addr = j address of the nearest neighbour (-1 if none), nn_id its id;
 *   ngb_count = true count; ngb_list (ni, ngb_cap) = the ngb_cap lowest
 *   addresses in ascending order (P8, P9), unused slots = -1.
 * ------------------------------------------------------------------------- */
void oracle_forces(int order, int N, const double *m, const int *id,
                   const double *xp, const double *vp, const double *ap,
                   int ni, const int *i_id, const double *xi, const double *vi, const double *ai,
                   const double *h2, double eps2,
                   double *acc, double *jerk, double *snap, double *pot,
                   int *nn_addr, int *nn_id, double *nn_d2, int *nn_addr_ld,
                   int *ngb_count, int *ngb_list, int ngb_cap,
                   double *nn_d2_ld, int *ngb_count_ld, int *ngb_list_ld)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int i = 0; i < ni; ++i) {
        ld A[3] = {0, 0, 0}, J[3] = {0, 0, 0}, S[3] = {0, 0, 0}, P = 0;
        double best = INFINITY;
        ld best_ld = INFINITY;
        int best_j = -1, best_j_ld = -1, cnt = 0, cnt_ld = 0;
        const double *Xi = xi + (size_t)3 * i, *Vi = vi + (size_t)3 * i;
        const double *Ai = (order == 6) ? ai + (size_t)3 * i : NULL;
        for (int j = 0; j < N; ++j) {
            if (id[j] == i_id[i]) continue;
            const double *Xj = xp + (size_t)3 * j, *Vj = vp + (size_t)3 * j;
            ld r[3], v[3], a[3] = {0, 0, 0};
            for (int k = 0; k < 3; ++k) {
                r[k] = (ld)Xj[k] - (ld)Xi[k];
                v[k] = (ld)Vj[k] - (ld)Vi[k];
                if (order == 6) a[k] = (ld)ap[(size_t)3 * j + k] - (ld)Ai[k];
            }
            ld rr = r[0] * r[0] + r[1] * r[1] + r[2] * r[2];
            ld s = rr + (ld)eps2;
            ld rinv = 1 / sqrtl(s);
            ld q = (ld)m[j] * rinv * rinv * rinv;
            ld alpha = (r[0] * v[0] + r[1] * v[1] + r[2] * v[2]) / s;
            ld A0[3], A1[3];
            for (int k = 0; k < 3; ++k) {
                A0[k] = q * r[k];
                A1[k] = q * v[k] - 3 * alpha * A0[k];
                A[k] += A0[k];
                J[k] += A1[k];
            }
            if (order == 6) {
                ld beta = (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]
                           + r[0] * a[0] + r[1] * a[1] + r[2] * a[2]) / s + alpha * alpha;
                for (int k = 0; k < 3; ++k)
                    S[k] += q * a[k] - 6 * alpha * A1[k] - 3 * beta * A0[k];
            }
            P -= (ld)m[j] * rinv;

            /* decisions: fp64 d2 with the stated operation order */
            double dx = Xj[0] - Xi[0], dy = Xj[1] - Xi[1], dz = Xj[2] - Xi[2];
            double d2 = fma(dz, dz, fma(dy, dy, dx * dx));
            if (d2 < best) { best = d2; best_j = j; }
            if (rr < best_ld) { best_ld = rr; best_j_ld = j; }
            if (h2 && rr < (ld)h2[i]) {
                if (ngb_list_ld && cnt_ld < ngb_cap) ngb_list_ld[(size_t)i * ngb_cap + cnt_ld] = j;
                ++cnt_ld;
            }
            if (h2 && d2 < h2[i]) {
                if (ngb_list && cnt < ngb_cap) ngb_list[(size_t)i * ngb_cap + cnt] = j;
                ++cnt;
            }
        }
        for (int k = 0; k < 3; ++k) {
            if (acc) acc[(size_t)3 * i + k] = (double)A[k];
            if (jerk) jerk[(size_t)3 * i + k] = (double)J[k];
            if (snap && order == 6) snap[(size_t)3 * i + k] = (double)S[k];
        }
        if (pot) pot[i] = (double)P;
        if (nn_addr) nn_addr[i] = best_j;
        if (nn_id) nn_id[i] = best_j >= 0 ? id[best_j] : -1;
        if (nn_d2) nn_d2[i] = best;
        if (nn_addr_ld) nn_addr_ld[i] = best_j_ld;
        if (ngb_count) ngb_count[i] = cnt;
        if (nn_d2_ld) nn_d2_ld[i] = (double)best_ld;
        if (ngb_count_ld) ngb_count_ld[i] = cnt_ld;
        if (ngb_list_ld)
            for (int k = cnt_ld; k < ngb_cap; ++k) ngb_list_ld[(size_t)i * ngb_cap + k] = -1;
        if (ngb_list)
            for (int k = cnt; k < ngb_cap; ++k) ngb_list[(size_t)i * ngb_cap + k] = -1;
    }
}

/* Sum over j of the Euclidean norms of the individual pair terms, per i (for the
 * symmetric-case error norm of reading P12: ||delta|| <= tol * sum_j ||term_j||), and
 * the root of the sum of their squares (racc, rjerk, rsnap; any may be NULL): the
 * scale of the rounding error of a sum whose terms are each evaluated to a fixed
 * relative accuracy (reading R-F32, the fp32 path's error norm). */
void oracle_term_norms(int order, int N, const double *m, const int *id,
                       const double *xp, const double *vp, const double *ap,
                       int ni, const int *i_id, const double *xi, const double *vi, const double *ai,
                       double eps2, double *nacc, double *njerk, double *nsnap,
                       double *racc, double *rjerk, double *rsnap)
{
#pragma omp parallel for schedule(dynamic, 8)
    for (int i = 0; i < ni; ++i) {
        ld NA = 0, NJ = 0, NS = 0, QA = 0, QJ = 0, QS = 0;
        for (int j = 0; j < N; ++j) {
            if (id[j] == i_id[i]) continue;
            ld r[3], v[3], a[3] = {0, 0, 0};
            for (int k = 0; k < 3; ++k) {
                r[k] = (ld)xp[(size_t)3 * j + k] - (ld)xi[(size_t)3 * i + k];
                v[k] = (ld)vp[(size_t)3 * j + k] - (ld)vi[(size_t)3 * i + k];
                if (order == 6) a[k] = (ld)ap[(size_t)3 * j + k] - (ld)ai[(size_t)3 * i + k];
            }
            ld s = r[0] * r[0] + r[1] * r[1] + r[2] * r[2] + (ld)eps2;
            ld rinv = 1 / sqrtl(s);
            ld q = (ld)m[j] * rinv * rinv * rinv;
            ld alpha = (r[0] * v[0] + r[1] * v[1] + r[2] * v[2]) / s;
            ld beta = (v[0] * v[0] + v[1] * v[1] + v[2] * v[2] + r[0] * a[0] + r[1] * a[1] + r[2] * a[2]) / s
                      + alpha * alpha;
            ld n0 = 0, n1 = 0, n2 = 0;
            for (int k = 0; k < 3; ++k) {
                ld A0 = q * r[k], A1 = q * v[k] - 3 * alpha * A0;
                ld A2 = q * a[k] - 6 * alpha * A1 - 3 * beta * A0;
                n0 += A0 * A0; n1 += A1 * A1; n2 += A2 * A2;
            }
            NA += sqrtl(n0); NJ += sqrtl(n1); NS += sqrtl(n2);
            QA += n0; QJ += n1; QS += n2;
        }
        if (nacc) nacc[i] = (double)NA;
        if (njerk) njerk[i] = (double)NJ;
        if (nsnap) nsnap[i] = (double)NS;
        if (racc) racc[i] = (double)sqrtl(QA);
        if (rjerk) rjerk[i] = (double)sqrtl(QJ);
        if (rsnap) rsnap[i] = (double)sqrtl(QS);
    }
}
