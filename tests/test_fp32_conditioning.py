"""Why the fp32 path re-evaluates ill-conditioned i-particles in fp64 (reading R-F32; s2_api.cu "fp32 fix-up";
GPU side: tests/test_gpu_precisions.py::test_fp32_fixup_meets_1e5_on_a_cancelling_sum).

north_star asks for 1e-5 in fp32.  Each fp32 pair term carries ~9 roundings of 2^-24 on the chain
r -> s -> s^(-1/2) -> m s^(-3/2), so the error of a particle's jerk is about 3e-7 * sqrt(sum_j ||term_j||^2), whatever the
total is.  Config 3 holds a particle (address 17198, found by the 4096-i GPU sample) whose jerk is the small remainder
of one strong pair term and the rest of the cluster.  This CPU test evaluates that particle's jerk with CORRECTLY ROUNDED
fp32 operations (numpy: every operation in fp64, rounded once to fp32 -- better than any hardware fp32 pipeline can
do, fused multiply-adds and an exactly rounded reciprocal square root included) in the formulation the fp32 kernel
uses (reading P10: (hi, lo) positions), with the sum of the terms taken exactly, and shows that it still misses
1e-5 of the total while sitting at ~2e-7 of the rms term.  No CUDA code is involved."""
import numpy as np

import oracle
from workloads import make_config

f32, f64 = np.float32, np.float64


def _r(x):
    return np.asarray(x, dtype=f64).astype(f32).astype(f64)


def _jerk_terms_fp32(i, xp, vp, mass, eps2):
    xh = _r(xp); xl = _r(xp - xh); vh = _r(vp); m = _r(mass)
    dx = _r(_r(xh - xh[i]) + _r(xl - xl[i]))
    dv = _r(vh - vh[i])
    e2 = float(f32(eps2))
    s = _r(dx[:, 2] * dx[:, 2] + _r(dx[:, 1] * dx[:, 1] + _r(dx[:, 0] * dx[:, 0] + e2)))
    y = _r(1.0 / np.sqrt(s)); y[i] = 0.0
    y2 = _r(y * y); q = _r(_r(m * y) * y2)
    rv = _r(dx[:, 2] * dv[:, 2] + _r(dx[:, 1] * dv[:, 1] + _r(dx[:, 0] * dv[:, 0])))
    a3 = _r(-3.0 * _r(rv * y2))
    t = np.stack([_r(a3 * dx[:, c] + dv[:, c]) for c in range(3)], 1)
    return q[:, None] * t          # products and the sum over j exact (fp64): only the per-term fp32 roundings remain


def test_correctly_rounded_fp32_misses_1e5_of_a_cancelling_sum():
    w = make_config(3)
    xp, vp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    i = 17198
    one = np.array([i], dtype=np.int32)
    ref = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, one, w.eps2)
    _, rj, _ = oracle.term_norms(4, w.mass, w.ident, xp, vp, None, w.ident[one], xp[one], vp[one], None, w.eps2, rms=True)
    _, nj, _ = oracle.term_norms(4, w.mass, w.ident, xp, vp, None, w.ident[one], xp[one], vp[one], None, w.eps2)
    J = np.linalg.norm(ref.jerk[0])
    assert 40 < rj[0] / J < 60 and nj[0] / J > 500           # rms cancellation ~48 : 1, sum of norms ~640 : 1
    got = _jerk_terms_fp32(i, xp, vp, w.mass, w.eps2).sum(0)
    err = np.linalg.norm(got - ref.jerk[0])
    assert err / J > 1e-5                                    # ideal fp32 arithmetic misses north_star's 1e-5 of the total ...
    assert err / rj[0] < 4e-7                                # ... at ~2.4e-7 of the rms pair term: ordinary fp32 rounding
    # the estimate the library flags with: sqrt(sum q^2) (|v_i| + v_esc) against 8 |jerk| -- this particle is flagged
    r = xp - xp[i]
    s_ = (r * r).sum(1) + w.eps2
    q = w.mass * s_ ** -1.5
    q[i] = 0.0
    est = np.sqrt((q * q).sum()) * (np.linalg.norm(vp[i]) + np.sqrt(2 * abs(ref.pot[0])))
    assert est > 8.0 * J and 0.4 < est / rj[0] < 8.0
    # a well-conditioned neighbour in the same sample: the plain criterion holds with a wide margin
    k = 9985
    onek = np.array([k], dtype=np.int32)
    refk = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, onek, w.eps2)
    gk = _jerk_terms_fp32(k, xp, vp, w.mass, w.eps2).sum(0)
    assert np.linalg.norm(gk - refk.jerk[0]) / np.linalg.norm(refk.jerk[0]) < 3e-6
