"""Pins for the CPU oracle (oracle/hermite_oracle.c) against things other than itself.

The paper prints no formula and no worked example, so the pins are
closed forms, high-precision numerical differentiation of the *definition*
A(t) = m r(t) (r.r + eps^2)^(-3/2), invariants, exact rational arithmetic and brute force
(SURVEY.md sec 8(c) "What pins each part").
"""
from decimal import Decimal, getcontext
from fractions import Fraction
import math

import numpy as np
import pytest

import oracle
from workloads import make_config, lattice_workload, A_PLUMMER

getcontext().prec = 80


# ----------------------------------------------------------------------------- helpers
def _one_pair(order, m, r, v, a, eps2):
    """oracle output for one sink at the origin at rest and one source at (r, v, a)."""
    z = np.zeros((1, 3))
    res = oracle.forces(order, np.array([m]), np.array([5], np.int32), np.array([r]), np.array([v]),
                        np.array([a]), np.array([9], np.int32), z, z, z, eps2)
    return res


def _dec_acc(m, r, v, a, eps2, t):
    """A(t) in 80-digit decimal arithmetic: the definition of the softened pair acceleration on
    the trajectory r(t) = r + v t + a t^2/2."""
    rt = [Decimal(r[k]) + Decimal(v[k]) * t + Decimal(a[k]) * t * t / 2 for k in range(3)]
    s = sum(x * x for x in rt) + Decimal(eps2)
    f = Decimal(m) / (s * s.sqrt())
    return [x * f for x in rt]


# ----------------------------------------------------------------------------- pair formulas
@pytest.mark.parametrize("seed", range(6))
def test_pair_jerk_snap_are_time_derivatives_of_acc(seed):
    """jerk = dA/dt, snap = d2A/dt2 at t = 0, by central differences in 80-digit arithmetic
    (step 1e-15 -> truncation ~1e-30): pins every sign, factor and term of O3."""
    rng = np.random.default_rng(seed)
    m = float(rng.uniform(0.1, 2.0))
    r, v, a = rng.normal(size=3), rng.normal(size=3), rng.normal(size=3)
    eps2 = float(rng.uniform(0.0, 0.3))
    res = _one_pair(6, m, r, v, a, eps2)
    h = Decimal(10) ** -15
    Ap, Am, A0 = _dec_acc(m, r, v, a, eps2, h), _dec_acc(m, r, v, a, eps2, -h), _dec_acc(m, r, v, a, eps2, Decimal(0))
    for k in range(3):
        acc = float(A0[k]); jerk = float((Ap[k] - Am[k]) / (2 * h)); snap = float((Ap[k] - 2 * A0[k] + Am[k]) / (h * h))
        assert res.acc[0, k] == pytest.approx(acc, rel=1e-15, abs=1e-17)
        assert res.jerk[0, k] == pytest.approx(jerk, rel=1e-14, abs=1e-16)
        assert res.snap[0, k] == pytest.approx(snap, rel=1e-14, abs=1e-15)
    s = Decimal(eps2) + sum(Decimal(x) ** 2 for x in r)
    assert res.pot[0] == pytest.approx(float(-Decimal(m) / s.sqrt()), rel=1e-15)
    # 4th-order call returns the same acc / jerk
    r4 = _one_pair(4, m, r, v, a, eps2)
    assert np.array_equal(r4.acc, res.acc) and np.array_equal(r4.jerk, res.jerk) and r4.snap is None


def test_circular_two_body_closed_form():
    """eps = 0, circular relative orbit of total mass M, separation R:
    r.v = 0 and v.v + r.a = 0, so acc = m r/R^3, jerk = m v/R^3, snap = m a/R^3 = -m M r/R^6."""
    m, M, R = 0.3, 1.7, 2.5
    r = np.array([R, 0.0, 0.0]); vc = math.sqrt(M / R)
    v = np.array([0.0, vc, 0.0]); a = -M * r / R ** 3
    res = _one_pair(6, m, r, v, a, 0.0)
    np.testing.assert_allclose(res.acc[0], m * r / R ** 3, rtol=1e-15, atol=1e-18)
    np.testing.assert_allclose(res.jerk[0], m * v / R ** 3, rtol=1e-15, atol=1e-18)
    np.testing.assert_allclose(res.snap[0], -m * M * r / R ** 6, rtol=1e-15, atol=1e-18)
    assert res.pot[0] == pytest.approx(-m / R, rel=1e-15)


@pytest.mark.parametrize("n", [3, 8, 17])
def test_ring_closed_form(n):
    """n equal masses on a regular n-gon of radius R rotating rigidly, eps = 0:
    inward acceleration (m / 4R^2) sum_k 1/sin(pi k / n); jerk = w x acc; snap = -w^2 acc."""
    m, R, w = 0.7 / n, 1.3, 0.9
    th = 2 * math.pi * np.arange(n) / n
    x = np.stack([R * np.cos(th), R * np.sin(th), np.zeros(n)], 1)
    v = np.stack([-w * x[:, 1], w * x[:, 0], np.zeros(n)], 1)
    a = -w * w * x
    ids = np.arange(n, dtype=np.int32)
    res = oracle.forces(6, np.full(n, m), ids, x, v, a, ids, x, v, a, 0.0)
    g = m / (4 * R * R) * sum(1 / math.sin(math.pi * k / n) for k in range(1, n))
    acc = -g * x / R
    np.testing.assert_allclose(res.acc, acc, rtol=1e-14, atol=1e-14 * g)   # inputs carry cos/sin rounding
    jerk = np.stack([-w * acc[:, 1], w * acc[:, 0], np.zeros(n)], 1)
    np.testing.assert_allclose(res.jerk, jerk, rtol=1e-13, atol=1e-13 * g * w)
    np.testing.assert_allclose(res.snap, -w * w * acc, rtol=1e-13, atol=1e-13 * g * w * w)
    potc = -m / (2 * R) * sum(1 / math.sin(math.pi * k / n) for k in range(1, n))
    np.testing.assert_allclose(res.pot, potc, rtol=1e-14)


def test_term_norms_closed_forms():
    """oracle_term_norms (the scale of the Newton's-third-law bound) is a second copy of the pair terms, so it gets
    its own pins.  Circular two-body orbit (eps = 0, r.v = 0, v.v + r.a = 0): ||A0|| = m / R^2, ||A1|| = m v / R^3,
    ||A2|| = m M / R^5.  Rigidly rotating regular n-gon: the pair (i, i + k) has separation d_k = 2 R sin(pi k / n),
    relative velocity w d_k perpendicular to it and relative acceleration -w^2 r, so alpha = beta = 0 and the norms are
    m / d_k^2, m w / d_k^2, m w^2 / d_k^2; sum_k 1 / sin^2(pi k / n) = (n^2 - 1) / 3."""
    m, M, R = 0.3, 1.7, 2.5
    r = np.array([[R, 0.0, 0.0]]); vc = math.sqrt(M / R)
    v = np.array([[0.0, vc, 0.0]]); a = -M * r / R ** 3
    z = np.zeros((1, 3))
    na, nj, ns = oracle.term_norms(6, np.array([m]), np.array([5], np.int32), r, v, a, np.array([9], np.int32), z, z, z, 0.0)
    assert na[0] == pytest.approx(m / R ** 2, rel=1e-15)
    assert nj[0] == pytest.approx(m * vc / R ** 3, rel=1e-15)
    assert ns[0] == pytest.approx(m * M / R ** 5, rel=1e-15)
    # a generic pair: the norms are those of the oracle's own single-pair outputs (which the 80-digit pins fix)
    rng = np.random.default_rng(3)
    r, v, a = rng.normal(size=(1, 3)), rng.normal(size=(1, 3)), rng.normal(size=(1, 3))
    one = _one_pair(6, m, r[0], v[0], a[0], 0.07)
    na, nj, ns = oracle.term_norms(6, np.array([m]), np.array([5], np.int32), r, v, a, np.array([9], np.int32), z, z, z, 0.07)
    ra, rj, rs = oracle.term_norms(6, np.array([m]), np.array([5], np.int32), r, v, a, np.array([9], np.int32), z, z, z, 0.07, rms=True)
    for got, got_rms, vec in ((na, ra, one.acc), (nj, rj, one.jerk), (ns, rs, one.snap)):
        assert got[0] == pytest.approx(np.linalg.norm(vec[0]), rel=1e-14)
        assert got_rms[0] == pytest.approx(np.linalg.norm(vec[0]), rel=1e-14)      # one term: both norms are its length
    for n in (3, 8, 17):
        m, R, w = 0.7 / n, 1.3, 0.9
        th = 2 * math.pi * np.arange(n) / n
        x = np.stack([R * np.cos(th), R * np.sin(th), np.zeros(n)], 1)
        vel = np.stack([-w * x[:, 1], w * x[:, 0], np.zeros(n)], 1)
        ids = np.arange(n, dtype=np.int32)
        na, nj, ns = oracle.term_norms(6, np.full(n, m), ids, x, vel, -w * w * x, ids, x, vel, -w * w * x, 0.0)
        base = m * (n * n - 1) / (12 * R * R)
        np.testing.assert_allclose(na, base, rtol=1e-13)
        np.testing.assert_allclose(nj, base * w, rtol=1e-12)
        np.testing.assert_allclose(ns, base * w * w, rtol=1e-12)
        # root of the sum of squares (reading R-F32): sum_k 1 / sin^4(pi k / n) = (n^2 - 1)(n^2 + 11) / 45
        ra, rj, rs = oracle.term_norms(6, np.full(n, m), ids, x, vel, -w * w * x, ids, x, vel, -w * w * x, 0.0, rms=True)
        rbase = m / (4 * R * R) * math.sqrt((n * n - 1) * (n * n + 11) / 45)
        np.testing.assert_allclose(ra, rbase, rtol=1e-13)
        np.testing.assert_allclose(rj, rbase * w, rtol=1e-12)
        np.testing.assert_allclose(rs, rbase * w * w, rtol=1e-12)
    # the 4th-order call returns the same acc / jerk norms (no snap terms needed)
    na4, nj4, _ = oracle.term_norms(4, np.full(n, m), ids, x, vel, None, ids, x, vel, None, 0.0)
    assert np.array_equal(na4, na) and np.array_equal(nj4, nj)


# ----------------------------------------------------------------------------- sums / invariants
def _predicted(w, order):
    return oracle.predict(order, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)


@pytest.mark.parametrize("order,cfg", [(4, 1), (6, 4)])
def test_newton_third_law_and_pot_symmetry(order, cfg):
    w = make_config(cfg, N=256)
    xp, vp, ap = _predicted(w, order)
    il = np.arange(w.N, dtype=np.int32)
    res = oracle.forces_ilist(order, w.mass, w.ident, xp, vp, ap, il, w.eps2)
    na, nj, ns = oracle.term_norms(order, w.mass, w.ident, xp, vp, ap, w.ident, xp, vp, ap, w.eps2)
    u = 2.0 ** -53
    for q, nq in ((res.acc, na), (res.jerk, nj)) + (((res.snap, ns),) if order == 6 else ()):
        tot = np.abs((w.mass[:, None] * q).sum(0)).max()
        assert tot <= 4 * w.N * u * (w.mass * nq).sum()
    # independent half-loop for the potential energy
    W = 0.0
    for i in range(w.N):
        d = xp[i + 1:] - xp[i]
        W -= (w.mass[i] * w.mass[i + 1:] / np.sqrt((d * d).sum(1) + w.eps2)).sum()
    assert (w.mass * res.pot).sum() == pytest.approx(2 * W, rel=1e-13)


def test_plummer_potential_energy_is_minus_half():
    """N-body units: W = -1/2 for a Plummer model (loose: sampling noise ~ few % at N = 1024)."""
    w = make_config(1)
    il = np.arange(w.N, dtype=np.int32)
    res = oracle.forces_ilist(4, w.mass, w.ident, w.pos, w.vel, None, il, w.eps2)
    assert 0.5 * (w.mass * res.pot).sum() == pytest.approx(-0.5, rel=0.08)
    # acceleration points inward on average: <a . x> < 0 and matches -W = sum m a.x (virial of the forces)
    vir = (w.mass[:, None] * res.acc * w.pos).sum()
    assert vir == pytest.approx(0.5 * (w.mass * res.pot).sum(), rel=0.02)


@pytest.mark.parametrize("order", [4, 6])
def test_finite_difference_jerk_snap_along_predictor(order):
    """Move every particle along its own predictor polynomial; jerk ~ dA/dt, snap ~ d2A/dt2 by
    5-point stencils of the oracle's own accelerations (ties predictor and pair terms together;
    4th-order predicted velocity is x_p', 6th-order a_p is x_p'')."""
    w = make_config(4, N=96)
    il = np.arange(w.N, dtype=np.int32)
    d = 2.0 ** -14

    def acc_at(t):
        xp, vp, ap = oracle.predict(order, t, w.t_j, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)
        return oracle.forces_ilist(order, w.mass, w.ident, xp, vp, ap, il, w.eps2 + 1e-3)

    t0 = w.t_pred
    A = {k: acc_at(t0 + k * d).acc for k in (-2, -1, 0, 1, 2)}
    ref = acc_at(t0)
    jerk_fd = (8 * (A[1] - A[-1]) - (A[2] - A[-2])) / (12 * d)
    err = np.linalg.norm(jerk_fd - ref.jerk, axis=1) / np.linalg.norm(ref.jerk, axis=1)
    assert err.max() < 2e-7
    if order == 6:
        snap_fd = (-A[2] + 16 * A[1] - 30 * A[0] + 16 * A[-1] - A[-2]) / (12 * d * d)
        err = np.linalg.norm(snap_fd - ref.snap, axis=1) / np.linalg.norm(ref.snap, axis=1)
        assert err.max() < 5e-5


# ----------------------------------------------------------------------------- predictor
@pytest.mark.parametrize("order", [4, 6])
def test_predictor_exact_rational(order):
    """The Taylor polynomial evaluated exactly with Fractions on the fp64 inputs, rounded once."""
    w = make_config(4, N=64)
    xp, vp, ap = _predicted(w, order)
    F = Fraction
    for p in range(0, w.N, 7):
        dt = F(w.t_pred) - F(w.t_j[p])
        for k in range(3):
            x, v, a, j, s, c = (F(float(arr[p, k])) for arr in (w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle))
            if order == 4:
                X = x + dt * v + dt ** 2 / 2 * a + dt ** 3 / 6 * j
                V = v + dt * a + dt ** 2 / 2 * j
                A = a
            else:
                X = x + dt * v + dt ** 2 / 2 * a + dt ** 3 / 6 * j + dt ** 4 / 24 * s + dt ** 5 / 120 * c
                V = v + dt * a + dt ** 2 / 2 * j + dt ** 3 / 6 * s + dt ** 4 / 24 * c
                A = a + dt * j + dt ** 2 / 2 * s + dt ** 3 / 6 * c
            for got, exact in ((xp[p, k], X), (vp[p, k], V), (ap[p, k], A)):
                ulp = math.ulp(float(exact))
                assert abs(F(float(got)) - exact) <= F(ulp) * F(51, 100)   # correctly rounded (+ double-rounding slack)


def test_predictor_dt_zero_is_identity_and_negative_dt():
    w = make_config(1, N=32)
    t_same = np.full(w.N, 0.5)
    xp, vp, ap = oracle.predict(6, 0.5, t_same, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)
    assert np.array_equal(xp, w.pos) and np.array_equal(vp, w.vel) and np.array_equal(ap, w.acc)
    # a pure quadratic trajectory is reproduced for dt < 0 as well
    z = np.zeros_like(w.pos)
    xp, vp, _ = oracle.predict(4, 0.25, t_same, w.pos, w.vel, w.acc, z)
    np.testing.assert_allclose(xp, w.pos - 0.25 * w.vel + 0.03125 * w.acc, rtol=1e-15, atol=1e-17)
    np.testing.assert_allclose(vp, w.vel - 0.25 * w.acc, rtol=1e-15, atol=1e-17)


# ----------------------------------------------------------------------------- neighbours
def test_bruteforce_neighbours_tiny():
    w = make_config(5, N=64)
    h2 = w.h2 * 0.4
    res = oracle.forces_ilist(4, w.mass, w.ident, w.pos, w.vel, None, w.ident, w.eps2, h2_i=h2, ngb_cap=8)
    for i in range(w.N):
        d = w.pos - w.pos[i]
        d2 = d[:, 0] * d[:, 0] + d[:, 1] * d[:, 1] + d[:, 2] * d[:, 2]
        order = [j for j in np.argsort(d2, kind="stable") if j != i]
        assert res.nn_addr[i] == order[0] and res.nn_id[i] == w.ident[order[0]]
        assert res.nn_d2[i] == pytest.approx(d2[order[0]], rel=1e-15)
        members = sorted(j for j in order if d2[j] < h2[i] * (1 - 1e-14))
        fuzzy = [j for j in order if abs(d2[j] - h2[i]) <= 1e-14 * h2[i]]
        assert not fuzzy
        assert res.ngb_count[i] == len(members)
        got = [int(x) for x in res.ngb_list[i] if x >= 0]
        assert got == members[:8]            # P8: lowest addresses, ascending, truncated at cap
        # the long-double decisions (the ones the GPU tests are judged against) pinned by the same brute force
        assert res.nn_addr_ld[i] == order[0] and res.nn_d2_ld[i] == pytest.approx(d2[order[0]], rel=1e-15)
        assert res.ngb_count_ld[i] == len(members)
        assert [int(x) for x in res.ngb_list_ld[i] if x >= 0] == members[:8]
    assert (res.ngb_count > 8).any() and (res.ngb_count <= 8).any()


def test_lattice_ties_and_strictness():
    """Integer lattice: every d2 exact.  Tie -> lowest address (P6); d2 == h2 is NOT a neighbour (P7)."""
    w = lattice_workload(4, 0.25)
    s2 = 0.25 ** 2
    for h2v, nmax in ((s2, 0), (2 * s2, 6), (2 * s2 * (1 + 2 ** -40), 18)):
        res = oracle.forces_ilist(4, w.mass, w.ident, w.pos, w.vel, None, w.ident, w.eps2,
                                  h2_i=np.full(w.N, h2v), ngb_cap=32)
        for i in range(w.N):
            d = w.pos - w.pos[i]
            d2 = (d * d).sum(1)
            d2[i] = np.inf
            assert res.nn_d2[i] == s2
            assert res.nn_addr[i] == int(np.flatnonzero(d2 == s2)[0])      # lowest address among ties
            assert res.ngb_count[i] == int((d2 < h2v).sum())
        assert res.ngb_count.max() == nmax
        assert np.array_equal(res.nn_addr, res.nn_addr_ld) and np.array_equal(res.nn_d2, res.nn_d2_ld)
        assert np.array_equal(res.ngb_count, res.ngb_count_ld) and np.array_equal(res.ngb_list, res.ngb_list_ld)


def test_self_skip_and_empty_cases():
    one = np.zeros((1, 3))
    r = oracle.forces(6, np.array([1.0]), np.array([0], np.int32), one, one, one, np.array([0], np.int32),
                      one, one, one, 1e-4, h2=np.array([1.0]))
    assert not r.acc.any() and not r.jerk.any() and not r.snap.any() and r.pot[0] == 0.0
    assert r.nn_addr[0] == -1 and r.nn_id[0] == -1 and np.isinf(r.nn_d2[0]) and r.ngb_count[0] == 0
    # N = 2: each sees only the other, even with a finite softening (no -m/eps self term, P3)
    x = np.array([[0.0, 0, 0], [2.0, 0, 0]]); z = np.zeros((2, 3)); ids = np.array([10, 11], np.int32)
    r = oracle.forces(4, np.array([1.0, 3.0]), ids, x, z, None, ids, x, z, None, 0.0, h2=np.array([5.0, 1.0]))
    np.testing.assert_allclose(r.acc, [[0.75, 0, 0], [-0.25, 0, 0]])
    np.testing.assert_allclose(r.pot, [-1.5, -0.5])
    assert list(r.nn_id) == [11, 10] and list(r.ngb_count) == [1, 0]
    # explicit sink with id < 0 matches no j
    r = oracle.forces(4, np.array([1.0, 3.0]), ids, x, z, None, np.array([-1], np.int32), x[:1] + [[1.0, 0, 0]],
                      z[:1], None, 0.0)
    np.testing.assert_allclose(r.acc, [[-1.0 + 3.0, 0, 0]])


# ----------------------------------------------------------------------------- golden fixtures
def test_golden_ring_sums_and_regression_fixture():
    import os
    g = os.path.join(os.path.dirname(__file__), "golden")
    # n = 2, 4, 6 have elementary values: 1, 1 + 2 sqrt2, 2*2 + 2*2/sqrt3 + 1
    vals = {int(l.split()[0]): float(l.split()[1]) for l in open(os.path.join(g, "ring_sums.txt")) if l[0] != "#"}
    assert vals[2] == pytest.approx(1.0, rel=1e-15)
    assert vals[4] == pytest.approx(1 + 2 * math.sqrt(2), rel=1e-15)
    assert vals[6] == pytest.approx(4 + 4 / math.sqrt(3) + 1, rel=1e-15)
    # square of unit radius, m = 1: the stored sum reproduces the oracle
    x = np.array([[1.0, 0, 0], [0, 1.0, 0], [-1.0, 0, 0], [0, -1.0, 0]]); z = np.zeros((4, 3))
    ids = np.arange(4, dtype=np.int32)
    r = oracle.forces(4, np.ones(4), ids, x, z, None, ids, x, z, None, 0.0)
    np.testing.assert_allclose(r.acc, -x * vals[4] / 4, rtol=1e-15, atol=1e-16)
    # regression fixture written by tests/golden/make_golden.py (oracle only)
    w = make_config(1, N=64)
    xp, vp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    res = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, w.ident, w.eps2, h2_i=w.h2 * 0.4, ngb_cap=16)
    for line in open(os.path.join(g, "cfg1_n64.txt")):
        if line[0] == "#":
            continue
        t = line.split()
        i = int(t[0]); f = [float.fromhex(v) for v in t[1:8]]
        assert list(res.acc[i]) + list(res.jerk[i]) + [res.pot[i]] == f
        assert res.nn_addr[i] == int(t[8]) and res.nn_d2[i] == float.fromhex(t[9]) and res.ngb_count[i] == int(t[10])
