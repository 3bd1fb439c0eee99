"""Block-time-step 4th- and 6th-order Hermite integrators on top of the force library (host side).

This is the layer the paper calls the host integrator (sec 3.7): it "picks the active set,
corrects, computes time steps" on the CPU and leaves "predict, gravity, particle copy" to the GPU.  It is the
second workload of SURVEY sec 8(f): it drives every entry point of include/s2b200.h the way a production code
does -- partial j updates (s2_set_j + s2_commit_j of the corrected particles only), s2_predict to the block
time, s2_calc_ilist for an i-list whose length varies between 1 and N, s2_get_results.

All pairwise arithmetic and the Taylor prediction of the j-particles run in the CUDA kernels.  The host part
below is the textbook corrector and time-step rule of the 4th-order Hermite scheme the paper names (ref [27],
L92, L251), written for NumPy arrays of the active particles only:

    corrector   v1 = v0 + (a0 + a1) dt / 2 + (j0 - j1) dt^2 / 12
                x1 = x0 + (v0 + v1) dt / 2 + (a0 - a1) dt^2 / 12
    derivatives s0 = (-6 (a0 - a1) - dt (4 j0 + 2 j1)) / dt^2,   c0 = (12 (a0 - a1) + 6 dt (j0 + j1)) / dt^3
                s1 = s0 + c0 dt,  c1 = c0
    time step   dt = sqrt(eta (|a1| |s1| + |j1|^2) / (|j1| |c1| + |s1|^2))      (Aarseth criterion, eta = 0.01, L152)
                quantised to a power of two, block-aligned, at most doubled per step.

The force source is a small backend object, so the same driver can be run against any implementation of
`set_j / forces` (the tests run it against the CPU oracle to check the GPU run step by step).
"""
from __future__ import annotations

import numpy as np


class S2Backend:
    """Forces from libs2b200 (4th or 6th order, any precision mode)."""

    def __init__(self, n: int, eps2: float, precision: int = 0, device: int = 0, order: int = 4):
        from . import binding as s2
        self.s2, self.n, self.eps2, self.order = s2, n, float(eps2), order
        self.ctx = s2.s2_open(device, order, precision, nj_capacity=n, ngb_cap=0)
        self.ident = np.arange(n, dtype=np.int32)
        self.calls = 0
        self.pairs = 0

    def set_j(self, idx, t, mass, pos, vel, acc, jerk, snap=None, crackle=None):
        s2 = self.s2
        idx = np.ascontiguousarray(idx, dtype=np.int32)
        s2.s2_set_j(self.ctx, idx, self.ident[idx], t, mass, pos, vel, acc, jerk, snap, crackle)
        s2.s2_commit_j(self.ctx)

    def forces(self, t: float, idx):
        """acc, jerk, pot (and snap for order 6) of the listed particles at time t."""
        s2 = self.s2
        idx = np.ascontiguousarray(idx, dtype=np.int32)
        s2.s2_predict(self.ctx, float(t), self.n)
        s2.s2_calc_ilist(self.ctx, idx, None, self.eps2, 0)
        r = s2.s2_get_results(self.ctx, idx.size)
        self.calls += 1
        self.pairs += idx.size * self.n
        if self.order == 6:
            return r["acc"], r["jerk"], r["pot"], r["snap"]
        return r["acc"], r["jerk"], r["pot"]

    def close(self):
        self.s2.s2_close(self.ctx)


def _pow2_floor(x):
    """Largest power of two <= x (element-wise, x > 0)."""
    return np.exp2(np.floor(np.log2(x)))


class Hermite4:
    """Individual (block) time steps, 4th-order Hermite predictor-corrector."""

    def __init__(self, backend, mass, pos, vel, eta: float = 0.01, eta_start: float = 0.0025,
                 dt_max: float = 2.0 ** -3, dt_min: float = 2.0 ** -40):
        self.b = backend
        self.n = mass.shape[0]
        self.m = np.ascontiguousarray(mass, dtype=np.float64)
        self.x = np.array(pos, dtype=np.float64, order="C")
        self.v = np.array(vel, dtype=np.float64, order="C")
        self.a = np.zeros_like(self.x)
        self.j = np.zeros_like(self.x)
        self.pot = np.zeros(self.n)
        self.t = np.zeros(self.n)
        self.dt = np.full(self.n, dt_max)
        self.eta, self.dt_max, self.dt_min = eta, dt_max, dt_min
        self.time = 0.0
        self.block_steps = 0
        self.particle_steps = 0
        self.active_hist = []
        # start-up: forces at t = 0 from positions and velocities alone, then dt = eta_s |a| / |j|
        everyone = np.arange(self.n, dtype=np.int32)
        self.b.set_j(everyone, self.t, self.m, self.x, self.v, self.a, self.j)
        self.a, self.j, self.pot = (np.array(q) for q in self.b.forces(0.0, everyone))
        an, jn = np.linalg.norm(self.a, axis=1), np.linalg.norm(self.j, axis=1)
        raw = eta_start * an / np.maximum(jn, 1e-300)
        self.dt = np.clip(_pow2_floor(np.maximum(raw, dt_min)), dt_min, dt_max)
        self.b.set_j(everyone, self.t, self.m, self.x, self.v, self.a, self.j)

    # ------------------------------------------------------------------ one block step
    def step(self):
        t_new = float((self.t + self.dt).min())
        act = np.flatnonzero(self.t + self.dt == t_new).astype(np.int32)
        a1, j1, pot = self.b.forces(t_new, act)
        dt = self.dt[act][:, None]
        x0, v0, a0, j0 = self.x[act], self.v[act], self.a[act], self.j[act]
        v1 = v0 + (a0 + a1) * (dt / 2) + (j0 - j1) * (dt * dt / 12)
        x1 = x0 + (v0 + v1) * (dt / 2) + (a0 - a1) * (dt * dt / 12)
        s0 = (-6.0 * (a0 - a1) - dt * (4.0 * j0 + 2.0 * j1)) / (dt * dt)
        c0 = (12.0 * (a0 - a1) + 6.0 * dt * (j0 + j1)) / (dt * dt * dt)
        s1 = s0 + c0 * dt
        nrm = lambda q: np.linalg.norm(q, axis=1)
        an, jn, sn, cn = nrm(a1), nrm(j1), nrm(s1), nrm(c0)
        raw = np.sqrt(self.eta * (an * sn + jn * jn) / np.maximum(jn * cn + sn * sn, 1e-300))
        old = self.dt[act]
        new = np.minimum(_pow2_floor(np.maximum(raw, self.dt_min)), 2.0 * old)
        grow = new > old
        new[grow & (np.fmod(t_new, 2.0 * old) != 0.0)] = old[grow & (np.fmod(t_new, 2.0 * old) != 0.0)]   # block alignment
        new = np.clip(new, self.dt_min, self.dt_max)
        self.x[act], self.v[act], self.a[act], self.j[act], self.pot[act] = x1, v1, a1, j1, pot
        self.t[act] = t_new
        self.dt[act] = new
        self.b.set_j(act, self.t[act], self.m[act], x1, v1, a1, j1)   # only the corrected particles are re-sent (L88)
        self.time = t_new
        self.block_steps += 1
        self.particle_steps += act.size
        self.active_hist.append(act.size)
        return act.size

    def run_until(self, t_end: float):
        """Advances until every particle sits at t_end (a multiple of dt_max)."""
        assert np.fmod(t_end, self.dt_max) == 0.0, "t_end must be a multiple of dt_max"
        while self.time < t_end:
            self.step()
        assert (self.t == t_end).all()

    # ------------------------------------------------------------------ diagnostics
    def energy(self):
        """Total energy at a synchronisation time (all particles at the same t): T + 1/2 sum m pot."""
        assert (self.t == self.t[0]).all(), "energy() needs a synchronisation time"
        pot = self.b.forces(float(self.t[0]), np.arange(self.n, dtype=np.int32))[2]
        kin = 0.5 * float((self.m * (self.v * self.v).sum(axis=1)).sum())
        return kin + 0.5 * float((self.m * pot).sum())


class Hermite6(Hermite4):
    """6th-order Hermite scheme (the paper's sec 3.7 integrator, ref [5]; L152-L156): forces, jerks and snaps at
    both ends of a step define a 5th-degree interpolation polynomial of the acceleration.  With h = dt / 2,
    A+- = a1 +- a0, J+- = h (j1 +- j0), S+- = h^2 (s1 +- s0):

        v1 = v0 + h (A+ - 2/5 J- + 1/15 S+)
        x1 = x0 + h (v1 + v0) - 2/5 h^2 (a1 - a0) + 1/15 h^3 (j1 + j0)
        F5 = (S- - 3 J+ + 3 A-) / 16,  F4 = (S+ - J-) / 16,  F3 = (5 J+ - 5 A- - S-) / 8     (F_k = h^k a^(k)_mid / k!)
        at t1:  a^(3) = 6 (F3 + 4 F4 + 10 F5) / h^3,  a^(4) = 24 (F4 + 5 F5) / h^4,  a^(5) = 120 F5 / h^5
        dt = eta (A1 / A4)^(1/3),  A_k = sqrt(|a^(k-1)| |a^(k+1)| + |a^(k)|^2)            (generalised Aarseth)

    The library's 6th-order predictor uses the stored snap and the interpolated crackle a^(3)."""

    def __init__(self, backend, mass, pos, vel, eta: float = 0.1, eta_start: float = 0.001,
                 dt_max: float = 2.0 ** -3, dt_min: float = 2.0 ** -40, averaged: bool = False, eta4: float = 0.01):
        # eta_start: the first step is dt = eta_start |a| / |jerk| (only a and jerk exist yet) and the first corrector starts
        # without a snap history; 0.01 leaves dE/E = 6e-8 after one time unit at N = 16384 ALL of which is made in that first
        # step, 0.001 leaves 1.5e-11 (the paper quotes ~1e-12, L164; its start-up is not stated) for five more block steps
        # averaged: the paper's runs (L156) take the mean of this generalised step and the 4th-order Aarseth step
        self.averaged, self.eta4 = averaged, eta4
        self.b = backend
        self.n = mass.shape[0]
        self.m = np.ascontiguousarray(mass, dtype=np.float64)
        self.x = np.array(pos, dtype=np.float64, order="C")
        self.v = np.array(vel, dtype=np.float64, order="C")
        z = np.zeros_like(self.x)
        self.a, self.j, self.s, self.c = z.copy(), z.copy(), z.copy(), z.copy()
        self.pot = np.zeros(self.n)
        self.t = np.zeros(self.n)
        self.eta, self.dt_max, self.dt_min = eta, dt_max, dt_min
        self.time = 0.0
        self.block_steps = 0
        self.particle_steps = 0
        self.active_hist = []
        everyone = np.arange(self.n, dtype=np.int32)
        # start-up: acc and jerk first; the snap needs every particle's acceleration, so a second pass
        self.b.set_j(everyone, self.t, self.m, self.x, self.v, self.a, self.j, self.s, self.c)
        self.a, self.j, _, _ = (np.array(q) for q in self.b.forces(0.0, everyone))
        self.b.set_j(everyone, self.t, self.m, self.x, self.v, self.a, self.j, self.s, self.c)
        self.a, self.j, self.pot, self.s = (np.array(q) for q in self.b.forces(0.0, everyone))
        an, jn = np.linalg.norm(self.a, axis=1), np.linalg.norm(self.j, axis=1)
        raw = eta_start * an / np.maximum(jn, 1e-300)
        self.dt = np.clip(_pow2_floor(np.maximum(raw, dt_min)), dt_min, dt_max)
        self.b.set_j(everyone, self.t, self.m, self.x, self.v, self.a, self.j, self.s, self.c)

    def step(self):
        t_new = float((self.t + self.dt).min())
        act = np.flatnonzero(self.t + self.dt == t_new).astype(np.int32)
        a1, j1, pot, s1 = self.b.forces(t_new, act)
        dt = self.dt[act][:, None]
        h = 0.5 * dt
        x0, v0, a0, j0, s0 = self.x[act], self.v[act], self.a[act], self.j[act], self.s[act]
        Ap, Am = a1 + a0, a1 - a0
        Jp, Jm = h * (j1 + j0), h * (j1 - j0)
        Sp, Sm = h * h * (s1 + s0), h * h * (s1 - s0)
        v1 = v0 + h * (Ap - 0.4 * Jm + Sp / 15.0)
        x1 = x0 + h * (v1 + v0) - 0.4 * h * h * Am + (h * h * h / 15.0) * (j1 + j0)
        F5 = (Sm - 3.0 * Jp + 3.0 * Am) / 16.0
        F4 = (Sp - Jm) / 16.0
        F3 = (5.0 * Jp - 5.0 * Am - Sm) / 8.0
        c1 = 6.0 * (F3 + 4.0 * F4 + 10.0 * F5) / h ** 3          # crackle a^(3) at t1
        p1 = 24.0 * (F4 + 5.0 * F5) / h ** 4                     # a^(4)
        q1 = 120.0 * F5 / h ** 5                                 # a^(5), constant over the step
        nrm = lambda q: np.linalg.norm(q, axis=1)
        A1 = np.sqrt(nrm(a1) * nrm(s1) + nrm(j1) ** 2)
        A4 = np.sqrt(nrm(c1) * nrm(q1) + nrm(p1) ** 2)
        raw = self.eta * np.cbrt(A1 / np.maximum(A4, 1e-300))
        if self.averaged:
            jn, sn, cn = nrm(j1), nrm(s1), nrm(c1)
            raw4 = np.sqrt(self.eta4 * (nrm(a1) * sn + jn * jn) / np.maximum(jn * cn + sn * sn, 1e-300))
            raw = 0.5 * (raw + raw4)
        old = self.dt[act]
        new = np.minimum(_pow2_floor(np.maximum(raw, self.dt_min)), 2.0 * old)
        blocked = (new > old) & (np.fmod(t_new, 2.0 * old) != 0.0)
        new[blocked] = old[blocked]
        new = np.clip(new, self.dt_min, self.dt_max)
        self.x[act], self.v[act], self.a[act], self.j[act], self.s[act], self.c[act] = x1, v1, a1, j1, s1, c1
        self.pot[act] = pot
        self.t[act] = t_new
        self.dt[act] = new
        self.b.set_j(act, self.t[act], self.m[act], x1, v1, a1, j1, s1, c1)
        self.time = t_new
        self.block_steps += 1
        self.particle_steps += act.size
        self.active_hist.append(act.size)
        return act.size


class DeviceHermite:
    """The same two schemes with everything on the device (include/s2b200.h, s2_bts_*): the library's j-store is the
    particle state, corrector / time-step rule / active-set selection are kernels, and a block step costs the host one
    12-byte read.  Hermite4 / Hermite6 above are its host reference (the tests run both in lock-step)."""

    def __init__(self, mass, pos, vel, eps2: float, order: int = 4, precision: int = 0, eta: float | None = None,
                 eta_start: float | None = None, dt_max: float = 2.0 ** -3, dt_min: float = 2.0 ** -40, device: int = 0,
                 averaged: bool = False, eta4: float = 0.01):
        from . import binding as s2
        self.s2, self.order, self.eps2 = s2, order, float(eps2)
        self.n = int(np.asarray(mass).shape[0])
        self.m = np.ascontiguousarray(mass, dtype=np.float64)
        eta = (0.01 if order == 4 else 0.1) if eta is None else eta
        eta_start = (0.0025 if order == 4 else 0.001) if eta_start is None else eta_start
        self.ctx = s2.s2_open(device, order, precision, nj_capacity=self.n, ngb_cap=0)
        self.bts = s2.s2_bts_open(self.ctx, self.n, eps2, eta, eta_start, dt_max, dt_min, averaged, eta4)
        s2.s2_bts_init(self.bts, self.m, pos, vel)

    def step(self) -> int:
        """One block step; returns its active count."""
        assert self.s2.s2_bts_run(self.bts, np.inf, 1) == 1
        return int(self.s2.s2_bts_get_history(self.bts, self.stats()["block_steps"] - 1, 1)[0])

    def run_until(self, t_end: float, time_device: bool = False) -> int:
        return self.s2.s2_bts_run(self.bts, float(t_end), time_device=time_device)

    def state(self) -> dict:
        return self.s2.s2_bts_get_state(self.bts)

    def stats(self) -> dict:
        st = self.s2.s2_bts_stats(self.bts)
        st["small"] = self.s2.s2_bts_small_stats(self.bts)   # the share taken by the small-step kernel
        return st

    def history(self) -> np.ndarray:
        return self.s2.s2_bts_get_history(self.bts)

    @property
    def time(self) -> float:
        return self.stats()["time"]

    def energy(self) -> float:
        """T + 1/2 sum m pot at a synchronisation time (every particle at the same t), potential from a force call."""
        s2 = self.s2
        st = self.state()
        assert (st["t"] == st["t"][0]).all(), "energy() needs a synchronisation time"
        s2.s2_predict(self.ctx, float(st["t"][0]), self.n)
        s2.s2_calc_ilist(self.ctx, np.arange(self.n, dtype=np.int32), None, self.eps2, 0)
        pot = s2.s2_get_results(self.ctx, self.n)["pot"]
        kin = 0.5 * float((self.m * (st["vel"] * st["vel"]).sum(axis=1)).sum())
        return kin + 0.5 * float((self.m * pot).sum())

    def close(self):
        self.s2.s2_bts_close(self.bts)
        self.s2.s2_close(self.ctx)
