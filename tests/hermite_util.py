"""Oracle-backed force source for the block-time-step driver (tests only)."""
import numpy as np

import oracle


class OracleBackend:
    """Same interface as paper_1510_04068_b200.hermite.S2Backend, forces from the CPU oracle."""

    def __init__(self, n, eps2):
        self.n, self.eps2 = n, float(eps2)
        self.ident = np.arange(n, dtype=np.int32)
        self.t, self.m = np.zeros(n), np.zeros(n)
        self.x, self.v, self.a, self.j = (np.zeros((n, 3)) for _ in range(4))

    def set_j(self, idx, t, mass, pos, vel, acc, jerk):
        self.t[idx], self.m[idx] = t, mass
        self.x[idx], self.v[idx], self.a[idx], self.j[idx] = pos, vel, acc, jerk

    def forces(self, t, idx):
        xp, vp, _ = oracle.predict(4, float(t), self.t, self.x, self.v, self.a, self.j)
        r = oracle.forces_ilist(4, self.m, self.ident, xp, vp, None, np.ascontiguousarray(idx, dtype=np.int32), self.eps2)
        return r.acc, r.jerk, r.pot

    def close(self):
        pass
