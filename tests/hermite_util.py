"""Oracle-backed force source for the block-time-step driver (tests only)."""
import numpy as np

import oracle


class OracleBackend:
    """Same interface as paper_1510_04068_b200.hermite.S2Backend, forces from the CPU oracle."""

    def __init__(self, n, eps2, order=4):
        self.n, self.eps2, self.order = n, float(eps2), order
        self.ident = np.arange(n, dtype=np.int32)
        self.t, self.m = np.zeros(n), np.zeros(n)
        self.x, self.v, self.a, self.j, self.s, self.c = (np.zeros((n, 3)) for _ in range(6))

    def set_j(self, idx, t, mass, pos, vel, acc, jerk, snap=None, crackle=None):
        self.t[idx], self.m[idx] = t, mass
        self.x[idx], self.v[idx], self.a[idx], self.j[idx] = pos, vel, acc, jerk
        if snap is not None:
            self.s[idx], self.c[idx] = snap, crackle

    def forces(self, t, idx):
        o = self.order
        xp, vp, ap = oracle.predict(o, float(t), self.t, self.x, self.v, self.a, self.j, self.s, self.c)
        r = oracle.forces_ilist(o, self.m, self.ident, xp, vp, ap if o == 6 else None,
                                np.ascontiguousarray(idx, dtype=np.int32), self.eps2)
        return (r.acc, r.jerk, r.pot, r.snap) if o == 6 else (r.acc, r.jerk, r.pot)

    def close(self):
        pass
