"""Seeded Plummer-sphere workloads (stand-ins for the paper's Plummer runs).

The paper measures on Plummer spheres ("131072 source particles",
L118 N_sink = N_source sweeps, L152 "simulations of Plummer [32] spheres").  No
dataset is involved: everything here is generated from a seed, on the host, in
fp64, once, and the same arrays feed the CPU oracle and the GPU library.

Recipe (SURVEY.md §8(d) "Synthetic inputs", restated in DESIGN.md):
  1. counter-based PRNG: SplitMix64-style mixer, u = (z >> 11) * 2^-53;
  2. radius X ~ U(0, 0.999], r = (X^(-2/3) - 1)^(-1/2); isotropic direction;
  3. speed by rejection on g(q) = q^2 (1 - q^2)^3.5; |v| = q sqrt(2) (1 + r^2)^(-1/4);
  4. scaling to N-body units (G = M = 1, E = -1/4): lengths * 3 pi / 16,
     velocities * sqrt(16 / (3 pi));
  5. masses equal (1/N) or Salpeter (slope -2.35 on [0.1, 100], normalised);
  6. centre-of-mass position and velocity removed (mass weighted);
  7. stored derivatives = smooth analytic Plummer field of unit mass, scale a_P
     (closed-form time derivatives of -x (x.x + a_P^2)^(-3/2) along (x, v));
     crackle = snap * gauss / 0.1;
  8. particle times t_j = 1 - 2^-k_j, k_j uniform in [4, 12]; prediction time
     t = 1 - 2^-13 (all dt exactly representable);
  9. id_j = address_j = j; active sets = prefixes of one seeded permutation.

No particle-particle interaction and no Taylor predictor is evaluated here.  Step 7 does write out the closed-form
first and second time derivatives of ONE smooth field (a unit point mass with softening a_P at the origin) to give the
stored derivatives plausible magnitudes: that is generator data, never an expected value.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

A_PLUMMER = 3.0 * math.pi / 16.0          # Plummer scale length in N-body units
_BASE_SEED = 151004068 * 10

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix(z: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on a uint64 array (wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def splitmix64_uniform(seed: int, stream: int, counter: np.ndarray) -> np.ndarray:
    """u in [0, 1) for each counter value; independent streams per quantity."""
    with np.errstate(over="ignore"):
        key = _mix(np.asarray([(seed * 1000 + stream) & 0xFFFFFFFFFFFFFFFF], dtype=np.uint64))[0]
        z = key + (np.asarray(counter, dtype=np.uint64) + np.uint64(1)) * np.uint64(0x9E3779B97F4A7C15)
    z = _mix(z)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


# stream numbers
_S_RADIUS, _S_DIR1, _S_DIR2, _S_SPEED_Q, _S_SPEED_Y, _S_VDIR1, _S_VDIR2 = 1, 2, 3, 4, 5, 6, 7
_S_MASS, _S_LEVEL, _S_CRK1, _S_CRK2, _S_PERM = 8, 9, 10, 11, 12


@dataclass
class Workload:
    """One synthetic problem instance.  All arrays are host fp64 / int32, C-contiguous."""
    name: str
    N: int
    order: int                 # 4 or 6
    eps2: float
    t_pred: float
    ident: np.ndarray          # (N,)  int32, == address
    t_j: np.ndarray            # (N,)
    mass: np.ndarray           # (N,)
    pos: np.ndarray            # (N,3)
    vel: np.ndarray            # (N,3)
    acc: np.ndarray            # (N,3)
    jerk: np.ndarray           # (N,3)
    snap: np.ndarray           # (N,3)
    crackle: np.ndarray        # (N,3)
    h2: np.ndarray             # (N,)  squared neighbour radius of each particle
    perm: np.ndarray           # (N,)  int32 seeded permutation; active set = perm[:n_i]
    seed: int = 0
    notes: dict = field(default_factory=dict)

    def ilist(self, n_i: int) -> np.ndarray:
        return np.ascontiguousarray(self.perm[:n_i])


def _isotropic(u1: np.ndarray, u2: np.ndarray) -> np.ndarray:
    z = 1.0 - 2.0 * u1
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    phi = 2.0 * math.pi * u2
    return np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)


def make_workload(name: str, N: int, order: int, eps: float, seed: int,
                  salpeter: bool = False) -> Workload:
    idx = np.arange(N, dtype=np.uint64)

    # 2. radii and directions (structural units)
    X = 0.999 * (1.0 - splitmix64_uniform(seed, _S_RADIUS, idx))          # (0, 0.999]
    r = 1.0 / np.sqrt(X ** (-2.0 / 3.0) - 1.0)
    pos = r[:, None] * _isotropic(splitmix64_uniform(seed, _S_DIR1, idx),
                                  splitmix64_uniform(seed, _S_DIR2, idx))

    # 3. speeds by rejection; round k uses counter idx * 256 + k
    q = np.zeros(N)
    todo = np.arange(N)
    for k in range(256):
        if todo.size == 0:
            break
        c = idx[todo] * np.uint64(256) + np.uint64(k)
        qq = splitmix64_uniform(seed, _S_SPEED_Q, c)
        yy = 0.1 * splitmix64_uniform(seed, _S_SPEED_Y, c)
        ok = yy < qq * qq * (1.0 - qq * qq) ** 3.5
        q[todo[ok]] = qq[ok]
        todo = todo[~ok]
    assert todo.size == 0, "rejection sampling did not converge"
    speed = q * math.sqrt(2.0) * (1.0 + r * r) ** (-0.25)
    vel = speed[:, None] * _isotropic(splitmix64_uniform(seed, _S_VDIR1, idx),
                                      splitmix64_uniform(seed, _S_VDIR2, idx))

    # 4. N-body units
    pos *= A_PLUMMER
    vel *= math.sqrt(1.0 / A_PLUMMER)

    # 5. masses
    if salpeter:
        u = splitmix64_uniform(seed, _S_MASS, idx)
        lo, hi, p = 0.1, 100.0, 1.35
        mass = (lo ** (-p) - u * (lo ** (-p) - hi ** (-p))) ** (-1.0 / p)
        mass /= mass.sum()
    else:
        mass = np.full(N, 1.0 / N)

    # 6. centre of mass
    pos -= (mass[:, None] * pos).sum(axis=0) / mass.sum()
    vel -= (mass[:, None] * vel).sum(axis=0) / mass.sum()

    # 7. smooth-field derivatives: closed-form d/dt and d2/dt2 of -x s^(-3/2), s = x.x + a_P^2
    s = (pos * pos).sum(axis=1) + A_PLUMMER ** 2
    xv = (pos * vel).sum(axis=1)
    f3, f5, f7 = s ** -1.5, s ** -2.5, s ** -3.5
    acc = -pos * f3[:, None]
    jerk = -vel * f3[:, None] + 3.0 * pos * (xv * f5)[:, None]
    vv_xa = (vel * vel).sum(axis=1) + (pos * acc).sum(axis=1)
    d2f = -3.0 * vv_xa * f5 + 15.0 * xv * xv * f7
    snap = -acc * f3[:, None] + 6.0 * vel * (xv * f5)[:, None] - pos * d2f[:, None]
    u1 = splitmix64_uniform(seed, _S_CRK1, idx)
    u2 = splitmix64_uniform(seed, _S_CRK2, idx)
    gauss = np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * math.pi * u2)
    crackle = snap * (gauss / 0.1)[:, None]

    # 8. times
    level = 4 + np.minimum(8, (9.0 * splitmix64_uniform(seed, _S_LEVEL, idx)).astype(np.int64))
    t_j = 1.0 - np.ldexp(1.0, -level)
    t_pred = 1.0 - 2.0 ** -13

    # neighbour radius: holds ~32 particles at the local analytic Plummer number density
    r2 = (pos * pos).sum(axis=1)
    h = A_PLUMMER * (32.0 / N) ** (1.0 / 3.0) * (1.0 + r2 / A_PLUMMER ** 2) ** (5.0 / 6.0)

    # 9. ids and the active-set permutation
    ident = np.arange(N, dtype=np.int32)
    perm = np.argsort(splitmix64_uniform(seed, _S_PERM, idx), kind="stable").astype(np.int32)

    c = np.ascontiguousarray
    return Workload(name=name, N=N, order=order, eps2=float(eps) ** 2, t_pred=t_pred,
                    ident=ident, t_j=c(t_j), mass=c(mass), pos=c(pos), vel=c(vel), acc=c(acc),
                    jerk=c(jerk), snap=c(snap), crackle=c(crackle), h2=c(h * h), perm=perm,
                    seed=seed, notes={"salpeter": salpeter, "eps": float(eps)})


# BASELINE.json configs (1-based) plus the north_star headline point "H".
CONFIGS = {
    1: dict(name="cfg1_plummer_1k", N=1024, order=4, eps=1e-3, salpeter=False),
    2: dict(name="cfg2_small_64", N=64, order=4, eps=1e-4, salpeter=False),
    3: dict(name="cfg3_blockstep_64k", N=65536, order=4, eps=0.01 * 65536 ** (-1.0 / 3.0), salpeter=False),
    4: dict(name="cfg4_sixth_256k", N=262144, order=6, eps=1e-4, salpeter=True),
    5: dict(name="cfg5_neighbours_1m", N=1048576, order=4, eps=1e-4, salpeter=True),
    "H": dict(name="headline_256k", N=262144, order=4, eps=1e-4, salpeter=False),
}
_CFG_SEEDNO = {1: 1, 2: 2, 3: 3, 4: 4, 5: 5, "H": 6}


def make_config(k, N: int | None = None, order: int | None = None) -> Workload:
    """Workload for BASELINE.json config k (1..5) or 'H'; N/order may be overridden for
    scaled-down test variants of the same recipe (the name then says so)."""
    cfg = dict(CONFIGS[k])
    if N is not None and N != cfg["N"]:
        cfg["name"] += f"_N{N}"
        if k == 3:
            cfg["eps"] = 0.01 * N ** (-1.0 / 3.0)
        cfg["N"] = N
    if order is not None and order != cfg["order"]:
        cfg["name"] += f"_o{order}"
        cfg["order"] = order
    return make_workload(seed=_BASE_SEED + _CFG_SEEDNO[k], **cfg)


def lattice_workload(n_side: int = 4, scale: float = 0.25, order: int = 4, seed: int = 7) -> Workload:
    """Particles on a small-integer cubic lattice times a power of two: every squared
    distance is exact in fp32, fp64 and long double, so nearest-neighbour ties are real ties
    and h^2 can be set equal to an attained d^2 (strictness test)."""
    g = np.arange(n_side, dtype=np.float64)
    pos = np.stack(np.meshgrid(g, g, g, indexing="ij"), axis=-1).reshape(-1, 3) * scale
    N = pos.shape[0]
    idx = np.arange(N, dtype=np.uint64)
    # shuffle addresses so that "lowest address" is not "lowest coordinate"
    perm = np.argsort(splitmix64_uniform(seed, _S_PERM, idx), kind="stable")
    pos = np.ascontiguousarray(pos[perm])
    vel = np.round(8.0 * (splitmix64_uniform(seed, _S_VDIR1, np.arange(3 * N, dtype=np.uint64)) - 0.5)).reshape(N, 3) / 8.0
    z3 = np.zeros((N, 3))
    mass = np.full(N, 1.0 / N)
    return Workload(name=f"lattice_{n_side}", N=N, order=order, eps2=2.0 ** -10, t_pred=0.0,
                    ident=np.arange(N, dtype=np.int32), t_j=np.zeros(N), mass=mass, pos=pos, vel=vel,
                    acc=z3.copy(), jerk=z3.copy(), snap=z3.copy(), crackle=z3.copy(),
                    h2=np.full(N, 2.0 * scale * scale), perm=np.arange(N, dtype=np.int32)[::-1].copy(),
                    seed=seed, notes={"lattice": True})
