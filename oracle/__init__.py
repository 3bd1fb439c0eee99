"""CPU oracle for the Sapporo2 hot path -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Thin ctypes wrapper over ``hermite_oracle.c`` (long double direct summation).
Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  It imports nothing from the
CUDA package and the CUDA package imports nothing from here.

Citations are to /root/reference/PAPER.md lines (see hermite_oracle.c header) and
SURVEY.md sec 8(c) steps O1-O4.
"""
from __future__ import annotations

import ctypes as C
from dataclasses import dataclass

import numpy as np

from .build import build as _build

_lib = None


def lib() -> C.CDLL:
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build())
        _lib.oracle_ldbl_mant_dig.restype = C.c_int
        _lib.oracle_max_threads.restype = C.c_int
        assert _lib.oracle_ldbl_mant_dig() >= 64
    return _lib


def max_threads() -> int:
    return int(lib().oracle_max_threads())


def _p(a, dtype):
    if a is None:
        return None
    assert a.dtype == dtype and a.flags.c_contiguous, (a.dtype, dtype)
    return a.ctypes.data_as(C.c_void_p)


def _f64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float64)


def _i32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int32)


def predict(order: int, t: float, t_j, pos, vel, acc, jerk, snap=None, crackle=None):
    """O1: Taylor predictor.  Returns (x_p, v_p, a_p) as fp64 (n,3) arrays;
    a_p is the stored acceleration passed through when order == 4."""
    t_j, pos, vel, acc, jerk = map(_f64, (t_j, pos, vel, acc, jerk))
    snap, crackle = _f64(snap), _f64(crackle)
    n = t_j.shape[0]
    if order == 6:
        assert snap is not None and crackle is not None
    xp, vp, ap = np.empty((n, 3)), np.empty((n, 3)), np.empty((n, 3))
    d = np.float64
    lib().oracle_predict(C.c_int(n), C.c_int(order), C.c_double(t), _p(t_j, d), _p(pos, d), _p(vel, d),
                         _p(acc, d), _p(jerk, d), _p(snap, d), _p(crackle, d), _p(xp, d), _p(vp, d), _p(ap, d))
    return xp, vp, ap


@dataclass
class ForceResult:
    acc: np.ndarray
    jerk: np.ndarray
    snap: np.ndarray | None
    pot: np.ndarray
    nn_addr: np.ndarray       # fp64-decision nearest neighbour (j address, -1 if none)
    nn_id: np.ndarray
    nn_d2: np.ndarray
    nn_addr_ld: np.ndarray    # long-double-decision nearest neighbour (informational)
    ngb_count: np.ndarray | None
    ngb_list: np.ndarray | None   # (ni, cap), ascending addresses, -1 padded
    nn_d2_ld: np.ndarray | None = None        # long-double d2 of nn_addr_ld, rounded to fp64 once
    ngb_count_ld: np.ndarray | None = None    # neighbour set decided on the long-double d2 (rr < h2)
    ngb_list_ld: np.ndarray | None = None
    inputs: dict | None = None                # the geometry the decisions were taken on (xj, xi, h2, ident): lets a
                                              # test re-evaluate one pair's d2 in long double without another oracle run

    def ngb_sets(self):
        return [set(int(x) for x in row[row >= 0]) for row in self.ngb_list]


def forces(order: int, mass, ident, xp, vp, ap, i_id, xi, vi, ai, eps2: float,
           h2=None, ngb_cap: int = 256) -> ForceResult:
    """O2-O4 with explicit i-particles: direct sum over all j with id_j != id_i."""
    mass, xp, vp = _f64(mass), _f64(xp), _f64(vp)
    ident, i_id = _i32(ident), _i32(i_id)
    xi, vi = _f64(xi), _f64(vi)
    N, ni = mass.shape[0], i_id.shape[0]
    if order == 6:
        ap, ai = _f64(ap), _f64(ai)
        assert ap is not None and ai is not None
    else:
        ap = ai = None
    h2 = _f64(h2)
    acc, jerk, pot = np.zeros((ni, 3)), np.zeros((ni, 3)), np.zeros(ni)
    snap = np.zeros((ni, 3)) if order == 6 else None
    nn_addr, nn_id = np.empty(ni, np.int32), np.empty(ni, np.int32)
    nn_addr_ld = np.empty(ni, np.int32)
    nn_d2 = np.empty(ni)
    cnt = np.zeros(ni, np.int32) if h2 is not None else None
    lst = np.full((ni, ngb_cap), -1, np.int32) if h2 is not None else None
    nn_d2_ld = np.empty(ni)
    cnt_ld = np.zeros(ni, np.int32) if h2 is not None else None
    lst_ld = np.full((ni, ngb_cap), -1, np.int32) if h2 is not None else None
    d, i = np.float64, np.int32
    lib().oracle_forces(C.c_int(order), C.c_int(N), _p(mass, d), _p(ident, i), _p(xp, d), _p(vp, d), _p(ap, d),
                        C.c_int(ni), _p(i_id, i), _p(xi, d), _p(vi, d), _p(ai, d), _p(h2, d), C.c_double(eps2),
                        _p(acc, d), _p(jerk, d), _p(snap, d), _p(pot, d),
                        _p(nn_addr, i), _p(nn_id, i), _p(nn_d2, d), _p(nn_addr_ld, i),
                        _p(cnt, i), _p(lst, i), C.c_int(ngb_cap), _p(nn_d2_ld, d), _p(cnt_ld, i), _p(lst_ld, i))
    return ForceResult(acc, jerk, snap, pot, nn_addr, nn_id, nn_d2, nn_addr_ld, cnt, lst, nn_d2_ld, cnt_ld, lst_ld,
                       dict(xj=xp, xi=xi, h2=h2, ident=ident, ngb_cap=ngb_cap, order=order, mass=mass, vj=vp, aj=ap,
                            i_id=i_id, vi=vi, ai=ai, eps2=eps2))


def forces_ilist(order: int, mass, ident, xp, vp, ap, i_address, eps2: float,
                 h2_i=None, ngb_cap: int = 256) -> ForceResult:
    """O2 by address: the i-state is the predicted j-state at i_address (reading P15)."""
    ia = np.asarray(i_address, dtype=np.int64)
    ident = _i32(ident)
    return forces(order, mass, ident, xp, vp, ap, ident[ia], np.asarray(xp)[ia], np.asarray(vp)[ia],
                  None if ap is None else np.asarray(ap)[ia], eps2, h2_i, ngb_cap)


def term_norms(order: int, mass, ident, xp, vp, ap, i_id, xi, vi, ai, eps2: float, rms: bool = False):
    """Per-i sum over j of the norms of the individual pair terms (error norm of reading P12): (nacc, njerk, nsnap).
    rms=True returns instead the roots of the sums of their squares (error norm of reading R-F32)."""
    mass, xp, vp = _f64(mass), _f64(xp), _f64(vp)
    ident, i_id = _i32(ident), _i32(i_id)
    xi, vi = _f64(xi), _f64(vi)
    N, ni = mass.shape[0], i_id.shape[0]
    if order == 6:
        ap, ai = _f64(ap), _f64(ai)
    else:
        ap = ai = None
    na, nj, ns = np.empty(ni), np.empty(ni), np.empty(ni)
    ra, rj, rs = np.empty(ni), np.empty(ni), np.empty(ni)
    d, i = np.float64, np.int32
    lib().oracle_term_norms(C.c_int(order), C.c_int(N), _p(mass, d), _p(ident, i), _p(xp, d), _p(vp, d), _p(ap, d),
                            C.c_int(ni), _p(i_id, i), _p(xi, d), _p(vi, d), _p(ai, d), C.c_double(eps2),
                            _p(na, d), _p(nj, d), _p(ns, d), _p(ra, d), _p(rj, d), _p(rs, d))
    return (ra, rj, rs) if rms else (na, nj, ns)
