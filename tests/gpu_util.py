"""Helpers for the -m gpu parity tests: drive the C ABI through the binding, run the oracle on
the same seeded inputs, compare with the error norms of DESIGN.md (reading P12)."""
from __future__ import annotations

import numpy as np

import oracle
import paper_1510_04068_b200 as s2

# tolerances of BASELINE.json north_star (max over i of the per-particle relative error)
TOL = {
    s2.S2_FP64: dict(acc=1e-13, pot=1e-13, jerk=1e-12, snap=1e-12),
    s2.S2_DS: dict(acc=1e-10, pot=1e-10, jerk=1e-10, snap=1e-10),
    s2.S2_FP32: dict(acc=1e-5, pot=1e-5, jerk=1e-5, snap=1e-5),
}


def open_and_load(w, order=None, precision=s2.S2_FP64, ngb_cap=256, nj=None, chunks=1):
    """s2_open + s2_set_j (optionally in several calls) + s2_commit_j for workload w."""
    order = order or w.order
    nj = nj or w.N
    ctx = s2.s2_open(0, order, precision, nj_capacity=max(nj, 1), ngb_cap=ngb_cap)
    addr = np.arange(nj, dtype=np.int32)
    for part in np.array_split(addr, chunks):
        if part.size == 0:
            continue
        s2.s2_set_j(ctx, part, w.ident[part], w.t_j[part], w.mass[part], w.pos[part], w.vel[part], w.acc[part],
                    w.jerk[part], w.snap[part] if order == 6 else None, w.crackle[part] if order == 6 else None)
    s2.s2_commit_j(ctx)
    return ctx


def rel_err(got, ref):
    """per-i ||got - ref|| / ||ref|| (vectors) or |got - ref| / |ref| (scalars)."""
    got, ref = np.asarray(got, dtype=np.longdouble), np.asarray(ref, dtype=np.longdouble)
    if got.ndim == 2:
        num = np.sqrt(((got - ref) ** 2).sum(1))
        den = np.sqrt((ref ** 2).sum(1))
    else:
        num, den = np.abs(got - ref), np.abs(ref)
    return (num / den).astype(np.float64)


def oracle_on_gpu_prediction(ctx, w, order, ilist, eps2, h2_i=None, ngb_cap=256, nj=None):
    """Stage (ii) of reading P1: the oracle's O2-O4 on the GPU's own fp64 predicted arrays."""
    nj = nj or w.N
    xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, nj)
    return oracle.forces_ilist(order, w.mass[:nj], w.ident[:nj], xp, vp, ap, ilist, eps2, h2_i, ngb_cap), (xp, vp, ap)


def check_forces(res, ref, precision, order, flags, what=""):
    tol = TOL[precision]
    errs = dict(acc=rel_err(res["acc"], ref.acc).max(), jerk=rel_err(res["jerk"], ref.jerk).max(),
                pot=rel_err(res["pot"], ref.pot).max())
    if order == 6:
        errs["snap"] = rel_err(res["snap"], ref.snap).max()
    for k, v in errs.items():
        assert v <= tol[k], f"{what}: {k} max rel err {v:.3e} > {tol[k]:.0e}"
    if flags & (s2.S2_WANT_NN | s2.S2_WANT_NGB):
        assert np.array_equal(res["nn_id"], ref.nn_id), f"{what}: nearest-neighbour ids differ"
        assert np.array_equal(res["nn_r2"], ref.nn_d2), f"{what}: nearest-neighbour d2 differ"
    if flags & s2.S2_WANT_NGB:
        assert np.array_equal(res["ngb_count"], ref.ngb_count), f"{what}: neighbour counts differ"
    return errs


def check_neighbour_lists(ctx, ref, ni, cap, what=""):
    off, lst = s2.s2_get_neighbours_csr(ctx, ni)
    for i in range(ni):
        got = lst[off[i]:off[i + 1]]
        want = ref.ngb_list[i][ref.ngb_list[i] >= 0][:cap]
        assert np.array_equal(got, want), f"{what}: neighbour list of i={i} differs: {got} vs {want}"
