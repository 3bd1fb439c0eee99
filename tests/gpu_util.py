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


# ---- integer decisions: judged against the oracle's LONG-DOUBLE decisions within north_star's band ------------
# north_star: "nearest-neighbour index: bit-exact, with ties broken by lowest index; neighbour sets: exact, except
# pairs within 1e-12 relative of the radius boundary".  The kernels decide on an fp64 d2, the oracle on its own
# long-double d2 (no shared formula); the two can only differ where two candidates (or a pair and h2) are closer
# than fp64 resolves, which the band allows.  Every accepted difference is counted and printed; expect 0.
BAND = 1e-12
DECISION_STATS = {"nn_checked": 0, "nn_in_band": 0, "ngb_checked": 0, "ngb_in_band": 0}


def _d2_ld(xj, xi):
    d = np.asarray(xj, dtype=np.longdouble) - np.asarray(xi, dtype=np.longdouble)
    return d[..., 0] * d[..., 0] + d[..., 1] * d[..., 1] + d[..., 2] * d[..., 2]


def _addr_of_id(ident):
    ident = np.asarray(ident)
    if np.array_equal(ident, np.arange(ident.size)):
        return lambda i: int(i)
    table = {int(v): k for k, v in enumerate(ident)}
    return lambda i: table[int(i)]


def check_nn_ld(res, ref, what=""):
    """GPU nearest neighbour (id, r2) against the oracle's long-double decision (ref.nn_addr_ld, ref.nn_d2_ld)."""
    g = ref.inputs
    ident = np.asarray(g["ident"])
    want = np.where(ref.nn_addr_ld >= 0, ident[np.maximum(ref.nn_addr_ld, 0)], -1)
    got = np.asarray(res["nn_id"])
    DECISION_STATS["nn_checked"] += got.size
    same = got == want
    fin = same & (want >= 0)
    # the returned squared distance is the fp64 evaluation of the same pair: within a few ulp of the long-double one
    assert (np.abs(res["nn_r2"][fin] - ref.nn_d2_ld[fin]) <= 8 * 2.0 ** -53 * ref.nn_d2_ld[fin]).all(), f"{what}: nn r2 off"
    assert np.isinf(res["nn_r2"][same & (want < 0)]).all(), f"{what}: empty nn must report +inf"
    a_of = _addr_of_id(ident)
    for i in np.flatnonzero(~same):
        assert got[i] >= 0 and want[i] >= 0, f"{what}: i={i} nn {got[i]} vs long-double decision {want[i]}"
        ag, ao = a_of(got[i]), int(ref.nn_addr_ld[i])
        dg, do = _d2_ld(g["xj"][ag], g["xi"][i]), _d2_ld(g["xj"][ao], g["xi"][i])
        # an exact long-double tie must have gone to the lowest address; otherwise only the band excuses a difference
        assert dg != do and abs(dg - do) <= BAND * do, \
            f"{what}: i={i} nn addr {ag} (d2 {dg!r}) vs long-double decision {ao} (d2 {do!r}): outside the 1e-12 band"
        DECISION_STATS["nn_in_band"] += 1
    return int((~same).sum())


def check_sets_ld(counts, lists, ref, what=""):
    """GPU neighbour counts and lists (lists[i] = ascending addresses, truncated at cap) against the oracle's
    long-double sets; a pair may differ only within 1e-12 relative of h2."""
    g = ref.inputs
    cap = g["ngb_cap"]
    n_band = 0
    DECISION_STATS["ngb_checked"] += len(lists)
    for i, got in enumerate(lists):
        row = ref.ngb_list_ld[i]
        want = row[row >= 0][:cap]
        if counts[i] == ref.ngb_count_ld[i] and np.array_equal(got, want):
            continue
        assert ref.ngb_count_ld[i] <= cap and counts[i] <= cap, \
            f"{what}: i={i} truncated lists differ from the long-double decision ({counts[i]} vs {ref.ngb_count_ld[i]})"
        diff = np.setxor1d(got, want)
        assert diff.size and len(got) == counts[i], f"{what}: i={i} count {counts[i]} does not match its list"
        d2 = _d2_ld(g["xj"][diff], g["xi"][i])
        h2 = np.longdouble(g["h2"][i])
        assert (np.abs(d2 - h2) <= BAND * h2).all(), f"{what}: i={i} members {diff} differ outside the 1e-12 band of h2"
        n_band += diff.size
    DECISION_STATS["ngb_in_band"] += n_band
    return n_band


def check_forces(res, ref, precision, order, flags, what=""):
    tol = TOL[precision]
    errs = dict(acc=rel_err(res["acc"], ref.acc).max(), jerk=rel_err(res["jerk"], ref.jerk).max(),
                pot=rel_err(res["pot"], ref.pot).max())
    if order == 6:
        errs["snap"] = rel_err(res["snap"], ref.snap).max()
    for k, v in errs.items():
        assert v <= tol[k], f"{what}: {k} max rel err {v:.3e} > {tol[k]:.0e}"
    if flags & (s2.S2_WANT_NN | s2.S2_WANT_NGB):
        # primary: the oracle's long-double decision within north_star's band ("parity criterion")
        errs["nn_in_band"] = check_nn_ld(res, ref, what)
        # secondary: the fp64 decision with the kernel's operation order (reading R-D2) is reproduced bit for bit
        assert np.array_equal(res["nn_id"], ref.nn_id), f"{what}: nearest-neighbour ids differ"
        assert np.array_equal(res["nn_r2"], ref.nn_d2), f"{what}: nearest-neighbour d2 differ"
    if flags & s2.S2_WANT_NGB:
        inband = np.flatnonzero(np.asarray(res["ngb_count"]) != ref.ngb_count_ld)
        if inband.size:   # counts may differ from the long-double sets only through band pairs: the list check decides
            assert (ref.ngb_count_ld[inband] <= ref.inputs["ngb_cap"]).all(), f"{what}: counts differ on truncated lists"
        assert np.array_equal(res["ngb_count"], ref.ngb_count), f"{what}: neighbour counts differ"
    return errs


def check_neighbour_lists(ctx, ref, ni, cap, what="", counts=None):
    off, lst = s2.s2_get_neighbours_csr(ctx, ni)
    lists = [lst[off[i]:off[i + 1]] for i in range(ni)]
    if counts is None:
        counts = s2.s2_get_results(ctx, ni)["ngb_count"]
    assert ref.inputs["ngb_cap"] == cap
    n_band = check_sets_ld(counts, lists, ref, what)           # primary: long-double sets within the band
    for i in range(ni):                                         # secondary: the fp64 decision, bit for bit
        want = ref.ngb_list[i][ref.ngb_list[i] >= 0][:cap]
        assert np.array_equal(lists[i], want), f"{what}: neighbour list of i={i} differs: {lists[i]} vs {want}"
    return n_band
