"""Uniform-operand sweep (force_sweep_bank_kernel): j-particles read from the constant bank chunk by
chunk.  The balancer only picks it for very large i-lists, so these tests force it (s2_set_tuning key 8 = 2) at sizes
the oracle finishes in seconds: one chunk, exactly one chunk, a ragged last chunk, several chunks, every order and flag."""
import numpy as np
import pytest

import oracle
import paper_1510_04068_b200 as s2
from workloads import lattice_workload, make_config

from gpu_util import TOL, check_neighbour_lists, check_nn_ld, open_and_load, rel_err

pytestmark = pytest.mark.gpu

NN, NGB = s2.S2_WANT_NN, s2.S2_WANT_NGB


def _load(w, order, N, cap):
    ctx = s2.s2_open(0, order, s2.S2_FP64, nj_capacity=N, ngb_cap=cap)
    addr = np.arange(N, dtype=np.int32)
    s2.s2_set_j(ctx, addr, w.ident[:N], w.t_j[:N], w.mass[:N], w.pos[:N], w.vel[:N], w.acc[:N], w.jerk[:N],
                w.snap[:N] if order == 6 else None, w.crackle[:N] if order == 6 else None)
    s2.s2_commit_j(ctx)
    s2.s2_predict(ctx, w.t_pred, N)
    return ctx


@pytest.mark.parametrize("order", [4, 6, 2])
def test_bank_sweep_parity_all_chunkings(order):
    rng = np.random.default_rng(40 + order)
    cap = 24
    # chunk lengths: 1024 (4th order), 680 (6th), 1360 (2nd): below, at, just above, and several times a chunk
    for N in (1, 2, 679, 680, 681, 1024, 1025, 1360, 1361, 3000, 5000):
        w = make_config(4 if order == 6 else 5, N=max(N, 4), order=order if order != 2 else 4)
        ctx = _load(w, order, N, cap)
        xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, N)
        s2.s2_set_tuning(ctx, 8, 2)
        for ni in sorted({1, N, max(1, N // 3)}):
            for flags in (0, NN, NN | NGB):
                il = rng.permutation(N)[:ni].astype(np.int32)
                h2 = (w.h2[il] * 2.0) if flags & NGB else None
                s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
                res = s2.s2_get_results(ctx, ni)
                info = s2.s2_last_launch_info(ctx)
                assert info["reduced"] == 3, info
                ref = oracle.forces_ilist(4 if order == 2 else order, w.mass[:N], w.ident[:N], xp, vp,
                                          ap if order == 6 else None, il, w.eps2, h2, cap)
                what = f"order {order} N {N} n_i {ni} flags {flags} {info}"
                tol = TOL[s2.S2_FP64]
                if N > 1:
                    assert rel_err(res["acc"], ref.acc).max() <= tol["acc"], what
                    assert rel_err(res["pot"], ref.pot).max() <= tol["pot"], what
                    if order >= 4:
                        assert rel_err(res["jerk"], ref.jerk).max() <= tol["jerk"], what
                    if order == 6:
                        assert rel_err(res["snap"], ref.snap).max() <= tol["snap"], what
                else:
                    assert not res["acc"].any() and res["pot"][0] == 0.0, what
                if flags:
                    check_nn_ld(res, ref, what)      # primary: the oracle's long-double decision (north_star's band)
                    assert np.array_equal(res["nn_id"], ref.nn_id) and np.array_equal(res["nn_r2"], ref.nn_d2), what
                if flags & NGB:
                    assert np.array_equal(res["ngb_count"], ref.ngb_count), what
                    assert res["overflow"] == bool((ref.ngb_count > cap).any()), what
                    check_neighbour_lists(ctx, ref, ni, cap, what)
        s2.s2_close(ctx)


def test_bank_sweep_explicit_sinks_and_lattice_ties():
    # explicit sinks (not j-particles; id < 0 matches nothing) through the chunked sweep
    w = make_config(3, N=2500)
    ctx = open_and_load(w, 4, ngb_cap=16)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)
    rng = np.random.default_rng(9)
    ni = 77
    pos = xp[rng.permutation(w.N)[:ni]] + 1e-3 * rng.standard_normal((ni, 3))
    vel = rng.standard_normal((ni, 3))
    ident = np.full(ni, -1, np.int32)
    ident[::3] = w.ident[:26]               # some sinks share the id of a source: that source is skipped
    h2 = np.full(ni, 0.02 ** 2)
    s2.s2_set_tuning(ctx, 8, 2)
    s2.s2_calc_explicit(ctx, ident, pos, vel, None, h2, w.eps2, NN | NGB)
    assert s2.s2_last_launch_info(ctx)["reduced"] == 3
    res = s2.s2_get_results(ctx, ni)
    ref = oracle.forces(4, w.mass, w.ident, xp, vp, None, ident, pos, vel, None, w.eps2, h2, 16)
    assert rel_err(res["acc"], ref.acc).max() <= 1e-13 and rel_err(res["jerk"], ref.jerk).max() <= 1e-12
    check_nn_ld(res, ref, "explicit sinks, bank sweep")
    assert np.array_equal(res["nn_id"], ref.nn_id) and np.array_equal(res["ngb_count"], ref.ngb_count)
    check_neighbour_lists(ctx, ref, ni, 16, "explicit sinks, bank sweep")
    s2.s2_close(ctx)

    # integer lattice: every d2 exact, real ties (lowest address wins), h2 equal to an attained d2 (strict <)
    w = lattice_workload(12, 0.25)   # 1728 particles: two chunks
    ctx = open_and_load(w, 4, ngb_cap=32)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)
    il = np.arange(w.N, dtype=np.int32)[::-1].copy()
    h2 = np.full(w.N, 2 * 0.25 ** 2)
    s2.s2_set_tuning(ctx, 8, 2)
    s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
    res = s2.s2_get_results(ctx, w.N)
    ref = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, h2, 32)
    check_nn_ld(res, ref, "lattice, bank sweep")
    assert np.array_equal(res["nn_id"], ref.nn_id) and np.array_equal(res["nn_r2"], ref.nn_d2)
    assert np.array_equal(res["ngb_count"], ref.ngb_count)
    check_neighbour_lists(ctx, ref, w.N, 32, "lattice, bank sweep")
    s2.s2_close(ctx)


def test_bank_sweep_reproducible_agrees_with_tiled_and_is_shared_safely():
    """Bit-identical run to run; equal to the shared-memory sweep within rounding; and two contexts on two streams
    that both use the (single, per-device) constant bank do not disturb each other."""
    import torch
    w = make_config(3, N=6000)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    s2.s2_set_tuning(ctx, 8, 1)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
    base = s2.s2_get_results(ctx, w.N)
    assert s2.s2_last_launch_info(ctx)["reduced"] != 3
    s2.s2_set_tuning(ctx, 8, 2)
    runs = []
    for _ in range(5):
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
        r = s2.s2_get_results(ctx, w.N)
        runs.append(np.concatenate([r["acc"].ravel(), r["jerk"].ravel(), r["pot"], r["nn_r2"], r["nn_id"]]))
    for r in runs[1:]:
        assert np.array_equal(r, runs[0])
    assert rel_err(runs[0][:3 * w.N].reshape(-1, 3), base["acc"]).max() < 1e-13
    assert np.array_equal(runs[0][-w.N:], base["nn_id"])

    # second context, different particles, its own stream; calls interleaved without synchronising in between
    w2 = make_config(1, N=3000)
    st2 = torch.cuda.Stream()
    ctx2 = open_and_load(w2)
    s2.s2_synchronize(ctx2)
    s2.s2_set_stream(ctx2, st2.cuda_stream)
    s2.s2_predict(ctx2, w2.t_pred, w2.N)
    s2.s2_set_tuning(ctx2, 8, 2)
    il2 = w2.ilist(w2.N)
    d_il, d_il2 = torch.from_numpy(il).cuda(), torch.from_numpy(il2).cuda()
    torch.cuda.synchronize()
    for _ in range(3):
        s2.s2_calc_ilist_device(ctx, d_il, None, w.eps2, NN)
        s2.s2_calc_ilist_device(ctx2, d_il2, None, w2.eps2, NN)
    r1 = s2.s2_get_results(ctx, w.N)
    r2 = s2.s2_get_results(ctx2, w2.N)
    assert np.array_equal(np.concatenate([r1["acc"].ravel(), r1["jerk"].ravel(), r1["pot"], r1["nn_r2"], r1["nn_id"]]), runs[0])
    xp2, vp2, _ = s2.s2_get_predicted_j(ctx2, 0, w2.N)
    ref2 = oracle.forces_ilist(4, w2.mass, w2.ident, xp2, vp2, None, il2, w2.eps2, None, 256)
    assert rel_err(r2["acc"], ref2.acc).max() <= 1e-13 and np.array_equal(r2["nn_id"], ref2.nn_id)
    s2.s2_close(ctx2)
    s2.s2_close(ctx)


@pytest.mark.timeout(300)
def test_bank_sweep_overlapping_launches_at_residency_boundaries():
    """The chunk launches overlap (programmatic dependent launch) and hand the two banks over through device flags.
    Grids just below, at and above whole residency rounds (296 CTAs of 256 i on a 148-SM part) and a 1-CTA grid,
    several sweeps back to back without synchronising: equal to the shared-memory sweep within rounding, bit-identical
    from call to call, and no launch waits on work that is not resident (the test would hang)."""
    import torch
    N = 8192                                      # 8 chunks
    w = make_config(3, N=N)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, N)
    rng = np.random.default_rng(12)
    # 100 and 256 CTAs: launches of less than one round, whose CTAs find the next ticket only by looking again inside
    # the chunk, and whose successors then share the round with them
    for ni in (1, 255, 100 * 256 + 17, 256 * 256, 295 * 256, 296 * 256, 297 * 256 + 3, 2 * 296 * 256, 3 * 296 * 256 - 1):
        il = torch.from_numpy(rng.integers(0, N, ni).astype(np.int32)).cuda()     # i-particles may repeat
        for flags in (0, NN):
            s2.s2_set_tuning(ctx, 8, 1)
            s2.s2_calc_ilist_device(ctx, il, None, w.eps2, flags)
            ref = s2.s2_get_results(ctx, ni)
            s2.s2_set_tuning(ctx, 8, 2)
            for _ in range(3):
                s2.s2_calc_ilist_device(ctx, il, None, w.eps2, flags)
            a = s2.s2_get_results(ctx, ni)
            assert s2.s2_last_launch_info(ctx)["reduced"] == 3
            s2.s2_calc_ilist_device(ctx, il, None, w.eps2, flags)
            b = s2.s2_get_results(ctx, ni)
            for k in ("acc", "jerk", "pot", "nn_id", "nn_r2"):
                assert np.array_equal(a[k], b[k]), (ni, flags, k)
            assert rel_err(a["acc"], ref["acc"]).max() < 1e-13 and rel_err(a["jerk"], ref["jerk"]).max() < 1e-12
            assert np.array_equal(a["nn_id"], ref["nn_id"])
    s2.s2_close(ctx)


@pytest.mark.timeout(900)
@pytest.mark.parametrize("N,reps", [(8192, 30), (65536, 15), (262144, 5)])
def test_bank_sweep_stress_changing_jstore_back_to_back(N, reps):
    """The self-refilling uniform-operand sweep rewrites its constant banks from device code and overlaps its chunk
    launches (DESIGN.md 5.2 states what that assumes).  Stress: 4 x reps sweeps per N (200 over the three N), enqueued
    BACK TO BACK WITHOUT ANY HOST SYNCHRONISATION, the j-store changing between consecutive sweeps (alternating
    s2_predict times, and half-way a partial s2_commit_j_device), at the sizes where the automatic rule picks this
    sweep -- n_i = 49152, 65536, 131072 (128-thread instance) and 262144 (256-thread instance).  Every i of every
    sweep is compared with the shared-memory sweep of the same j-state (acc, pot 1e-13, jerk 1e-12), and sweeps of
    the same state must agree bit for bit: a stale bank, a chunk read before its refill or a constant-cache line
    surviving a launch would show up as a wrong chunk of j in some sweep."""
    import torch
    w = make_config("H" if N == 262144 else 3, N=N)
    ctx = open_and_load(w)
    dev = torch.device("cuda", 0)
    rng = np.random.default_rng(N)
    # partial commit: every 5th particle moves a little (device arrays: nothing synchronises)
    sub = np.arange(0, N, 5, dtype=np.int32)
    T = lambda a: torch.from_numpy(np.ascontiguousarray(a)).to(dev)
    orig = [T(sub), T(w.ident[sub]), T(w.t_j[sub]), T(w.mass[sub]), T(w.pos[sub]), T(w.vel[sub]), T(w.acc[sub]), T(w.jerk[sub])]
    moved = list(orig)
    moved[4] = T(w.pos[sub] + 0.03125 * w.vel[sub])
    moved[3] = T(w.mass[sub] * 1.5)
    times = {"A": w.t_pred, "B": w.t_pred + 2.0 ** -9, "C": w.t_pred, "D": w.t_pred + 2.0 ** -9}

    def enqueue(state, il, out):
        s2.s2_predict(ctx, times[state], N)
        s2.s2_calc_ilist_device(ctx, il, None, w.eps2, 0)
        s2.s2_get_results_device(ctx, il.numel(), acc=out[0], jerk=out[1], pot=out[2])

    def buffers(ni):
        return [torch.empty(ni * 3, dtype=torch.float64, device=dev), torch.empty(ni * 3, dtype=torch.float64, device=dev),
                torch.empty(ni, dtype=torch.float64, device=dev)]

    def rel(a, b, vec):
        if vec:
            a, b = a.view(-1, 3), b.view(-1, 3)
            return float(((a - b).norm(dim=1) / b.norm(dim=1)).max())
        return float(((a - b).abs() / b.abs()).max())

    total = 0
    for ni in (49152, 65536, 131072, 262144):
        il = torch.from_numpy(rng.integers(0, N, ni).astype(np.int32)).to(dev)
        # references: shared-memory sweep of each of the four j-states
        s2.s2_set_tuning(ctx, 8, 1)
        ref = {}
        for st in "AB":
            ref[st] = buffers(ni); enqueue(st, il, ref[st])
        assert s2.s2_last_launch_info(ctx)["reduced"] not in (3, 5)
        s2.s2_commit_j_device(ctx, *moved)
        for st in "CD":
            ref[st] = buffers(ni); enqueue(st, il, ref[st])
        s2.s2_commit_j_device(ctx, *orig)
        # the stress: automatic rule, no host synchronisation between the sweeps
        s2.s2_set_tuning(ctx, 8, 0)
        seq = [("AB"[k & 1]) for k in range(reps // 2)] + ["commit"] + [("CD"[k & 1]) for k in range(reps - reps // 2)]
        outs = []
        for st in seq:
            if st == "commit":
                s2.s2_commit_j_device(ctx, *moved)
                continue
            o = buffers(ni); enqueue(st, il, o); outs.append((st, o))
        info = s2.s2_last_launch_info(ctx)
        assert info["reduced"] == 3 and info["threads"] == (128 if ni < 200000 else 256), info
        s2.s2_commit_j_device(ctx, *orig)
        s2.s2_synchronize(ctx)
        first = {}
        for k, (st, o) in enumerate(outs):
            what = f"N={N} n_i={ni} sweep {k} state {st}"
            assert rel(o[0], ref[st][0], True) <= 1e-13, what
            assert rel(o[1], ref[st][1], True) <= 1e-12, what
            assert rel(o[2], ref[st][2], False) <= 1e-13, what
            if st in first:
                for a, b in zip(o, first[st]):
                    assert torch.equal(a, b), what + ": differs from an earlier sweep of the same state"
            else:
                first[st] = o
        assert rel(ref["A"][0], ref["C"][0], True) > 1e-6          # the partial commit really changed the forces
        total += len(outs)
        del outs, ref, first
    assert total == 4 * reps
    s2.s2_close(ctx)


def test_bank_sweep_documented_fallback_has_the_same_bits():
    """s2_set_tuning key 8 = 4: the banks are refilled by stream-ordered copies between ordinary launches (documented
    CUDA semantics; the path the library falls back to for good if its first-use self-test of the self-refilling sweep
    fails).  Same chunks, same order, same kernel: bit-identical records, decisions and lists."""
    w = make_config(5, N=7000)
    ctx = open_and_load(w, 4, ngb_cap=24)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    h2 = w.h2[il]
    for flags in (0, NN, NN | NGB):
        got = {}
        for key8, code in ((2, 3), (4, 5)):
            s2.s2_set_tuning(ctx, 8, key8)
            s2.s2_calc_ilist(ctx, il, h2 if flags & NGB else None, w.eps2, flags)
            assert s2.s2_last_launch_info(ctx)["reduced"] == code
            r = s2.s2_get_results(ctx, w.N)
            lists = s2.s2_get_neighbours_csr(ctx, w.N) if flags & NGB else None
            got[key8] = (r, lists)
        for k in ("acc", "jerk", "pot") + (("nn_id", "nn_r2") if flags else ()) + (("ngb_count",) if flags & NGB else ()):
            assert np.array_equal(got[2][0][k], got[4][0][k]), (flags, k)
        if flags & NGB:
            assert np.array_equal(got[2][1][0], got[4][1][0]) and np.array_equal(got[2][1][1], got[4][1][1])
    s2.s2_close(ctx)
