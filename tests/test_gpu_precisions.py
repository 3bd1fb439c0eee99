"""GPU parity of the double-single and fp32 force paths, and the large configurations (4, 5), against the
CPU oracle through the C ABI.  Tolerances: BASELINE.json north_star (max over i): DS 1e-10, fp32 1e-5;
nearest neighbour and neighbour sets exact in every mode (decisions are taken in fp64, reading P13)."""
import numpy as np
import pytest

import oracle
import paper_1510_04068_b200 as s2
from workloads import make_config, lattice_workload

from gpu_util import (check_forces, check_neighbour_lists, check_nn_ld, check_sets_ld, open_and_load,
                      oracle_on_gpu_prediction, rel_err)

pytestmark = pytest.mark.gpu

NN, NGB = s2.S2_WANT_NN, s2.S2_WANT_NGB
PREC = {"ds": s2.S2_DS, "fp32": s2.S2_FP32}
SAMPLE = 4096      # seeded i-sample where the full oracle is too slow (SURVEY 8(c) "Oracle cost and sampling")


@pytest.mark.parametrize("prec", ["ds", "fp32"])
@pytest.mark.parametrize("order", [4, 6])
@pytest.mark.parametrize("flags", [0, NN | NGB])
def test_precision_paths_all_shapes_ragged(prec, order, flags):
    """Every launch shape on a ragged problem (N = 1000, n_i = 37), both orders, with and without the
    decision outputs, in double-single and fp32."""
    P = PREC[prec]
    w = make_config(4 if order == 6 else 5, N=1000, order=order)
    ctx = open_and_load(w, order, precision=P, ngb_cap=24)
    s2.s2_predict(ctx, w.t_pred, w.N)
    ni = 37
    il = w.ilist(ni)
    h2 = w.h2[il] * 0.6 if flags & NGB else None
    ref, _ = oracle_on_gpu_prediction(ctx, w, order, il, w.eps2, h2, ngb_cap=24)
    shapes = [(L, 1, S, tile) for L in (1, 2, 4, 8, 16, 32) for S, tile in ((1, 0), (3, 64), (13, 32))]
    shapes += [(32, Wj, S, 0) for Wj in (2, 8) for S in (1, 5)] + [(8, 4, 3, 64), (4, 2, 1, 0)]
    worst = {}
    shapes = [s + (1,) for s in shapes]
    if P == s2.S2_FP32:                                   # register-tiled sweep (two i per thread) exists for fp32 and fp64
        shapes += [(1, 1, 1, 0, 2), (1, 1, 3, 64, 2), (1, 1, 13, 32, 2)]
        if flags == 0:                                    # ... with several lanes per i-slot (plain sums)
            shapes += [(L, 1, S, tile, 2) for L in (2, 8, 32) for S, tile in ((1, 0), (5, 64))]
    for L, Wj, S, tile, tiled in shapes:
        s2.s2_set_tuning(ctx, 1, L); s2.s2_set_tuning(ctx, 2, Wj); s2.s2_set_tuning(ctx, 0, S); s2.s2_set_tuning(ctx, 4, tile)
        s2.s2_set_tuning(ctx, 7, tiled)
        s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
        res = s2.s2_get_results(ctx, ni)
        info = s2.s2_last_launch_info(ctx)
        errs = check_forces(res, ref, P, order, flags, f"{prec} shape {info}")
        for k, v in errs.items():
            worst[k] = max(worst.get(k, 0.0), v)
        if flags & NGB:
            check_neighbour_lists(ctx, ref, ni, 24, f"{prec} shape {info}")
    print(f"{prec} order {order} flags {flags}: worst rel errors", {k: f"{v:.2e}" for k, v in worst.items()})
    s2.s2_close(ctx)


@pytest.mark.parametrize("prec", ["ds", "fp32"])
def test_cfg3_blockstep_ds_fp32(prec):
    """BASELINE config 3, DS and fp32 legs: N = 65536, n_i in {1, 32, 256, 2048, 16384, 65536}."""
    P = PREC[prec]
    w = make_config(3)
    ctx = open_and_load(w, 4, precision=P)
    s2.s2_predict(ctx, w.t_pred, w.N)
    for ni in (1, 32, 256, 2048, 16384, 65536):
        il = w.ilist(ni)
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=0)
        res = s2.s2_get_results(ctx, ni)
        pick = np.arange(ni) if ni <= SAMPLE else np.sort(np.random.default_rng(3).choice(ni, SAMPLE, replace=False))
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il[pick], w.eps2)
        sub = {k: (v[pick] if isinstance(v, np.ndarray) else v) for k, v in res.items()}
        errs = check_forces(sub, ref, P, 4, 0, f"cfg3 {prec} n_i={ni} {s2.s2_last_launch_info(ctx)}")
        print(f"cfg3 {prec} n_i={ni} (oracle on {pick.size} i, sample seed 3)", {k: f"{v:.2e}" for k, v in errs.items()})
    s2.s2_close(ctx)


@pytest.mark.parametrize("prec", ["ds", "fp32"])
def test_lattice_ties_exact_in_every_precision(prec):
    """Exact ties on an integer lattice: nn tie-break and the strict neighbour test must be bit-exact in
    every precision (reading P13)."""
    P = PREC[prec]
    w = lattice_workload(4, 0.25)
    ctx = open_and_load(w, 4, precision=P, ngb_cap=32)
    s2.s2_predict(ctx, 0.0, w.N)
    il = w.ilist(w.N)
    s2v = 0.25 ** 2
    for h2v in (s2v, 2 * s2v, 2 * s2v * (1 + 2 ** -40)):
        h2 = np.full(w.N, h2v)
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, h2, ngb_cap=32)
        for L in (0, 1, 8, 32):
            s2.s2_set_tuning(ctx, 1, L)
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
            res = s2.s2_get_results(ctx, w.N)
            check_forces(res, ref, P, 4, NN | NGB, f"lattice {prec} h2={h2v} L={L}")
            check_neighbour_lists(ctx, ref, w.N, 32)
    s2.s2_close(ctx)


@pytest.mark.parametrize("prec", ["ds", "fp32"])
def test_explicit_sinks_ds_fp32(prec):
    P = PREC[prec]
    w = make_config(4, N=500, order=6)
    ctx = open_and_load(w, 6, precision=P, ngb_cap=16)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, w.N)
    rng = np.random.default_rng(11)
    ni = 45
    xi, vi, ai = rng.normal(size=(ni, 3)) * 0.5, rng.normal(size=(ni, 3)) * 0.3, rng.normal(size=(ni, 3))
    ids = np.full(ni, -1, np.int32)
    ids[::3] = w.ident[:15]
    h2 = np.full(ni, 0.05)
    s2.s2_calc_explicit(ctx, ids, xi, vi, ai, h2, w.eps2, NN | NGB)
    res = s2.s2_get_results(ctx, ni)
    ref = oracle.forces(6, w.mass, w.ident, xp, vp, ap, ids, xi, vi, ai, w.eps2, h2, 16)
    check_forces(res, ref, P, 6, NN | NGB, f"explicit {prec}")
    check_neighbour_lists(ctx, ref, ni, 16)
    s2.s2_close(ctx)


def test_cfg4_sixth_order_all_active_sampled():
    """BASELINE config 4 at n_i = N = 262144 (6.9e10 pairs): oracle on a seeded sample of 4096 i, plus
    Newton's third law on the full GPU output."""
    w = make_config(4)
    ctx = open_and_load(w, 6)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2)
    res = s2.s2_get_results(ctx, w.N)
    pick = np.sort(np.random.default_rng(4).choice(w.N, SAMPLE, replace=False))
    ref, _ = oracle_on_gpu_prediction(ctx, w, 6, il[pick], w.eps2)
    sub = {k: (v[pick] if isinstance(v, np.ndarray) else v) for k, v in res.items()}
    errs = check_forces(sub, ref, s2.S2_FP64, 6, 0, f"cfg4 n_i=N {s2.s2_last_launch_info(ctx)}")
    print(f"cfg4 n_i=N sample {SAMPLE} (seed 4)", {k: f"{v:.2e}" for k, v in errs.items()})
    for q in ("acc", "jerk", "snap"):
        tot = np.abs((w.mass[il, None] * res[q]).sum(0)).max()
        scale = (w.mass[il] * np.linalg.norm(res[q], axis=1)).sum()
        assert tot <= 1e-10 * scale, (q, tot, scale)
    s2.s2_close(ctx)


_CFG5 = {}   # the 4096-i oracle result of config 5, shared by the two precision legs


@pytest.mark.parametrize("prec", ["fp64", "fp32"])
def test_cfg5_neighbour_path_sampled(prec):
    """BASELINE config 5: N = n_i = 2^20 Salpeter Plummer, nn + neighbour lists (cap 256), fp64 and fp32.
    Oracle on a seeded sample of 4096 i (sets judged against the long-double decision within north_star's band);
    counts, overflow flag and the third-law invariants on the full output.  The oracle runs once for both
    precisions: its inputs are the fp64 predicted planes, which every precision mode writes identically (checked)."""
    P = s2.S2_FP64 if prec == "fp64" else s2.S2_FP32
    w = make_config(5)
    ctx = open_and_load(w, 4, precision=P, ngb_cap=256)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    h2 = w.h2[il]
    s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
    res = s2.s2_get_results(ctx, w.N)
    pick = np.sort(np.random.default_rng(5).choice(w.N, SAMPLE, replace=False))
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)
    if "ref" not in _CFG5:
        _CFG5["ref"] = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il[pick], w.eps2, h2[pick], 256)
        _CFG5["xp"], _CFG5["vp"] = xp, vp
    assert np.array_equal(xp, _CFG5["xp"]) and np.array_equal(vp, _CFG5["vp"])
    ref = _CFG5["ref"]
    sub = {k: (v[pick] if isinstance(v, np.ndarray) else v) for k, v in res.items()}
    errs = check_forces(sub, ref, P, 4, NN | NGB, f"cfg5 {prec}")
    # all lists in one compacted read-back (device-side CSR), then the sampled ones against the oracle
    off, lst = s2.s2_get_neighbours_csr(ctx, w.N)
    cnt = res["ngb_count"]
    assert np.array_equal(np.diff(off), np.minimum(cnt, 256))
    lists = [lst[off[i]:off[i + 1]] for i in pick]
    n_band = check_sets_ld(cnt[pick], lists, ref, f"cfg5 {prec}")
    for k in range(0, SAMPLE, 64):                           # the single-list getter returns the same segment
        assert np.array_equal(s2.s2_get_neighbours(ctx, int(pick[k]), 256), lists[k])
    for k in range(SAMPLE):                                  # secondary: the fp64 decision, bit for bit
        assert np.array_equal(lists[k], ref.ngb_list[k][ref.ngb_list[k] >= 0][:256]), f"cfg5 {prec}: list of i={pick[k]}"
    print(f"cfg5 {prec} sample {SAMPLE} (seed 5)", {k: f"{v:.2e}" for k, v in errs.items()}, "pairs accepted in the 1e-12 band:",
          n_band, "mean/max neighbour count", cnt.mean(), cnt.max(), "overflows", int((cnt > 256).sum()),
          "list entries", int(off[-1]), s2.s2_last_launch_info(ctx))
    assert res["overflow"] == bool((cnt > 256).any())
    assert 8 < cnt.mean() < 128
    tol = 1e-10 if prec == "fp64" else 1e-4
    for q in ("acc", "jerk"):
        tot = np.abs((w.mass[il, None] * res[q]).sum(0)).max()
        scale = (w.mass[il] * np.linalg.norm(res[q], axis=1)).sum()
        assert tot <= tol * scale, (q, tot, scale)
    # symmetric nearest-neighbour sanity: the nn of i has i within the same distance
    nn = res["nn_id"]
    inv = np.empty(w.N, np.int64); inv[il] = np.arange(w.N)
    assert (res["nn_r2"][inv[nn]] <= res["nn_r2"]).all()
    s2.s2_close(ctx)


def test_headline_point_in_bench_configuration_sampled():
    """The bench workload (north_star target point): N = n_i = 2^18 equal-mass Plummer, eps = 1e-4, 4th order fp64,
    in the launch configuration bench.py times (device-resident i-list, automatic shape = uniform-operand sweep).
    Oracle on a seeded sample of 4096 i; Newton's third law and the potential symmetry on the full output."""
    import torch
    w = make_config("H")
    ctx = open_and_load(w, 4)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    d_il = torch.from_numpy(il).cuda()
    s2.s2_calc_ilist_device(ctx, d_il, None, w.eps2, 0)
    info = s2.s2_last_launch_info(ctx)
    assert info["reduced"] == 3 and info["lanes_per_i"] == 1 and info["S"] == w.N // 1024   # one launch per chunk
    res = s2.s2_get_results(ctx, w.N)
    pick = np.sort(np.random.default_rng(6).choice(w.N, SAMPLE, replace=False))
    ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il[pick], w.eps2)
    sub = {k: (v[pick] if isinstance(v, np.ndarray) else v) for k, v in res.items()}
    errs = check_forces(sub, ref, s2.S2_FP64, 4, 0, f"headline {info}")
    print(f"headline sample {SAMPLE} (seed 6)", info, {k: f"{v:.2e}" for k, v in errs.items()})
    for q in ("acc", "jerk"):
        tot = np.abs((w.mass[il, None] * res[q]).sum(0)).max()
        scale = (w.mass[il] * np.linalg.norm(res[q], axis=1)).sum()
        assert tot <= 1e-11 * scale, (q, tot, scale)
    # 1/2 sum m pot is the potential energy of a Plummer sphere in N-body units: -1/2 within sampling noise
    assert abs(0.5 * (w.mass[il] * res["pot"]).sum() + 0.5) < 0.02
    s2.s2_close(ctx)


def test_double_single_primitives_against_long_double():
    """Every double-single primitive of the S2_DS path on random operands against numpy long double
    (SURVEY sec 8(c) pin "DS arithmetic": error <= 2^-44 relative; round trip <= 2^-48)."""
    rng = np.random.default_rng(44)
    n = 20000
    a = rng.normal(size=n) * np.exp(rng.uniform(-8, 8, n))
    b = rng.normal(size=n) * np.exp(rng.uniform(-8, 8, n))
    b[: n // 4] = a[: n // 4] * (1 + rng.normal(size=n // 4) * 1e-6)       # nearly equal operands: cancellation in a - b
    ctx = s2.s2_open(0, 4, s2.S2_DS, nj_capacity=16, ngb_cap=0)
    out = s2.s2_test_ds_ops(ctx, a, b).astype(np.longdouble)
    s2.s2_close(ctx)
    A, B = a.astype(np.longdouble), b.astype(np.longdouble)
    u44, u48 = np.longdouble(2.0) ** -44, np.longdouble(2.0) ** -48
    assert (np.abs(out[:, 0] - A) <= u48 * np.abs(A)).all()
    # the operands the device really works with are the round-tripped ones
    Ar = out[:, 0]
    hi = b.astype(np.float32)
    Br = hi.astype(np.longdouble) + (b - hi.astype(np.float64)).astype(np.float32).astype(np.longdouble)
    assert (np.abs(out[:, 1] - (Ar + Br)) <= u44 * (np.abs(Ar) + np.abs(Br))).all()
    assert (np.abs(out[:, 2] - (Ar - Br)) <= u44 * (np.abs(Ar) + np.abs(Br))).all()
    assert (np.abs(out[:, 3] - Ar * Br) <= u44 * np.abs(Ar * Br)).all()
    assert (np.abs(out[:, 4] - Ar * Ar) <= u44 * Ar * Ar).all()
    assert (np.abs(out[:, 5] + 3 * Ar) <= u44 * 3 * np.abs(Ar)).all()
    rs = 1 / np.sqrt(np.abs(Ar))
    assert (np.abs(out[:, 6] - rs) <= 4 * u44 * rs).all()
    assert (np.abs(out[:, 7] - (Ar * Br + Ar)) <= u44 * (np.abs(Ar * Br) + np.abs(Ar))).all()


@pytest.mark.parametrize("prec", ["fp64", "ds", "fp32"])
def test_second_order_acc_pot_only(prec):
    """2nd-order (GRAPE-5 style) contexts: acc + pot (+ nn, neighbour lists) without jerk terms.
    acc and pot of the pair sum do not depend on velocities, so the oracle's 4th-order acc / pot on the GPU's
    predicted positions is the reference; the predictor with acc = jerk = NULL reduces to x + v dt."""
    P = {"fp64": s2.S2_FP64, "ds": s2.S2_DS, "fp32": s2.S2_FP32}[prec]
    w = make_config(5, N=3000)
    ctx = s2.s2_open(0, 2, P, nj_capacity=w.N, ngb_cap=24)
    addr = np.arange(w.N, dtype=np.int32)
    s2.s2_set_j(ctx, addr, w.ident, w.t_j, w.mass, w.pos, w.vel)          # no acc / jerk
    s2.s2_commit_j(ctx)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)
    dt = (w.t_pred - w.t_j)[:, None]
    assert np.abs(xp - (w.pos + w.vel * dt)).max() <= 4e-16 * np.abs(w.pos).max() and np.array_equal(vp, w.vel)
    from gpu_util import TOL, rel_err
    for ni, flags, tune in ((w.N, 0, {}), (w.N, NN | NGB, {}), (37, NN | NGB, {1: 8, 0: 5}), (37, 0, {1: 32, 2: 8, 0: 3}),
                            (700, NN, {7: 1, 1: 1, 0: 3}), (1, NN, {})):
        for k in range(8):
            s2.s2_set_tuning(ctx, k, tune.get(k, 0))
        il = w.ilist(ni)
        h2 = w.h2[il] * 0.6 if flags & NGB else None
        s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
        res = s2.s2_get_results(ctx, ni)
        ref = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, h2, 24)
        what = f"order 2 {prec} n_i={ni} flags={flags} {s2.s2_last_launch_info(ctx)}"
        assert rel_err(res["acc"], ref.acc).max() <= TOL[P]["acc"], what
        assert rel_err(res["pot"], ref.pot).max() <= TOL[P]["pot"], what
        assert not res["jerk"].any(), what
        if flags:
            check_nn_ld(res, ref, what)
            assert np.array_equal(res["nn_id"], ref.nn_id) and np.array_equal(res["nn_r2"], ref.nn_d2), what
        if flags & NGB:
            assert np.array_equal(res["ngb_count"], ref.ngb_count), what
            check_neighbour_lists(ctx, ref, ni, 24, what)
    # explicit sinks without velocities
    rng = np.random.default_rng(2)
    xi = rng.normal(size=(20, 3)) * 0.4
    ids = np.full(20, -1, np.int32)
    s2.s2_calc_explicit(ctx, ids, xi, None, None, None, w.eps2, 0)
    res = s2.s2_get_results(ctx, 20)
    ref = oracle.forces(4, w.mass, w.ident, xp, vp, None, ids, xi, np.zeros((20, 3)), None, w.eps2)
    assert rel_err(res["acc"], ref.acc).max() <= TOL[P]["acc"] and rel_err(res["pot"], ref.pot).max() <= TOL[P]["pot"]
    s2.s2_close(ctx)


def test_largest_store_small_ilist_sampled():
    """Maximum-size edge case: N = 2^22 j-particles (4x config 5; base store 0.5 GB, 10^4 times the 32-particle
    i-list), j-split path with many slices, NN + neighbour lists; and one explicit-sink call.  Full oracle (1.3e8 pairs)."""
    w = make_config(5, N=1 << 22)
    ctx = open_and_load(w, 4, ngb_cap=64, chunks=3)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(32)
    h2 = w.h2[il]
    s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
    res = s2.s2_get_results(ctx, 32)
    info = s2.s2_last_launch_info(ctx)
    ref, (xp, vp, _) = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, h2, ngb_cap=64)
    check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, f"N=2^22 n_i=32 {info}")
    check_neighbour_lists(ctx, ref, 32, 64, "N=2^22 n_i=32")
    assert info["S"] * info["warp_columns"] > 1            # the j range really was split
    s2.s2_calc_ilist(ctx, il[:1], None, w.eps2, 0)          # one active particle against 4M sources
    r1 = s2.s2_get_results(ctx, 1)
    assert rel_err(r1["acc"], ref.acc[:1]).max() <= 1e-13 and rel_err(r1["jerk"], ref.jerk[:1]).max() <= 1e-12
    s2.s2_close(ctx)


@pytest.mark.parametrize("order", [2, 4, 6])
@pytest.mark.parametrize("flags", [0, NN | NGB])
def test_fp32_packed_tiled_sweep_has_the_bits_of_the_scalar_sweep(order, flags):
    """The register-tiled fp32 sweep evaluates the two i-particles of a thread in packed FP32 instructions
    (FADD2 / FMUL2 / FFMA2); every half is rounded like the scalar instruction, so with the same slices and tiles
    it must return exactly the bits of the one-lane-per-i scalar sweep -- and both must match the oracle."""
    w = make_config(4 if order == 6 else 5, N=3000, order=max(order, 4))
    if order == 2:
        ctx = s2.s2_open(0, 2, s2.S2_FP32, nj_capacity=w.N, ngb_cap=24)
        s2.s2_set_j(ctx, np.arange(w.N, dtype=np.int32), w.ident, w.t_j, w.mass, w.pos, w.vel)
        s2.s2_commit_j(ctx)
    else:
        ctx = open_and_load(w, order, precision=s2.S2_FP32, ngb_cap=24)
    s2.s2_predict(ctx, w.t_pred, w.N)
    ni = 700                                              # two CTAs of 2 x 256 i-slots, ragged second one
    il = w.ilist(ni)
    h2 = w.h2[il] * 0.6 if flags & NGB else None
    keys = ("acc", "pot") + (("jerk",) if order >= 4 else ()) + (("snap",) if order == 6 else ())
    keys += ("nn_id", "nn_r2", "ngb_count") if flags else ()
    for S, tile, L in ((1, 0, 1), (3, 64, 1), (7, 256, 1)) + (((1, 0, 4), (5, 64, 16)) if flags == 0 else ()):
        got = {}
        for tiled in (1, 2):
            s2.s2_set_tuning(ctx, 1, L); s2.s2_set_tuning(ctx, 2, 1); s2.s2_set_tuning(ctx, 0, S)
            s2.s2_set_tuning(ctx, 4, tile); s2.s2_set_tuning(ctx, 7, tiled)
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
            got[tiled] = s2.s2_get_results(ctx, ni)
            assert s2.s2_last_launch_info(ctx)["i_per_thread"] == tiled and s2.s2_last_launch_info(ctx)["lanes_per_i"] == L
        for k in keys:
            assert np.array_equal(got[1][k], got[2][k]), (order, flags, S, tile, k)
    if order >= 4:
        ref, _ = oracle_on_gpu_prediction(ctx, w, order, il, w.eps2, h2, ngb_cap=24)
        check_forces(got[2], ref, s2.S2_FP32, order, flags, f"fp32 packed order {order}")
    s2.s2_close(ctx)


def test_fp32_fixup_meets_1e5_on_a_cancelling_sum():
    """Reading R-F32: config 3 holds a particle (address 17198) whose jerk is a 48 : 1 cancellation; plain fp32 pair
    arithmetic is at 1.9e-5 of the total there (and cannot do better, tests/test_fp32_conditioning.py).  The fp32 path
    flags such particles from sum_j q_j^2 and re-evaluates them with the fp64 sweep: with the fix-up every particle is
    within 1e-5; without it (s2_set_tuning key 9 = 4) this one is not; decisions and lists are untouched by it."""
    w = make_config(3)
    ctx = open_and_load(w, 4, precision=s2.S2_FP32, ngb_cap=32)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = np.concatenate([[17198], w.ilist(4095)]).astype(np.int32)
    il = il[np.sort(np.unique(il, return_index=True)[1])]
    h2 = np.full(il.size, (0.03) ** 2)
    ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, h2, ngb_cap=32)
    out = {}
    for fix in (4, 0):
        s2.s2_set_tuning(ctx, 9, fix)
        for shape in ({}, {0: 5, 1: 4}, {0: 3, 7: 2}):          # automatic, a j-split shape with slices, the tiled sweep with slices
            for k in range(8):
                s2.s2_set_tuning(ctx, k, shape.get(k, 0))
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
            res = s2.s2_get_results(ctx, il.size)
            lists = s2.s2_get_neighbours_csr(ctx, il.size)
            e = rel_err(res["jerk"], ref.jerk)
            out[(fix, tuple(shape.items()))] = (res, lists, e)
            n_fix = s2.s2_fp32_fixup_count(ctx)
            if fix == 4:
                assert e[0] > 1e-5 and n_fix == 0                 # plain fp32: the cancelling sum misses the tolerance
            else:
                assert e.max() <= 1e-5 and e[0] < 1e-12 and 1 <= n_fix <= il.size // 20, (e.max(), e[0], n_fix)
                check_forces(res, ref, s2.S2_FP32, 4, NN | NGB, f"fp32 fix-up {shape}")
    for key in [k for k in out if k[0] == 0]:
        a, b = out[key], out[(4, key[1])]
        for k in ("nn_id", "nn_r2", "ngb_count"):
            assert np.array_equal(a[0][k], b[0][k])
        assert np.array_equal(a[1][0], b[1][0]) and np.array_equal(a[1][1], b[1][1])
        same = a[2] == b[2]
        assert same.mean() > 0.9                                   # unflagged particles keep their fp32 bits
    print("fp32 fix-up: flagged", s2.s2_fp32_fixup_count(ctx), "of", il.size, "worst jerk error with / without:",
          out[(0, ())][2].max(), out[(4, ())][2].max())
    s2.s2_close(ctx)


@pytest.mark.parametrize("order", [4, 6])
def test_fp32_fixup_kernels_give_fp64_sums_when_every_particle_is_flagged(order):
    """The fix-up re-evaluates flagged i-particles with the fp64 pair arithmetic, cut into j-slices that the last warp
    to arrive adds up; flagged particles beyond the room of its partial-row buffer are swept unsliced.  Forcing EVERY
    particle to be flagged (s2_set_tuning key 9 = 5) runs both branches on all i: an fp32 context must then return
    sums within the FP64 tolerances of the oracle, bit-identically from call to call, for address lists and explicit
    sinks, with decisions and lists unchanged."""
    w = make_config(4 if order == 6 else 5, N=3000, order=order)
    ctx = open_and_load(w, order, precision=s2.S2_FP32, ngb_cap=24)
    s2.s2_predict(ctx, w.t_pred, w.N)
    tol = dict(acc=1e-13, pot=1e-13, jerk=1e-12, snap=1e-12)
    for ni, shape in ((700, {}), (700, {0: 3, 1: 4}), (3000, {}), (37, {0: 5, 1: 32}), (1, {})):
        il = w.ilist(ni)
        h2 = w.h2[il] * 0.6
        ref, (xp, vp, ap) = oracle_on_gpu_prediction(ctx, w, order, il, w.eps2, h2, ngb_cap=24)
        for k in range(9):
            s2.s2_set_tuning(ctx, k, shape.get(k, 0))
        s2.s2_set_tuning(ctx, 9, 5)
        runs = []
        for _ in range(2):
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
            runs.append(s2.s2_get_results(ctx, ni))
        res = runs[0]
        assert s2.s2_fp32_fixup_count(ctx) == ni
        for q in ("acc", "jerk", "pot") + (("snap",) if order == 6 else ()):
            assert np.array_equal(runs[0][q], runs[1][q]), (ni, q)
            e = rel_err(res[q], getattr(ref, q)).max()
            assert e <= tol[q], f"order {order} n_i {ni} {shape}: {q} {e:.2e} with every particle re-evaluated in fp64"
        check_nn_ld(res, ref, f"all flagged n_i {ni}")
        assert np.array_equal(res["ngb_count"], ref.ngb_count)
        check_neighbour_lists(ctx, ref, ni, 24, f"all flagged n_i {ni}", counts=res["ngb_count"])
    # explicit sinks (the i-state comes from the caller's planes, not from the j-store)
    rng = np.random.default_rng(3)
    ni = 90
    xi, vi, ai = rng.normal(size=(ni, 3)) * 0.5, rng.normal(size=(ni, 3)) * 0.3, rng.normal(size=(ni, 3))
    ids = np.full(ni, -1, np.int32)
    for k in range(9):
        s2.s2_set_tuning(ctx, k, 0)
    s2.s2_set_tuning(ctx, 9, 5)
    s2.s2_calc_explicit(ctx, ids, xi, vi, ai if order == 6 else None, None, w.eps2, 0)
    res = s2.s2_get_results(ctx, ni)
    xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, w.N)
    ref = oracle.forces(order, w.mass, w.ident, xp, vp, ap, ids, xi, vi, ai if order == 6 else None, w.eps2)
    for q in ("acc", "jerk", "pot") + (("snap",) if order == 6 else ()):
        assert rel_err(res[q], getattr(ref, q)).max() <= tol[q], ("explicit", q)
    s2.s2_close(ctx)
