"""GPU parity tests: the CUDA library (through the C ABI) against the CPU oracle, element by
element, on the same seeded inputs.  Run on the B200 box with  pytest -m gpu."""
import numpy as np
import pytest

import oracle
import paper_1510_04068_b200 as s2
from workloads import make_config, lattice_workload

from gpu_util import (TOL, check_forces, check_neighbour_lists, open_and_load, oracle_on_gpu_prediction, rel_err)

pytestmark = pytest.mark.gpu

NN, NGB = s2.S2_WANT_NN, s2.S2_WANT_NGB


# ------------------------------------------------------------------------------- a1 / a2
@pytest.mark.parametrize("cfg,order,N", [(1, 4, 1024), (4, 6, 5000)])
def test_commit_roundtrip_and_predictor(cfg, order, N):
    w = make_config(cfg, N=N)
    ctx = open_and_load(w, order, chunks=3)
    ident, t, mass, pos = s2.s2_get_j(ctx, 0, N)
    assert np.array_equal(ident, w.ident) and np.array_equal(t, w.t_j)
    assert np.array_equal(mass, w.mass) and np.array_equal(pos, w.pos)
    s2.s2_predict(ctx, w.t_pred, N)
    xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, N)
    oxp, ovp, oap = oracle.predict(order, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk, w.snap, w.crackle)
    # reading P1(i): within 2 ulp of the magnitude of the Taylor terms
    dt = (w.t_pred - w.t_j)[:, None]
    u = 2.0 ** -52
    mx = np.abs(w.pos) + np.abs(w.vel * dt) + np.abs(w.acc * dt ** 2 / 2) + np.abs(w.jerk * dt ** 3 / 6)
    mv = np.abs(w.vel) + np.abs(w.acc * dt) + np.abs(w.jerk * dt ** 2 / 2)
    if order == 6:
        mx += np.abs(w.snap * dt ** 4 / 24) + np.abs(w.crackle * dt ** 5 / 120)
        mv += np.abs(w.snap * dt ** 3 / 6) + np.abs(w.crackle * dt ** 4 / 24)
        ma = np.abs(w.acc) + np.abs(w.jerk * dt) + np.abs(w.snap * dt ** 2 / 2) + np.abs(w.crackle * dt ** 3 / 6)
        assert (np.abs(ap - oap) <= 2 * u * ma).all()
    assert (np.abs(xp - oxp) <= 2 * u * mx).all()
    assert (np.abs(vp - ovp) <= 2 * u * mv).all()
    # dt = 0 returns the input bit-exactly; a second commit of a subset overwrites only that subset
    sub = np.arange(0, N, 7, dtype=np.int32)
    s2.s2_set_j(ctx, sub, w.ident[sub], np.full(sub.size, 0.5), w.mass[sub], w.pos[sub] + 1.0, w.vel[sub], w.acc[sub],
                w.jerk[sub], w.snap[sub] if order == 6 else None, w.crackle[sub] if order == 6 else None)
    s2.s2_commit_j(ctx)
    s2.s2_predict(ctx, 0.5, N)
    xp2, vp2, _ = s2.s2_get_predicted_j(ctx, 0, N)
    assert np.array_equal(xp2[sub], w.pos[sub] + 1.0) and np.array_equal(vp2[sub], w.vel[sub])
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- config 1
def test_cfg1_fp64_all_active_with_nn():
    """BASELINE config 1: N = 1024 Plummer, eps = 1e-3, all active, acc + jerk + pot + nn, fp64."""
    w = make_config(1)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(w.N)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
    res = s2.s2_get_results(ctx, w.N)
    ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2)
    errs = check_forces(res, ref, s2.S2_FP64, 4, NN, "cfg1")
    # end to end as well (oracle predictor + oracle forces; closest pair ~5e-3 -> P1)
    oxp, ovp, _ = oracle.predict(4, w.t_pred, w.t_j, w.pos, w.vel, w.acc, w.jerk)
    ref2 = oracle.forces_ilist(4, w.mass, w.ident, oxp, ovp, None, il, w.eps2)
    assert rel_err(res["acc"], ref2.acc).max() < 1e-13 and rel_err(res["jerk"], ref2.jerk).max() < 1e-12
    assert np.array_equal(res["nn_id"], ref2.nn_id)
    print("cfg1 max rel errors:", {k: f"{v:.2e}" for k, v in errs.items()})
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- config 2
def test_cfg2_small_n_sweep():
    """BASELINE config 2: N = 64, eps = 1e-4, n_i = 1, 2, 4 ... 64 (j-split path at every n_i)."""
    w = make_config(2)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    for ni in (1, 2, 3, 4, 8, 16, 32, 33, 64):
        il = w.ilist(ni)
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
        res = s2.s2_get_results(ctx, ni)
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2)
        check_forces(res, ref, s2.S2_FP64, 4, NN, f"cfg2 n_i={ni} shape={s2.s2_last_launch_info(ctx)}")
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- forced shapes
@pytest.mark.parametrize("order", [4, 6])
@pytest.mark.parametrize("flags", [0, NN, NN | NGB])
def test_all_launch_shapes_ragged(order, flags):
    """Every lanes-per-i / warp-column / slice shape on a ragged problem (N = 1000 is not a multiple
    of any tile, n_i = 37 leaves idle lanes) against the oracle, neighbour lists included."""
    w = make_config(4 if order == 6 else 5, N=1000, order=order)
    ctx = open_and_load(w, order, ngb_cap=24)
    s2.s2_predict(ctx, w.t_pred, w.N)
    ni = 37
    il = w.ilist(ni)
    h2 = w.h2[il] * 0.6 if flags & NGB else None
    ref, _ = oracle_on_gpu_prediction(ctx, w, order, il, w.eps2, h2, ngb_cap=24)
    shapes = [(L, 1, S, tile) for L in (1, 2, 4, 8, 16, 32) for S, tile in ((1, 0), (3, 64), (13, 32))]
    shapes += [(32, Wj, S, 0) for Wj in (2, 4, 8) for S in (1, 2, 5)]
    shapes += [(8, 4, 1, 0), (8, 8, 3, 64), (2, 2, 5, 128), (16, 2, 2, 32)]   # warp columns with several i per warp
    for L, Wj, S, tile in shapes:
        s2.s2_set_tuning(ctx, 1, L); s2.s2_set_tuning(ctx, 2, Wj); s2.s2_set_tuning(ctx, 0, S); s2.s2_set_tuning(ctx, 4, tile)
        # fused combine (auto / no / 2 / 8 CTA clusters), separate reduce kernel, and for one lane per i the
        # register-tiled sweep (several i per thread)
        # ... register-tiled sweep (several i per thread; with L > 1 lanes per i-slot for plain sums)
        modes = [(0, 0, 1), (3, 0, 1), (0, 2, 1), (0, 8, 1), (1, 0, 1)] + ([(0, 0, 2)] if (L == 1 or flags == 0) and Wj == 1 else [])
        for unfused, cluster, tiled in modes:
            s2.s2_set_tuning(ctx, 5, unfused); s2.s2_set_tuning(ctx, 6, cluster); s2.s2_set_tuning(ctx, 7, tiled)
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
            res = s2.s2_get_results(ctx, ni)
            info = s2.s2_last_launch_info(ctx)
            assert info["lanes_per_i"] == L and info["warp_columns"] == Wj and (info["i_per_thread"] > 1) == (tiled == 2)
            check_forces(res, ref, s2.S2_FP64, order, flags, f"shape {info}")
        if flags & NGB:
            assert res["overflow"] == bool((ref.ngb_count > 24).any())
            check_neighbour_lists(ctx, ref, ni, 24, f"shape {info}")
    s2.s2_close(ctx)


def test_neighbour_overflow_and_single_list():
    w = make_config(5, N=2048)
    ctx = open_and_load(w, 4, ngb_cap=8)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(300)
    h2 = w.h2[il]
    ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, h2, ngb_cap=8)
    assert (ref.ngb_count > 8).any()
    for S in (0, 1, 7):
        s2.s2_set_tuning(ctx, 0, S)
        s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
        res = s2.s2_get_results(ctx, 300)
        assert res["overflow"]
        assert np.array_equal(res["ngb_count"], ref.ngb_count)      # true counts (P8)
        check_neighbour_lists(ctx, ref, 300, 8, f"S={S}")              # the 8 lowest addresses, ascending
        k = int(np.argmax(ref.ngb_count))
        one = s2.s2_get_neighbours(ctx, k, 5)
        assert np.array_equal(one, ref.ngb_list[k][:5])
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- config 3
@pytest.mark.parametrize("ni", [1, 32, 256, 2048, 16384, 65536])
def test_cfg3_blockstep_fp64(ni):
    """BASELINE config 3 (fp64 leg): N = 65536, n_i in {1, 32, 256, 2048, 16384, 65536}, acc + jerk + pot.
    FULL oracle at every n_i (4.3e9 long-double pair terms at n_i = N, ~20 s on the box's cores)."""
    w = make_config(3)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(ni)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=0)
    res = s2.s2_get_results(ctx, ni)
    ref, (xp, vp, _) = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2)
    errs = check_forces(res, ref, s2.S2_FP64, 4, 0, f"cfg3 n_i={ni} {s2.s2_last_launch_info(ctx)}")
    print(f"cfg3 n_i={ni} (oracle on all {ni} i, workload seed {w.seed})", s2.s2_last_launch_info(ctx),
          {k: f"{v:.2e}" for k, v in errs.items()})
    if ni == w.N:   # Newton's third law on the full GPU output
        for q in ("acc", "jerk"):
            tot = np.abs((w.mass[il, None] * res[q]).sum(0)).max()
            scale = (w.mass[il] * np.linalg.norm(res[q], axis=1)).sum()
            assert tot <= 1e-11 * scale
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- determinism
def test_bit_reproducible_and_paths_agree():
    w = make_config(3, N=8192)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(96)
    outs = {}
    for S in (0, 1, 9):
        s2.s2_set_tuning(ctx, 0, S)
        runs = []
        for _ in range(10):
            s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
            r = s2.s2_get_results(ctx, 96)
            runs.append(np.concatenate([r["acc"].ravel(), r["jerk"].ravel(), r["pot"], r["nn_r2"]]))
        for r in runs[1:]:
            assert np.array_equal(r, runs[0]), "results differ run to run"
        outs[S] = runs[0]
    assert np.allclose(outs[1], outs[9], rtol=1e-12, atol=0)
    assert np.allclose(outs[0], outs[1], rtol=1e-12, atol=0)
    # the fused combine (last CTA of an i-group reduces) and the separate reduce kernel add the slice
    # partials in the same fixed order: bit-identical results
    s2.s2_set_tuning(ctx, 0, 9)
    s2.s2_set_tuning(ctx, 5, 3)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
    assert s2.s2_last_launch_info(ctx)["reduced"] == 2
    s2.s2_set_tuning(ctx, 5, 1)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)
    assert s2.s2_last_launch_info(ctx)["reduced"] == 1
    r = s2.s2_get_results(ctx, 96)
    assert np.array_equal(np.concatenate([r["acc"].ravel(), r["jerk"].ravel(), r["pot"], r["nn_r2"]]), outs[9])
    s2.s2_close(ctx)


@pytest.mark.parametrize("order", [4, 6])
def test_thread_per_i_reduce_has_the_bits_of_the_warp_reduce(order):
    """With 2-16 partial rows and >= 4096 i-particles reduce_thread_kernel (one thread per i, coalesced) replaces
    reduce_kernel (one warp per i); it adds the rows in the tree order of the warp butterfly, so an i-particle gets
    the same bits from a 4095-particle call (warp kernel) and a 4096-particle call (thread kernel)."""
    w = make_config(4 if order == 6 else 3, N=8192)
    ctx = open_and_load(w, order)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(4096)
    for S in (2, 3, 5, 8, 9, 13, 16):
        for flags in (0, NN):
            s2.s2_set_tuning(ctx, 0, S); s2.s2_set_tuning(ctx, 1, 1); s2.s2_set_tuning(ctx, 7, 1); s2.s2_set_tuning(ctx, 5, 1)
            s2.s2_calc_ilist(ctx, il[:4095], eps2=w.eps2, flags=flags)
            a = s2.s2_get_results(ctx, 4095)
            s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=flags)
            assert s2.s2_last_launch_info(ctx)["reduced"] == 1 and s2.s2_last_launch_info(ctx)["S"] == S
            b = s2.s2_get_results(ctx, 4096)
            for k in ("acc", "jerk", "pot", "nn_id", "nn_r2") + (("snap",) if order == 6 else ()):
                assert np.array_equal(a[k], b[k][:4095]), (S, flags, k)
            ref, _ = oracle_on_gpu_prediction(ctx, w, order, il, w.eps2)
            check_forces(b, ref, s2.S2_FP64, order, flags, f"thread reduce S={S}")
    s2.s2_close(ctx)


def test_atomic_combine_option():
    """the paper's single-kernel combine by atomics (L88) as an opt-in (s2_set_tuning key 5 = 2).
    Within tolerance of the oracle, equal to the deterministic combine up to summation order, and never used when
    nearest neighbours are requested (those need the ordered min-by-address combine)."""
    w = make_config(3, N=8192)
    ctx = open_and_load(w)
    s2.s2_predict(ctx, w.t_pred, w.N)
    for ni, shape in ((96, {0: 9}), (700, {0: 5, 1: 1}), (3000, {0: 3, 7: 2})):
        il = w.ilist(ni)
        for k in range(9):
            s2.s2_set_tuning(ctx, k, 0)
        for k, v in shape.items():
            s2.s2_set_tuning(ctx, k, v)
        s2.s2_set_tuning(ctx, 5, 1)
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2)
        det = s2.s2_get_results(ctx, ni)
        assert s2.s2_last_launch_info(ctx)["reduced"] == 1
        s2.s2_set_tuning(ctx, 5, 2)
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2)
        info = s2.s2_last_launch_info(ctx)
        assert info["reduced"] == 4, info
        res = s2.s2_get_results(ctx, ni)
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2)
        check_forces(res, ref, s2.S2_FP64, 4, 0, f"atomic combine {info}")
        assert np.allclose(res["acc"], det["acc"], rtol=1e-12, atol=0) and np.allclose(res["pot"], det["pot"], rtol=1e-13)
        assert (res["nn_id"] == -1).all() and np.isinf(res["nn_r2"]).all()
        s2.s2_calc_ilist(ctx, il, eps2=w.eps2, flags=NN)     # decisions requested: deterministic combine
        assert s2.s2_last_launch_info(ctx)["reduced"] == 1
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2)
        check_forces(s2.s2_get_results(ctx, ni), ref, s2.S2_FP64, 4, NN, "atomic option with NN")
    s2.s2_close(ctx)


def test_zero_copy_small_calls_equal_copied_ones():
    """Small host calls (n_i <= 128) let the kernels read the i-list from and write the records to pinned host memory
    (no copy operation enqueued).  Results, neighbour lists and error codes are bit-identical to the copied path
    (s2_set_tuning key 9 = 1), also when several calls are enqueued back to back (alternating i-list buffers)."""
    for cfg, N in ((2, 64), (3, 8192)):
        w = make_config(cfg, N=N)
        ctx = open_and_load(w, 4, ngb_cap=8)
        s2.s2_predict(ctx, w.t_pred, w.N)
        for ni in (1, 7, 64, 128, 129):
            ni = min(ni, N)
            il = w.ilist(ni)
            h2 = w.h2[il] * 4.0
            out = {}
            for zc in (1, 0):
                s2.s2_set_tuning(ctx, 9, zc)
                for junk in (w.ilist(min(N, 3)), w.ilist(min(N, 100))):      # enqueued before, never read back
                    s2.s2_calc_ilist(ctx, junk, None, w.eps2, 0)
                s2.s2_calc_ilist(ctx, il, h2, w.eps2, NN | NGB)
                r = s2.s2_get_results(ctx, ni)
                off, lst = s2.s2_get_neighbours_csr(ctx, ni)
                one = s2.s2_get_neighbours(ctx, ni - 1, 8)
                out[zc] = (r, off, lst, one)
            a, b = out[1], out[0]
            for k in ("acc", "jerk", "pot", "nn_id", "nn_r2", "ngb_count"):
                assert np.array_equal(a[0][k], b[0][k]), (cfg, ni, k)
            assert a[0]["overflow"] == b[0]["overflow"]
            assert np.array_equal(a[1], b[1]) and np.array_equal(a[2], b[2]) and np.array_equal(a[3], b[3])
            ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, h2, ngb_cap=8)
            check_forces(b[0], ref, s2.S2_FP64, 4, NN | NGB, f"zero-copy cfg {cfg} n_i {ni}")
        s2.s2_close(ctx)


# ------------------------------------------------------------------------------- ties
def test_lattice_ties_and_strictness_gpu():
    w = lattice_workload(4, 0.25)
    ctx = open_and_load(w, 4, ngb_cap=32)
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
            check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, f"lattice h2={h2v} L={L}")
            check_neighbour_lists(ctx, ref, w.N, 32)
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- explicit i, edge cases
def test_explicit_sinks_and_degenerate_sizes():
    w = make_config(1, N=300)
    ctx = open_and_load(w, 4, ngb_cap=16)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)
    rng = np.random.default_rng(5)
    ni = 45
    xi = rng.normal(size=(ni, 3)) * 0.5
    vi = rng.normal(size=(ni, 3)) * 0.3
    ids = np.full(ni, -1, np.int32)
    ids[::3] = w.ident[:15]                 # some sinks coincide in id with a source: that source is skipped
    h2 = np.full(ni, 0.05)
    s2.s2_calc_explicit(ctx, ids, xi, vi, None, h2, w.eps2, NN | NGB)
    res = s2.s2_get_results(ctx, ni)
    ref = oracle.forces(4, w.mass, w.ident, xp, vp, None, ids, xi, vi, None, w.eps2, h2, 16)
    check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, "explicit")
    check_neighbour_lists(ctx, ref, ni, 16)
    s2.s2_close(ctx)

    # N = 1 (only self): all zero, nn = -1 / +inf;  N = 2: each sees only the other
    for N in (1, 2):
        w = make_config(1, N=64)
        ctx = open_and_load(w, 4, nj=N)
        s2.s2_predict(ctx, w.t_pred, N)
        il = np.arange(N, dtype=np.int32)
        s2.s2_calc_ilist(ctx, il, np.full(N, 100.0), w.eps2, NN | NGB)
        res = s2.s2_get_results(ctx, N)
        ref, _ = oracle_on_gpu_prediction(ctx, w, 4, il, w.eps2, np.full(N, 100.0), nj=N)
        if N == 1:
            assert not res["acc"].any() and not res["jerk"].any() and res["pot"][0] == 0.0
            assert res["nn_id"][0] == -1 and np.isinf(res["nn_r2"][0]) and res["ngb_count"][0] == 0
        else:
            check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, "N=2")
            assert list(res["ngb_count"]) == [1, 1]
        s2.s2_close(ctx)


def test_state_and_argument_errors():
    w = make_config(1, N=64)
    ctx = s2.s2_open(0, 4, s2.S2_FP64, nj_capacity=64, ngb_cap=0)
    with pytest.raises(s2.S2Error) as e:
        s2.s2_predict(ctx, 0.0, 64)
    assert e.value.code == s2.S2_ESTATE
    with pytest.raises(s2.S2Error) as e:
        s2.s2_set_j(ctx, np.array([64], np.int32), w.ident[:1], w.t_j[:1], w.mass[:1], w.pos[:1], w.vel[:1], w.acc[:1], w.jerk[:1])
    assert e.value.code == s2.S2_ERANGE
    a = np.arange(64, dtype=np.int32)
    s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
    with pytest.raises(s2.S2Error) as e:      # staged but not committed
        s2.s2_predict(ctx, 0.0, 64)
    assert e.value.code == s2.S2_ESTATE
    s2.s2_commit_j(ctx)
    with pytest.raises(s2.S2Error) as e:
        s2.s2_calc_ilist(ctx, a[:4], eps2=1e-4)
    assert e.value.code == s2.S2_ESTATE
    s2.s2_predict(ctx, 0.0, 64)
    with pytest.raises(s2.S2Error) as e:
        s2.s2_get_results(ctx, 4)
    assert e.value.code == s2.S2_ESTATE
    with pytest.raises(s2.S2Error) as e:      # neighbour lists need ngb_cap > 0 and h2
        s2.s2_calc_ilist(ctx, a[:4], np.ones(4), 1e-4, NGB)
    assert e.value.code == s2.S2_EINVAL
    with pytest.raises(s2.S2Error) as e:
        s2.s2_calc_ilist(ctx, np.array([70], np.int32), eps2=1e-4)
    assert e.value.code == s2.S2_ERANGE
    s2.s2_calc_ilist(ctx, a[:4], eps2=1e-4)
    assert s2.s2_get_results(ctx, 4)["pot"].shape == (4,)
    assert s2.s2_kernel_launches(ctx) >= 3
    s2.s2_close(ctx)


# ------------------------------------------------------------------------------- config 4 (6th order)
def test_cfg4_sixth_order_ni1024():
    """BASELINE config 4: N = 262144 Salpeter Plummer, 6th order fp64, n_i = 1024 (full oracle)."""
    w = make_config(4)
    ctx = open_and_load(w, 6)
    s2.s2_predict(ctx, w.t_pred, w.N)
    il = w.ilist(1024)
    s2.s2_calc_ilist(ctx, il, eps2=w.eps2)
    res = s2.s2_get_results(ctx, 1024)
    ref, _ = oracle_on_gpu_prediction(ctx, w, 6, il, w.eps2)
    errs = check_forces(res, ref, s2.S2_FP64, 6, 0, f"cfg4 n_i=1024 {s2.s2_last_launch_info(ctx)}")
    print("cfg4 n_i=1024", s2.s2_last_launch_info(ctx), {k: f"{v:.2e}" for k, v in errs.items()})
    s2.s2_close(ctx)


@pytest.mark.parametrize("kind", ["plummer", "lattice", "plummer-fp32"])
def test_j_sharded_partials_combine_to_the_unsharded_result(kind):
    """j-sharding: three "ranks" run one after the other on this GPU, each a context that
    holds the whole store and sums over its own address block (s2_set_j_range).  Their partial results, combined the
    way sharding.combine_partials / combine_neighbour_lists do across ranks (sum; nn by smallest r2, ties to the lower
    rank; lists concatenated in rank order, truncated to the cap), must equal the oracle over all j: sums within
    tolerance, nearest neighbours, counts and lists exactly -- exact ties on the lattice included."""
    import torch
    from paper_1510_04068_b200.sharding import ShardedForces, merge_rank_lists
    P = s2.S2_FP32 if kind.endswith("fp32") else s2.S2_FP64     # fp32: every shard flags and re-evaluates on its own partial sums
    w = make_config(5, N=5000) if kind.startswith("plummer") else lattice_workload(12, 0.25)
    cap = 16
    world = 3
    ni = 700
    il = w.ilist(ni)
    h2 = w.h2[il] * (2.0 if kind.startswith("plummer") else 1.0)
    d_il, d_h2 = torch.from_numpy(il).cuda(), torch.from_numpy(np.ascontiguousarray(h2)).cuda()
    parts = []
    for r in range(world):
        sf = ShardedForces(w.N, order=4, precision=P, ngb_cap=cap, rank=r, world=world)
        sf.set_all_j(w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
        p = sf.partial(w.t_pred, d_il, d_h2, w.eps2, NN | NGB)
        parts.append({k: (v.clone() if v is not None else None) for k, v in p.items()})
        if r == 0:
            xp, vp, _ = s2.s2_get_predicted_j(sf.ctx, 0, w.N)
        sf.close()
    acc = sum(p["acc"] for p in parts).view(-1, 3).cpu().numpy()
    jerk = sum(p["jerk"] for p in parts).view(-1, 3).cpu().numpy()
    pot = sum(p["pot"] for p in parts).cpu().numpy()
    cnt = sum(p["ngb_count"] for p in parts).cpu().numpy()
    best_r2, best_id = parts[0]["nn_r2"].clone(), parts[0]["nn_id"].clone()
    for p in parts[1:]:
        better = p["nn_r2"] < best_r2
        best_r2, best_id = torch.where(better, p["nn_r2"], best_r2), torch.where(better, p["nn_id"], best_id)
    off, lst = merge_rank_lists([(p["offsets"][1:] - p["offsets"][:-1]) for p in parts], [p["list"] for p in parts], cap)
    off, lst = off.cpu().numpy(), lst.cpu().numpy()
    ref = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, h2, cap)
    res = dict(acc=acc, jerk=jerk, pot=pot, nn_id=best_id.cpu().numpy(), nn_r2=best_r2.cpu().numpy(), ngb_count=cnt)
    check_forces(res, ref, P, 4, NN | NGB, f"j-sharded {kind}")
    assert (ref.ngb_count > cap).any() or kind == "lattice"
    for i in range(ni):
        want = ref.ngb_list[i][ref.ngb_list[i] >= 0]
        assert np.array_equal(lst[off[i]:off[i + 1]], want), (kind, i)


def _nccl_jshard_worker(rank, world, port, q):
    import os
    import torch
    import torch.distributed as dist
    from paper_1510_04068_b200.sharding import ShardedForces
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    w = make_config(5, N=5000)
    il = w.ilist(700)
    sf = ShardedForces(w.N, order=4, device=rank, ngb_cap=16)
    sf.set_all_j(w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
    dev = torch.device("cuda", rank)
    out = sf.forces(w.t_pred, torch.from_numpy(il).to(dev), torch.from_numpy(np.ascontiguousarray(w.h2[il] * 2.0)).to(dev),
                    w.eps2, NN | NGB)
    if rank == 0:
        xp, vp, _ = s2.s2_get_predicted_j(sf.ctx, 0, w.N)
        q.put(({k: (v.cpu().numpy() if v is not None else None) for k, v in out.items()}, xp, vp))
    dist.barrier()
    sf.close()
    dist.destroy_process_group()


def test_j_sharded_forces_two_ranks_nccl():
    """The same combine through NCCL with one process per GPU; needs two devices (skips on the one-GPU test box)."""
    import socket
    import torch
    import torch.multiprocessing as mp
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_nccl_jshard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got, xp, vp = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    w = make_config(5, N=5000)
    il = w.ilist(700)
    ref = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2, w.h2[il] * 2.0, 16)
    res = dict(acc=got["acc"].reshape(-1, 3), jerk=got["jerk"].reshape(-1, 3), pot=got["pot"], nn_id=got["nn_id"],
               nn_r2=got["nn_r2"], ngb_count=got["ngb_count"])
    check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, "j-sharded, 2 ranks over NCCL")
    for i in range(il.size):
        want = ref.ngb_list[i][ref.ngb_list[i] >= 0]
        assert np.array_equal(got["list"][got["offsets"][i]:got["offsets"][i + 1]], want), i


def test_batched_small_calls_match_single_calls():
    """s2_calc_ilist_batch: k i-lists in one launch sequence and one synchronisation (config 2's regime: a small call is
    latency-bound).  Each list's segment of the results equals the list's own call within rounding, decisions and
    neighbour lists exactly, and the whole matches the oracle."""
    w = make_config(2)
    ctx = open_and_load(w, 4, ngb_cap=16)
    s2.s2_predict(ctx, w.t_pred, w.N)
    rng = np.random.default_rng(8)
    lists = [rng.permutation(w.N)[:n].astype(np.int32) for n in (1, 7, 64, 3, 32, 1, 20)]
    h2s = [w.h2[l] * 3.0 for l in lists]
    off = s2.s2_calc_ilist_batch(ctx, lists, h2s, w.eps2, NN | NGB)
    tot = int(off[-1])
    res = s2.s2_get_results(ctx, tot)
    coff, clst = s2.s2_get_neighbours_csr(ctx, tot)
    cat, h2 = np.concatenate(lists), np.concatenate(h2s)
    ref, _ = oracle_on_gpu_prediction(ctx, w, 4, cat, w.eps2, h2, ngb_cap=16)
    check_forces(res, ref, s2.S2_FP64, 4, NN | NGB, "batch")
    check_neighbour_lists(ctx, ref, tot, 16, "batch", counts=res["ngb_count"])
    for b, (l, hh) in enumerate(zip(lists, h2s)):
        s2.s2_calc_ilist(ctx, l, hh, w.eps2, NN | NGB)
        one = s2.s2_get_results(ctx, l.size)
        o1, l1 = s2.s2_get_neighbours_csr(ctx, l.size)
        seg = slice(off[b], off[b + 1])
        assert rel_err(res["acc"][seg], one["acc"]).max() < 1e-13 and rel_err(res["jerk"][seg], one["jerk"]).max() < 1e-12
        for k in ("nn_id", "nn_r2", "ngb_count"):
            assert np.array_equal(res[k][seg], one[k]), (b, k)
        assert np.array_equal(clst[coff[off[b]]:coff[off[b + 1]]], l1)
    s2.s2_close(ctx)


def test_contexts_on_two_devices_in_one_process():
    """The > 48 KB shared-memory opt-in and the bank hand-over state are per device: contexts on two devices of one
    process (the paper's multi-GPU mode is single-process, L80) must both run the large-tile sweeps and the
    uniform-operand sweep.  Needs two GPUs (skips on the one-GPU test box)."""
    import torch
    if torch.cuda.device_count() < 2:
        pytest.skip("needs two GPUs")
    w = make_config(3, N=9000)
    il = w.ilist(w.N)
    out = []
    for dev in (0, 1):
        with torch.cuda.device(dev):
            ctx = s2.s2_open(dev, 4, s2.S2_FP64, nj_capacity=w.N, ngb_cap=0)
            a = np.arange(w.N, dtype=np.int32)
            s2.s2_set_j(ctx, a, w.ident, w.t_j, w.mass, w.pos, w.vel, w.acc, w.jerk)
            s2.s2_commit_j(ctx)
            s2.s2_predict(ctx, w.t_pred, w.N)
            res = {}
            for key8 in (1, 2):
                s2.s2_set_tuning(ctx, 8, key8)
                s2.s2_calc_ilist(ctx, il, None, w.eps2, 0)
                res[key8] = s2.s2_get_results(ctx, w.N)
            out.append(res)
            s2.s2_close(ctx)
    for k in ("acc", "jerk", "pot"):
        assert np.array_equal(out[0][1][k], out[1][1][k]) and np.array_equal(out[0][2][k], out[1][2][k])
