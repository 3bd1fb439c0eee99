"""Randomised sweep over problem sizes with the AUTOMATIC launch shape (the other GPU tests mostly force shapes):
seeded random (N, n_i, order, precision, flags, neighbour cap) against the oracle.  Catches balancer choices that
the fixed-size tests never reach (odd slice counts, warp columns with few i, tiled path with ragged i-groups)."""
import numpy as np
import pytest

import oracle
import paper_1510_04068_b200 as s2
from workloads import make_config

from gpu_util import TOL, check_neighbour_lists, check_nn_ld, rel_err

pytestmark = pytest.mark.gpu

NN, NGB = s2.S2_WANT_NN, s2.S2_WANT_NGB


@pytest.mark.parametrize("seed", range(6))
def test_random_problems_automatic_shape(seed):
    rng = np.random.default_rng(1000 + seed)
    shapes_seen = set()
    for case in range(8):
        order = int(rng.choice([2, 4, 6]))
        P = int(rng.choice([s2.S2_FP64, s2.S2_DS, s2.S2_FP32]))
        N = int(rng.choice([1, 2, 3, 31, 33, 255, 257, 1000, 2049, 4097, 6000, 9001]))
        cap = int(rng.choice([4, 24, 64]))
        w = make_config(4 if order == 6 else 5, N=max(N, 4), order=order if order != 2 else 4)
        ctx = s2.s2_open(0, order, P, nj_capacity=max(N, 1), ngb_cap=cap)
        addr = np.arange(N, dtype=np.int32)
        s2.s2_set_j(ctx, addr, w.ident[:N], w.t_j[:N], w.mass[:N], w.pos[:N], w.vel[:N], w.acc[:N], w.jerk[:N],
                    w.snap[:N] if order == 6 else None, w.crackle[:N] if order == 6 else None)
        s2.s2_commit_j(ctx)
        s2.s2_predict(ctx, w.t_pred, N)
        xp, vp, ap = s2.s2_get_predicted_j(ctx, 0, N)
        for ni in sorted({1, N, int(rng.integers(1, N + 1)), int(rng.integers(1, N + 1))}):
            flags = int(rng.choice([0, NN, NN | NGB]))
            il = rng.permutation(N)[:ni].astype(np.int32)
            h2 = (w.h2[il] * rng.uniform(0.2, 3.0)) if flags & NGB else None
            s2.s2_calc_ilist(ctx, il, h2, w.eps2, flags)
            res = s2.s2_get_results(ctx, ni)
            info = s2.s2_last_launch_info(ctx)
            shapes_seen.add((info["lanes_per_i"], info["warp_columns"], info["i_per_thread"], info["reduced"]))
            oo = 4 if order == 2 else order
            ref = oracle.forces_ilist(oo, w.mass[:N], w.ident[:N], xp, vp, ap if order == 6 else None, il, w.eps2, h2, cap)
            what = f"seed {seed} case {case}: order {order} prec {P} N {N} n_i {ni} flags {flags} cap {cap} {info}"
            tol = TOL[P]
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
    assert len(shapes_seen) >= 3
