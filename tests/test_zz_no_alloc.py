"""s2_forces_noalloc (include/s2b200.h): the j-split sweep + combine with its partial sums in a static device array, for
callers that cannot call cudaMalloc.  Checked against the EXISTING path (s2_calc_ilist + s2_get_results on a context)
on the same predicted particles, within the tolerances the other fp64 GPU tests use (acc, pot 1e-13; jerk 1e-12), on
calls made in a row: the scratch array keeps the previous call's contents, so the sequence large list -> small list ->
another large list would expose any stale row that is read.

Collected last on purpose (the name sorts after every other test file): the suite runs with pytest -x, and a failure
here must not hide the other tests.  Runs the same alone in a fresh process and after the other tests."""
import numpy as np
import pytest

import oracle
import paper_1510_04068_b200 as s2
from workloads import make_config

from gpu_util import TOL, open_and_load, rel_err

pytestmark = pytest.mark.gpu


def test_noalloc_entry_point_matches_the_context_path_on_calls_in_a_row():
    import torch
    dev = torch.device("cuda", 0)
    lim = s2.s2_noalloc_limits()
    assert lim["max_ni"] == 4096 and lim["scratch_bytes"] == 4 << 20

    w = make_config(3, N=8192)
    ctx = open_and_load(w, 4)
    s2.s2_predict(ctx, w.t_pred, w.N)
    xp, vp, _ = s2.s2_get_predicted_j(ctx, 0, w.N)            # the fp64 predicted state both paths work on
    d_pos, d_vel = torch.from_numpy(xp).to(dev), torch.from_numpy(vp).to(dev)
    d_mass, d_id = torch.from_numpy(w.mass).to(dev), torch.from_numpy(w.ident).to(dev)

    rng = np.random.default_rng(77)
    lists = [rng.permutation(w.N)[:4096].astype(np.int32),    # the maximum: 16 slices x 4096 rows fill the scratch
             w.ilist(37),                                     # then a short list: other slice count, stale rows all around
             rng.permutation(w.N)[:1000].astype(np.int32),    # then a mid-sized one again
             np.array([5], dtype=np.int32)]                   # and a single particle
    tol = TOL[s2.S2_FP64]
    free_before = None
    for k, il in enumerate(lists):
        ni = il.size
        d_il = torch.from_numpy(il).to(dev)
        d_acc = torch.full((ni * 3,), float("nan"), dtype=torch.float64, device=dev)
        d_jerk = torch.full((ni * 3,), float("nan"), dtype=torch.float64, device=dev)
        d_pot = torch.full((ni,), float("nan"), dtype=torch.float64, device=dev)
        torch.cuda.synchronize()
        if k >= 1:                                            # (the first call may still load the module lazily)
            free_before = torch.cuda.mem_get_info(0)[0]
        s2.s2_forces_noalloc(d_pos, d_vel, d_mass, d_id, d_il, w.eps2, d_acc, d_jerk, d_pot)
        torch.cuda.synchronize()
        if k >= 1:
            assert torch.cuda.mem_get_info(0)[0] == free_before, "the call changed the device's free memory"
        got = dict(acc=d_acc.cpu().numpy().reshape(-1, 3), jerk=d_jerk.cpu().numpy().reshape(-1, 3), pot=d_pot.cpu().numpy())

        # the existing path, same particles, same i-list
        s2.s2_calc_ilist(ctx, il, None, w.eps2, 0)
        ref = s2.s2_get_results(ctx, ni)
        what = f"call {k} (n_i = {ni})"
        for q in ("acc", "jerk", "pot"):
            assert np.isfinite(got[q]).all(), what
            e = rel_err(got[q], ref[q]).max()
            assert e <= tol[q], f"{what}: {q} differs from the context path by {e:.2e} > {tol[q]:.0e}"
        if ni <= 1000:                                        # and against the oracle, like every other parity test
            orc = oracle.forces_ilist(4, w.mass, w.ident, xp, vp, None, il, w.eps2)
            for q in ("acc", "jerk", "pot"):
                assert rel_err(got[q], getattr(orc, q)).max() <= tol[q], (what, q)

        # bit-reproducible: the same call again gives the same bits
        d_acc2, d_jerk2, d_pot2 = torch.empty_like(d_acc), torch.empty_like(d_jerk), torch.empty_like(d_pot)
        s2.s2_forces_noalloc(d_pos, d_vel, d_mass, d_id, d_il, w.eps2, d_acc2, d_jerk2, d_pot2)
        torch.cuda.synchronize()
        assert torch.equal(d_acc, d_acc2) and torch.equal(d_jerk, d_jerk2) and torch.equal(d_pot, d_pot2), what

    # sizes beyond the fixed scratch are rejected with a clear error, before anything is launched
    too_many = torch.zeros(lim["max_ni"] + 1, dtype=torch.int32, device=dev)
    out3, out1 = torch.empty(3 * too_many.numel(), dtype=torch.float64, device=dev), torch.empty(too_many.numel(), dtype=torch.float64, device=dev)
    with pytest.raises(s2.S2Error) as e:
        s2.s2_forces_noalloc(d_pos, d_vel, d_mass, d_id, too_many, w.eps2, out3, out3.clone(), out1)
    assert e.value.code == s2.S2_ERANGE and "4096" in str(e.value)
    # an address outside the j-particles gives NaN for that i only
    d_il = torch.tensor([3, w.N, 9], dtype=torch.int32, device=dev)
    a, j, p = (torch.empty(9, dtype=torch.float64, device=dev), torch.empty(9, dtype=torch.float64, device=dev),
               torch.empty(3, dtype=torch.float64, device=dev))
    s2.s2_forces_noalloc(d_pos, d_vel, d_mass, d_id, d_il, w.eps2, a, j, p)
    p = p.cpu().numpy()
    assert np.isnan(p[1]) and np.isfinite(p[0]) and np.isfinite(p[2])
    s2.s2_close(ctx)
