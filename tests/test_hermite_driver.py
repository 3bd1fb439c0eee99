"""Block-time-step Hermite driver (sec 3.7).

CPU part: the host integrator itself, driven by the oracle, conserves energy and uses genuinely varying
active sets.  GPU part: the same driver on libs2b200 follows the oracle-driven run step for step."""
import numpy as np
import pytest

from paper_1510_04068_b200.hermite import Hermite4, Hermite6
from workloads import make_config

from hermite_util import OracleBackend


def _plummer(n):
    w = make_config(1, N=n)                       # equal masses, eps = 1e-3
    return w


def test_driver_on_oracle_conserves_energy_and_blocks_vary():
    w = _plummer(96)
    h = Hermite4(OracleBackend(w.N, w.eps2), w.mass, w.pos, w.vel, eta=0.01)
    e0 = h.energy()
    h.run_until(0.25)
    e1 = h.energy()
    assert abs((e1 - e0) / e0) < 2e-7, (e0, e1)
    sizes = np.array(h.active_hist)
    assert sizes.min() < w.N // 8 and sizes.max() == w.N            # from a few particles to a full synchronisation
    assert np.all(np.log2(h.dt) == np.round(np.log2(h.dt)))          # power-of-two steps
    assert np.all(np.fmod(h.t, h.dt) == 0.0)                         # block-aligned
    # individual time steps break exact pairwise symmetry in time; momentum stays at the truncation-error level
    p = (w.mass[:, None] * h.v).sum(0)
    assert np.abs(p).max() < 1e-7


@pytest.mark.gpu
@pytest.mark.parametrize("precision,tol", [("fp64", 1e-9), ("ds", 1e-7)])
def test_driver_gpu_follows_oracle_run(precision, tol):
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import S2Backend
    w = _plummer(256)
    P = {"fp64": s2.S2_FP64, "ds": s2.S2_DS}[precision]
    gb = S2Backend(w.N, w.eps2, precision=P)
    g = Hermite4(gb, w.mass, w.pos, w.vel)
    o = Hermite4(OracleBackend(w.N, w.eps2), w.mass, w.pos, w.vel)
    e0 = g.energy()
    for _ in range(150):                                             # block steps in lock-step
        na, nb = g.step(), o.step()
        assert na == nb and g.time == o.time
    assert np.array_equal(g.t, o.t) and np.array_equal(g.dt, o.dt)
    assert np.abs(g.x - o.x).max() < tol and np.abs(g.v - o.v).max() < tol
    g.run_until(0.125)
    o.run_until(0.125)
    assert np.abs(g.x - o.x).max() < 100 * tol
    e1 = g.energy()
    print(f"{precision}: block steps {g.block_steps}, mean active {np.mean(g.active_hist):.1f}, "
          f"force calls {gb.calls}, dE/E = {(e1 - e0) / e0:.2e}, max |dx| vs oracle run {np.abs(g.x - o.x).max():.2e}")
    assert abs((e1 - e0) / e0) < 1e-6
    gb.close()


def test_sixth_order_driver_on_oracle_conserves_energy():
    """6th-order scheme (sec 3.7: eta_6 = 0.1) driven by the oracle: energy and a 4th-order cross-check."""
    w = _plummer(64)
    h6 = Hermite6(OracleBackend(w.N, w.eps2, order=6), w.mass, w.pos, w.vel, eta=0.1)
    e0 = h6.energy()
    h6.run_until(0.25)
    e1 = h6.energy()
    assert abs((e1 - e0) / e0) < 1e-8, (e0, e1)
    h4 = Hermite4(OracleBackend(w.N, w.eps2), w.mass, w.pos, w.vel, eta=0.002)      # a tight 4th-order run
    h4.run_until(0.25)
    assert np.abs(h6.x - h4.x).max() < 2e-6                                         # same trajectory
    assert min(h6.active_hist) < w.N // 4 and max(h6.active_hist) == w.N


@pytest.mark.gpu
def test_sixth_order_driver_gpu_follows_oracle_run():
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import S2Backend
    w = _plummer(256)
    gb = S2Backend(w.N, w.eps2, precision=s2.S2_FP64, order=6)
    g = Hermite6(gb, w.mass, w.pos, w.vel)
    o = Hermite6(OracleBackend(w.N, w.eps2, order=6), w.mass, w.pos, w.vel)
    e0 = g.energy()
    for _ in range(120):
        na, nb = g.step(), o.step()
        assert na == nb and g.time == o.time
    assert np.array_equal(g.dt, o.dt)
    assert np.abs(g.x - o.x).max() < 1e-10 and np.abs(g.v - o.v).max() < 1e-9
    g.run_until(0.125)
    e1 = g.energy()
    print(f"6th order: block steps {g.block_steps}, mean active {np.mean(g.active_hist):.1f}, dE/E = {(e1 - e0) / e0:.2e}")
    assert abs((e1 - e0) / e0) < 1e-8
    gb.close()


@pytest.mark.gpu
@pytest.mark.parametrize("order,precision,steps,tol,averaged", [(4, "fp64", 300, 1e-9, False), (4, "ds", 150, 1e-7, False),
                                                                (6, "fp64", 150, 1e-9, False), (6, "fp64", 150, 1e-9, True),
                                                                (6, "ds", 100, 1e-7, True)])
def test_device_integrator_follows_host_reference_in_lockstep(order, precision, steps, tol, averaged):
    """The device-resident integrator (s2_bts_*: corrector, time-step rule and active-set selection in kernels, the
    j-store as particle state) against hermite.py driven by the ORACLE, block step by block step: same active counts and
    block times at every step, identical t and dt arrays, positions and velocities within tol."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = _plummer(256)
    P = {"fp64": s2.S2_FP64, "ds": s2.S2_DS}[precision]
    d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, precision=P, averaged=averaged)
    o = (Hermite4(OracleBackend(w.N, w.eps2), w.mass, w.pos, w.vel) if order == 4 else
         Hermite6(OracleBackend(w.N, w.eps2, order=6), w.mass, w.pos, w.vel, averaged=averaged))
    st = d.state()
    assert np.array_equal(st["dt"], o.dt) and np.allclose(st["acc"], o.a, rtol=1e-9, atol=0)
    for k in range(steps):
        na, nb = d.step(), o.step()
        assert na == nb and d.time == o.time, (k, na, nb, d.time, o.time)
    st = d.state()
    assert np.array_equal(st["t"], o.t) and np.array_equal(st["dt"], o.dt)
    assert np.abs(st["pos"] - o.x).max() < tol and np.abs(st["vel"] - o.v).max() < tol
    assert np.array_equal(d.history(), np.array(o.active_hist))
    stats = d.stats()
    assert stats["block_steps"] == steps and stats["particle_steps"] == sum(o.active_hist)
    d.close()


@pytest.mark.gpu
def test_device_integrator_conserves_energy_and_reaches_t_end():
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(1, N=1024)
    for order, lim in ((4, 1e-6), (6, 1e-7)):
        d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order)
        e0 = d.energy()
        d.run_until(0.125)
        st = d.state()
        assert (st["t"] == 0.125).all() and st["time"] == 0.125
        assert np.all(np.log2(st["dt"]) == np.round(np.log2(st["dt"]))) and np.all(np.fmod(st["t"], st["dt"]) == 0.0)
        e1 = d.energy()
        d.run_until(0.25, time_device=True)            # continues after the energy evaluation re-predicted the store
        e2 = d.energy()
        hist = d.history()
        stats = d.stats()
        print(f"order {order}: {stats['block_steps']} block steps, n_i min/median/max {hist.min()}/{np.median(hist)}/{hist.max()}, "
              f"dE/E {(e1 - e0) / e0:.2e} {(e2 - e0) / e0:.2e}, wall/step {stats['wall_ms'] / stats['block_steps'] * 1e3:.1f} us, "
              f"device/step {stats['device_ms'] / max(1, stats['timed_steps']) * 1e3:.1f} us")
        assert abs((e1 - e0) / e0) < lim and abs((e2 - e0) / e0) < lim
        assert hist.min() < w.N // 8 and hist.max() == w.N
        d.close()


@pytest.mark.gpu
def test_device_integrator_in_fp32_runs_and_conserves_energy():
    """fp32 pair arithmetic under the integrator (its force calls go through the fp64 re-evaluation of ill-conditioned
    sums, DESIGN.md R-F32): reaches t_end with block-aligned power-of-two steps and conserves energy at the fp32 level."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(1, N=1024)
    d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=4, precision=s2.S2_FP32)
    e0 = d.energy()
    d.run_until(0.125)
    st = d.state()
    assert (st["t"] == 0.125).all() and np.all(np.fmod(st["t"], st["dt"]) == 0.0)
    e1 = d.energy()
    hist = d.history()
    print(f"fp32 integrator: {d.stats()['block_steps']} block steps, n_i min/max {hist.min()}/{hist.max()}, dE/E {(e1 - e0) / e0:.2e}")
    assert abs((e1 - e0) / e0) < 2e-5 and hist.min() < w.N // 8 and hist.max() == w.N
    d.close()


@pytest.mark.gpu
@pytest.mark.parametrize("order", [4, 6])
def test_small_step_kernel_reproduces_the_step_by_step_run(order):
    """s2_bts_run hands runs of small block steps (<= 512 active particles) to ONE launch of bts_small_steps_kernel, which
    sweeps, combines, corrects, selects and predicts step after step behind grid barriers and returns at the first step
    that does not qualify.  The run must be the same run as with one synchronised force call per step (s2_set_tuning
    key 9 = 6): same block times and active counts step by step, same final t and dt arrays, positions equal to rounding
    (the kernel adds the j-ranges of the CTAs in another order than the force call adds its j-slices)."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(3, N=2048)
    runs = {}
    for mode in ("small", "small cap 48", "stepwise"):
        d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=order, averaged=order == 6)
        if mode == "stepwise":
            s2.s2_set_tuning(d.ctx, 9, 6)
        elif mode == "small cap 48":
            s2.s2_set_tuning(d.ctx, 10, 48)               # shorter runs: more hand-overs between the two kinds of step
        d.run_until(0.0625)
        d.run_until(0.125)                               # a second call continues the same run
        runs[mode] = (d.state(), d.history(), d.stats())
        d.close()
    sb, hb, tb = runs["stepwise"]
    assert tb["small"]["steps"] == 0
    for mode in ("small", "small cap 48"):
        sa, ha, ta = runs[mode]
        cap = 48 if mode.endswith("48") else 512
        assert np.array_equal(ha, hb), "active counts differ step by step"
        assert ta["block_steps"] == tb["block_steps"] and ta["particle_steps"] == tb["particle_steps"] == int(ha.sum())
        assert ta["time"] == tb["time"] == 0.125 and (sa["t"] == 0.125).all()
        assert np.array_equal(sa["dt"], sb["dt"])
        assert np.abs(sa["pos"] - sb["pos"]).max() < 1e-11 and np.abs(sa["vel"] - sb["vel"]).max() < 1e-10
        # every step that qualifies went through the kernel except the first of each s2_bts_run call at most, the rest not
        small = int((ha <= cap).sum())
        assert small - 2 <= ta["small"]["steps"] <= small and ha.max() == w.N
        print(f"order {order} {mode}: {ta['block_steps']} block steps, {ta['small']['steps']} in {ta['small']['launches']} launches; "
              f"wall per step {ta['wall_ms'] / ta['block_steps'] * 1e3:.1f} us, stepwise {tb['wall_ms'] / tb['block_steps'] * 1e3:.1f} us")


@pytest.mark.gpu
@pytest.mark.parametrize("n,cap,chunk", [(100, 0, 0), (100, 1, 3), (3000, 7, 0), (3000, 1024, 5), (1000, 33, 1)])
def test_small_step_kernel_edges(n, cap, chunk):
    """Corners of the small-step kernel's index arithmetic: fewer particles than SMs x 32 (most CTAs own none), a cap of one
    particle, caps that are no multiple of 32, more than 512 active particles in the kernel (two sweep rounds), and runs cut
    into launches of 1, 3 or 5 steps by max_block_steps.  Each must be the step-by-step run."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(3, N=n)
    t_end = 0.0625

    def run(stepwise):
        d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=4)
        if stepwise:
            s2.s2_set_tuning(d.ctx, 9, 6)
        elif cap:
            s2.s2_set_tuning(d.ctx, 10, cap)
        if chunk and not stepwise:
            while d.stats()["t_next"] <= t_end:
                assert 1 <= s2.s2_bts_run(d.bts, t_end, chunk) <= chunk
        else:
            d.run_until(t_end)
        out = (d.state(), d.history(), d.stats())
        d.close()
        return out

    (sa, ha, ta), (sb, hb, tb) = run(False), run(True)
    assert np.array_equal(ha, hb) and np.array_equal(sa["dt"], sb["dt"]) and np.array_equal(sa["t"], sb["t"])
    assert np.abs(sa["pos"] - sb["pos"]).max() < 1e-11 and np.abs(sa["vel"] - sb["vel"]).max() < 1e-10
    assert ta["time"] == tb["time"] == t_end
    lim = cap if cap else 512
    small = int((ha <= lim).sum())
    assert small > 0 and ta["small"]["steps"] >= small - (len(ha) // max(chunk, 1) + 2 if chunk else 2)
    assert ta["small"]["steps"] <= small


@pytest.mark.gpu
def test_integrator_steps_the_ordinary_way_when_an_sm_would_own_more_than_512_particles():
    """More than 512 particles per SM do not fit the small-step kernel's shared memory: s2_bts_run falls back to one force
    call per step (no error, no CPU path) and still follows the block-step scheme."""
    import torch
    from paper_1510_04068_b200.hermite import DeviceHermite
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    w = make_config(3, N=512 * sms + 1000)
    d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=4)
    for _ in range(12):
        d.step()
    st, h = d.stats(), d.history()
    d.close()
    assert st["small"]["steps"] == 0 and st["block_steps"] == 12 and h.min() >= 1


@pytest.mark.gpu
def test_small_step_profile_and_hop_latency_report_plausible_cycles():
    """The two diagnostics behind profiles/r02_blockstep.md: the per-part cycle sums of the small-step kernel count exactly
    the steps that kernel ran, every part of a step costs something, and the sums stay put once switched off; the hop
    microbenchmark returns a round trip of a few thousand SM cycles that does not shrink when more SMs answer."""
    import torch
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(3, N=4096)
    d = DeviceHermite(w.mass, w.pos, w.vel, w.eps2, order=4)
    d.run_until(0.03125)
    before = d.stats()["small"]["steps"]
    s2.s2_bts_small_profile(d.bts, 1)
    d.run_until(0.0625)
    p = s2.s2_bts_small_profile(d.bts, 0)
    ran = d.stats()["small"]["steps"] - before
    assert p["steps"] == ran > 100
    parts = [k for k in p if k != "steps"]
    assert len(parts) == 9 and all(p[k] > 0 for k in parts)
    per_step = sum(p[k] for k in parts) / ran
    assert 2e3 < per_step < 2e5, per_step                       # microseconds, not nanoseconds and not milliseconds
    d.run_until(0.09375)
    assert s2.s2_bts_small_profile(d.bts, 0) == p                # off: nothing added
    sms = torch.cuda.get_device_properties(0).multi_processor_count
    with pytest.raises(s2.S2Error):
        s2.s2_bts_small_profile(d.bts, sms + 1)
    two, many = s2.s2_hop_latency(d.ctx, 2, 500), s2.s2_hop_latency(d.ctx, sms, 500)
    assert 300 < two < 20000 and many > 0.8 * two, (two, many)
    with pytest.raises(s2.S2Error):
        s2.s2_hop_latency(d.ctx, sms + 1, 10)
    d.close()


@pytest.mark.gpu
def test_sixth_order_run_reaches_the_papers_energy_error_level():
    """PAPER.md sec 3.7 L164 quotes energy errors of about 1e-12 for its 6th-order double-precision runs (and 1e-10 in
    double-single) without stating softening, time-step cap or start-up.  With eta6 = 0.1 averaged with eta4 = 0.01 (L152,
    L156), dt_max = 1/64 and the default start-up factor the device integrator conserves the energy of an N = 4096 Plummer
    sphere over one time unit to a few 1e-12 -- in fp64 and, because this library's double-single pair arithmetic keeps
    ~48 bits (reading P11), in double-single as well.  A start-up factor ten times larger loses four orders of
    magnitude in the very first step: the test pins the default."""
    import paper_1510_04068_b200 as s2
    from paper_1510_04068_b200.hermite import DeviceHermite
    w = make_config(3, N=4096)
    eps2 = (4.0 / w.N) ** 2
    errs = {}
    for name, prec, kw in (("fp64", s2.S2_FP64, {}), ("ds", s2.S2_DS, {}), ("fp64, eta_start 0.01", s2.S2_FP64, {"eta_start": 0.01})):
        d = DeviceHermite(w.mass, w.pos, w.vel, eps2, order=6, precision=prec, averaged=True, dt_max=2.0 ** -6, **kw)
        e0 = d.energy()
        d.run_until(1.0)
        errs[name] = abs((d.energy() - e0) / e0)
        assert (d.state()["t"] == 1.0).all()
        d.close()
    print({k: f"{v:.2e}" for k, v in errs.items()})
    assert errs["fp64"] < 2e-11 and errs["ds"] < 2e-11
    assert errs["fp64, eta_start 0.01"] > 10 * errs["fp64"]
