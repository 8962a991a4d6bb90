"""Parity of the CUDA path (through the C ABI) with the CPU oracle, element by element on the same
seeded inputs.  Bar (BASELINE.json north_star): relative L-inf (norm S24) <= 1e-11 after one step,
<= 1e-9 after ten steps, fp64."""
import numpy as np
import pytest

from conftest import rel_linf
from paper_2603_11102_b200 import workloads as wl
from paper_2603_11102_b200.workloads import GridConfig

pytestmark = pytest.mark.gpu

TOL1, TOL10 = 1e-11, 1e-9
P, NS, SL, IN, OUT, EX = range(6)


def run_oracle(w, steps):
    from oracle import binding as ob
    o = ob.Oracle(w.cfg)
    if w.bulk_flux is not None:
        o.set_bulk_flux(*w.bulk_flux)
    if w.ibm is not None:
        o.ibm_set_points(*w.ibm)
    o.set_state(w.W0)
    for s in range(steps):
        if w.alm is not None:
            o.alm_set_points(*w.alm(s))
        o.step(w.dt)
    W = o.get_state()
    o.close()
    return W


def run_gpu(w, steps, sweep=None):
    from paper_2603_11102_b200 import gks
    return gks.run_workload(w, steps, sweep=sweep)


@pytest.mark.parametrize("sweep", [0, 1])
def test_C1_taylor_green_one_and_ten_steps(sweep):
    w = wl.by_name("C1")
    e1 = rel_linf(run_gpu(w, 1, sweep), run_oracle(w, 1))
    assert e1 <= TOL1, e1
    e10 = rel_linf(run_gpu(w, 10, sweep), run_oracle(w, 10))
    assert e10 <= TOL10, e10


@pytest.mark.parametrize("sweep", [0, 1])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_face_fluxes_match_the_oracle(d, sweep):
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.taylor_green(20)
    o = ob.Oracle(w.cfg)
    o.set_state(w.W0)
    Fo, dFo = o.eval_flux(d)
    g = gks.Gks(w.cfg, debug=True)
    g.debug_set_sweep(sweep)
    g.set_state(w.W0)
    Fg, dFg = g.debug_eval_flux(d)
    g.close()
    assert np.abs(Fg - Fo).max() <= 1e-13 * np.abs(Fo).max()
    assert np.abs(dFg - dFo).max() <= 1e-12 * np.abs(dFo).max()


@pytest.mark.parametrize("name", ["C2", "C3", "C4", "C5"])
def test_small_variants_of_the_configs(name):
    """reduced grids with the structure of configs 2-5 (walls + stretching + bulk flux; IBM cylinder with
    inflow/convective outflow; rotating ALM rotor; ALM + IBM nacelle/tower)"""
    w = wl.by_name(name, small=True)
    e1 = rel_linf(run_gpu(w, 1), run_oracle(w, 1))
    assert e1 <= TOL1, e1
    e10 = rel_linf(run_gpu(w, 10), run_oracle(w, 10))
    assert e10 <= TOL10, e10


@pytest.mark.parametrize("n", [(6, 6, 6), (37, 11, 9), (7, 70, 6), (9, 6, 45)])
@pytest.mark.parametrize("bc", [(P,) * 6, (IN, OUT, NS, SL, EX, EX), (EX, IN, P, P, OUT, NS), (SL, SL, OUT, IN, P, P)])
def test_ragged_sizes_and_every_boundary_kind(n, bc):
    """minimum size, sizes that are no multiple of any tile, stretched axes, all six boundary kinds"""
    rng = np.random.default_rng(hash((n, bc)) % 2 ** 32)
    zf = np.cumsum(np.r_[0.0, rng.uniform(0.8, 1.2, n[2])]) * 0.1
    cfg = GridConfig(n=n, faces=(None, None, zf), spacing=(0.1, 0.12, 0.1), nu=2e-3, bc=bc,
                     inflow=(1.0, 0.1, 0.1, 0.1))
    W0 = np.empty((4, n[2], n[1], n[0]))
    W0[0] = 1.0 + 0.02 * rng.standard_normal(W0[0].shape)
    W0[1:] = 0.1 + 0.03 * rng.standard_normal(W0[1:].shape)
    w = wl.Workload("ragged", cfg, W0, wl.cfl_dt(cfg, W0), 3)
    e1 = rel_linf(run_gpu(w, 1), run_oracle(w, 1))
    assert e1 <= TOL1, e1
    e3 = rel_linf(run_gpu(w, 3), run_oracle(w, 3))
    assert e3 <= 10 * TOL1, e3


def test_body_force_and_device_pointers():
    import torch
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C2", small=True)
    o = ob.Oracle(w.cfg)
    o.set_body_force(0.01, -0.02, 0.03)
    o.set_state(w.W0)
    o.step(w.dt)
    g = gks.Gks(w.cfg)
    g.set_body_force(0.01, -0.02, 0.03)
    with torch.cuda.stream(g.stream):
        Wd = torch.from_numpy(w.W0).to("cuda:0")
        out = torch.empty_like(Wd)
    g.stream.synchronize()
    g.set_state(Wd)                       # device pointers in and out
    g.step(w.dt)
    g.get_state(out)
    g.synchronize()
    assert rel_linf(out.cpu().numpy(), o.get_state()) <= TOL1
    g.check_finite()
    assert g.launch_count > 0
    g.close()


def test_error_paths_on_the_device():
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C1")
    g = gks.Gks(w.cfg)
    with pytest.raises(gks.GksError) as e:
        g.step(w.dt)                      # before set_state
    assert e.value.status == 4
    g.set_state(w.W0)
    with pytest.raises(gks.GksError):
        g.step(-1.0)
    with pytest.raises(gks.GksError):
        g.alm_set_points(np.zeros((1, 3)), np.zeros((1, 3)), 0.0)
    with pytest.raises(gks.GksError):
        g.alm_set_points(np.zeros((1, 3)), np.zeros((1, 3)), 2.0)      # 6 eps wider than the periodic box
    g.alm_set_points(np.zeros((0, 3)), np.zeros((0, 3)), 1.0)          # n = 0 clears
    bad = w.W0.copy()
    bad[1, 3, 4, 5] = np.nan
    g.set_state(bad)
    with pytest.raises(gks.GksError) as e:
        g.check_finite()
    assert e.value.status == 5
    g.close()
    cfg = GridConfig(n=(8, 8, 8), spacing=(0.1,) * 3, bc=(EX,) * 6)
    g = gks.Gks(cfg)
    with pytest.raises(gks.GksError):
        g.ibm_set_points(np.array([[-0.5, 0.1, 0.1]]), np.array([1.0]))  # outside the domain
    g.close()


def test_alm_cloud_wider_than_a_periodic_axis():
    """actuator points spread over more than a period of y and z (a rotor in a narrow periodic box): the gather box
    covers the whole axis once and takes the nearest image of every point; points outside [0, L) wrap"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    n, h = (16, 10, 12), 0.1
    cfg = GridConfig(n=n, spacing=(h, h, h), nu=1e-3, bc=(EX, EX, P, P, P, P))
    rng = np.random.default_rng(11)
    W0 = np.zeros((4, n[2], n[1], n[0]))
    W0[0] = 1.0 + 0.01 * rng.standard_normal(W0[0].shape)
    W0[1] = 0.1 * W0[0]
    pos = np.column_stack([rng.uniform(0.5, 1.1, 40), rng.uniform(-0.3, 1.4, 40), rng.uniform(-0.2, 1.5, 40)])
    force = 0.05 * rng.standard_normal((40, 3))
    eps = 0.15                                       # 6 eps = 0.9 < 1.0 = the y period
    o = ob.Oracle(cfg)
    o.alm_set_points(pos, force, eps)
    o.set_state(W0)
    o.step(0.02)
    g = gks.Gks(cfg)
    g.alm_set_points(pos, force, eps)
    g.set_state(W0)
    g.step(0.02)
    Wg, Wo = g.get_state(), o.get_state()
    g.close()
    o.close()
    assert rel_linf(Wg, Wo) <= TOL1
    free = ob.Oracle(cfg)
    free.set_state(W0)
    free.step(0.02)
    assert np.abs(Wo - free.get_state()).max() > 1e-5          # the forcing is there
    free.close()


@pytest.mark.parametrize("passes,tol", [(3, 0.0), (8, 0.0), (20, None)])
def test_ibm_multi_direct_forcing_passes(passes, tol):
    """IBM passes (Eq. 11-12, S25) on the small cylinder and turbine cases: a fixed number of passes, and the
    device-side stop rule with a tolerance that the oracle reaches after a few passes (tol = None: chosen from
    the oracle's own slip history so that the stop falls strictly inside the allowed passes)"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    for name in ("C3", "C5"):
        w = wl.by_name(name, small=True)
        t = tol
        if t is None:
            # slip seen by pass k of the first step = max |U_p| after k passes (v_p = 0)
            slips = []
            for k in (2, 3, 4):
                o = ob.Oracle(w.cfg)
                o.ibm_set_points(*w.ibm)
                o.ibm_set_iterations(k)
                o.set_state(w.W0)
                if w.alm is not None:
                    o.alm_set_points(np.zeros((0, 3)), np.zeros((0, 3)), 1.0)
                o.step(w.dt)
                slips.append(np.linalg.norm(o.ibm_interpolate(), axis=1).max())
                o.close()
            t = 0.5 * (slips[0] + slips[1])        # between the slip after 2 and after 3 passes
        o = ob.Oracle(w.cfg)
        g = gks.Gks(w.cfg)
        for s in (o, g):
            s.ibm_set_points(*w.ibm)
            s.ibm_set_iterations(passes, t)
            s.set_state(w.W0)
        for step in range(3):
            if w.alm is not None:
                o.alm_set_points(*w.alm(step))
                g.alm_set_points(*w.alm(step))
            o.step(w.dt)
            g.step(w.dt)
        e = rel_linf(g.get_state(), o.get_state())
        assert e <= 3 * TOL1, (name, e)
        # the passes did something: the result differs from the single-pass one
        g1 = gks.Gks(w.cfg)
        g1.ibm_set_points(*w.ibm)
        g1.set_state(w.W0)
        for step in range(3):
            if w.alm is not None:
                g1.alm_set_points(*w.alm(step))
            g1.step(w.dt)
        assert rel_linf(g1.get_state(), o.get_state()) > 1e-8
        g1.close()
        g.close()
        o.close()
    gg = gks.Gks(wl.by_name("C3", small=True).cfg)
    with pytest.raises(gks.GksError):
        gg.ibm_set_iterations(0)
    with pytest.raises(gks.GksError):
        gg.ibm_set_iterations(65)
    gg.close()


def test_cfl_dt_matches_the_oracle():
    """PAPER.md:91 on the device: the same number as the oracle's loop (both take max of sqrt(m.m)/rho; fma
    contraction may move the last bit), host and device output pointers, stretched grid, after a step"""
    import torch
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    for name in ("C1", "C2", "C5"):
        w = wl.by_name(name, small=(name != "C1"))
        o = ob.Oracle(w.cfg)
        g = gks.Gks(w.cfg)
        o.set_state(w.W0)
        g.set_state(w.W0)
        assert g.cfl_dt(0.4) == pytest.approx(o.cfl_dt(0.4), rel=1e-14)
        o.step(w.dt)
        g.step(w.dt)
        out = torch.zeros(1, dtype=torch.float64, device="cuda:0")
        g.cfl_dt(0.7, out)
        g.synchronize()
        assert float(out.cpu()[0]) == pytest.approx(o.cfl_dt(0.7), rel=1e-12)
        with pytest.raises(gks.GksError):
            g.cfl_dt(-1.0)
        g.close()
        o.close()


@pytest.mark.parametrize("switches", [{}, {"freestream_correction": True, "tip_correction": True},
                                      {"refine": True, "nsections": 3, "freestream_correction": True, "tip_correction": True}])
def test_online_rotor_matches_the_oracle(switches):
    """actuator-line front half on the device (S26-S28): point positions and forces of the test hook, then 1 and
    10 steps of the small rotor (C4) and turbine (C5: rotor + IBM nacelle and tower) boxes with the rotor on line;
    third variant: stations refined at root and tip with their own widths, three airfoil sections blended in r"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    for name in ("C4", "C5"):
        w = wl.by_name(name, small=True)
        pos0, _, eps = w.alm(0)
        hub = pos0.reshape(3, -1, 3).mean(axis=(0, 1))          # the prescribed blades are 120 degrees apart
        Rr = np.linalg.norm(pos0 - hub, axis=1).max() * 64.5 / 64.0
        r = wl.synthetic_rotor(hub=hub, R=float(Rr), eps=eps, npts=48, **switches)
        for steps, tol in ((1, TOL1), (10, TOL10)):
            o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg)
            for s in (o, g):
                if w.ibm is not None:
                    s.ibm_set_points(*w.ibm)
                s.set_state(w.W0)
                s.alm_set_rotor(r)
            if steps == 1:
                po, fo = o.alm_rotor_eval()
                pg, fg = g.alm_rotor_eval()
                assert np.abs(pg - po).max() <= 1e-14 * np.abs(po).max()
                assert np.abs(fg - fo).max() <= 1e-12 * np.abs(fo).max() and np.abs(fo).max() > 0
            for _ in range(steps):
                o.step(w.dt)
                g.step(w.dt)
            e = rel_linf(g.get_state(), o.get_state())
            assert e <= tol, (name, steps, e)
            if steps == 10:       # the clocks agree: the blades have turned by omega * 10 dt on both sides
                po, fo = o.alm_rotor_eval()
                pg, fg = g.alm_rotor_eval()
                assert np.abs(pg - po).max() <= 1e-13 * np.abs(po).max()
                assert np.abs(fg - fo).max() <= 1e-9 * np.abs(fo).max()
            g.close()
            o.close()
    g = gks.Gks(wl.by_name("C4", small=True).cfg)
    bad = wl.synthetic_rotor(hub=(1, 1, 1), R=0.5, eps=0.1)
    bad.alpha = bad.alpha[::-1].copy()
    with pytest.raises(gks.GksError):
        g.alm_set_rotor(bad)
    bad = wl.synthetic_rotor(hub=(1, 1, 1), R=0.5, eps=0.1, refine=True, nsections=3)
    bad.width = None                                             # radius without width
    with pytest.raises(gks.GksError):
        g.alm_set_rotor(bad)
    bad = wl.synthetic_rotor(hub=(1, 1, 1), R=0.5, eps=0.1, nsections=3)
    bad.section_r = bad.section_r[::-1].copy()
    with pytest.raises(gks.GksError):
        g.alm_set_rotor(bad)
    g.alm_set_rotor(None)
    g.close()


@pytest.mark.parametrize("sweep", [0, 1])
def test_linear_tangential_variant_matches_the_oracle(sweep):
    """scheme variant of SURVEY 8f f4 (linear weights in the two tangential passes): both sweep implementations
    against the oracle's variant on C1 (1 and 10 steps), the small channel and a ragged mixed-boundary box"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    rng = np.random.default_rng(12)
    n = (19, 9, 23)
    cfg = GridConfig(n=n, spacing=(0.1, 0.12, 0.1), nu=2e-3, bc=(IN, OUT, P, P, NS, SL), inflow=(1.0, 0.1, 0.0, 0.0))
    W0 = np.empty((4, n[2], n[1], n[0]))
    W0[0] = 1.0 + 0.02 * rng.standard_normal(W0[0].shape)
    W0[1:] = 0.1 + 0.03 * rng.standard_normal(W0[1:].shape)
    cases = [(wl.by_name("C1"), 1, TOL1), (wl.by_name("C1"), 10, TOL10), (wl.by_name("C2", small=True), 3, 10 * TOL1),
             (wl.Workload("ragged", cfg, W0, wl.cfl_dt(cfg, W0), 3), 3, 10 * TOL1)]
    for w, steps, tol in cases:
        o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg, debug=True)
        g.debug_set_sweep(sweep)
        for s in (o, g):
            s.set_reconstruction(1)
            if w.bulk_flux is not None:
                s.set_bulk_flux(*w.bulk_flux)
            s.set_state(w.W0)
        for _ in range(steps):
            o.step(w.dt)
            g.step(w.dt)
        Wg = g.get_state()
        e = rel_linf(Wg, o.get_state())
        assert e <= tol, (w.name, steps, e)
        o.close()
        if steps == 1:      # and it is not the WENO scheme
            g.set_reconstruction(0)
            g.set_state(w.W0)
            g.step(w.dt)
            assert rel_linf(g.get_state(), Wg) > 1e-9
            with pytest.raises(gks.GksError):
                g.set_reconstruction(3)
        g.close()


def test_split_step_equals_gks_step_and_enforces_the_call_order():
    """gks_step = gks_step_begin + gks_step_finish + gks_step_force (the form the x-slab driver uses), bit for bit on
    the small turbine box (IBM atomics aside: compared to 1e-14), and the calls refuse a wrong order"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C5", small=True)
    res = []
    for split in (False, True):
        g = gks.Gks(w.cfg)
        g.ibm_set_points(*w.ibm)
        g.set_state(w.W0)
        for k in range(3):
            g.alm_set_points(*w.alm(k))
            if split:
                g.step_begin(w.dt)
                g.step_finish(w.dt)
                g.step_force(w.dt)
            else:
                g.step(w.dt)
        res.append(g.get_state())
        if split:
            with pytest.raises(gks.GksError):
                g.step_force(w.dt)
            g.step_begin(w.dt)
            with pytest.raises(gks.GksError):
                g.step_begin(w.dt)
            with pytest.raises(gks.GksError):
                g.step(w.dt)
            with pytest.raises(gks.GksError):
                g.step_force(w.dt)
            g.step_finish(w.dt)
            g.step_force(w.dt)
        g.close()
    assert rel_linf(res[1], res[0]) <= 1e-14


def test_calls_inside_a_split_step_cannot_corrupt_it():
    """between gks_step_begin and gks_step_force the predictor P and the flux buffers are live: gks_set_state and
    gks_debug_eval_flux are refused (GKS_ERR_STATE), a diagnostic gks_get_state to HOST memory is allowed, reads W^n /
    the un-forced W^{n+1} and leaves the step untouched; the three parts of a step must be given the same dt"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C5", small=True)
    ref = gks.Gks(w.cfg)
    ref.ibm_set_points(*w.ibm)
    ref.set_state(w.W0)
    ref.alm_set_points(*w.alm(0))
    ref.step(w.dt)
    Wref = ref.get_state()
    ref.close()
    g = gks.Gks(w.cfg)
    g.ibm_set_points(*w.ibm)
    g.set_state(w.W0)
    g.alm_set_points(*w.alm(0))
    g.step_begin(w.dt)
    for call in (lambda: g.set_state(w.W0), lambda: g.debug_eval_flux(0)):
        with pytest.raises(gks.GksError) as e:
            call()
        assert e.value.status == 4
    assert np.array_equal(g.get_state(), w.W0)                # W^n, staged through a buffer that is free here
    with pytest.raises(gks.GksError) as e:
        g.step_finish(w.dt * (1 + 1e-12))                     # a driver that recomputed dt between the halves
    assert e.value.status == 1
    g.step_finish(w.dt)
    mid = g.get_state()                                       # the un-forced W^{n+1}
    assert np.isfinite(mid).all() and rel_linf(mid, Wref) > 1e-9
    with pytest.raises(gks.GksError):
        g.set_state(w.W0)
    with pytest.raises(gks.GksError) as e:
        g.step_force(0.5 * w.dt)
    assert e.value.status == 1
    g.step_force(w.dt)
    assert rel_linf(g.get_state(), Wref) <= 1e-14             # IBM atomics: order only
    g.set_state(w.W0)                                         # idle again: everything is allowed
    g.debug_eval_flux(1)
    g.close()


def test_two_contexts_on_their_own_streams_do_not_interfere():
    """include/gks.h: a context owns all of its state (workspace, stream, point sets); two contexts of different
    shape and forcing, stepped alternately on their own streams with no synchronisation in between, give what
    each gives alone - bit for bit on the periodic box, to round-off where the IBM spreading adds with atomics."""
    from paper_2603_11102_b200 import gks
    wa, wb = wl.by_name("C1"), wl.by_name("C5", small=True)
    steps = 3
    alone = [gks.run_workload(w, steps=steps) for w in (wa, wb)]
    ga, gb = gks.Gks(wa.cfg), gks.Gks(wb.cfg)
    assert ga.stream.cuda_stream != gb.stream.cuda_stream
    gb.ibm_set_points(*wb.ibm)
    ga.set_state(wa.W0)
    gb.set_state(wb.W0)
    for s in range(steps):
        gb.alm_set_points(*wb.alm(s))
        ga.step(wa.dt)
        gb.step(wb.dt)
    Wb, Wa = gb.get_state(), ga.get_state()
    ga.close()
    gb.close()
    assert np.array_equal(Wa, alone[0])
    assert rel_linf(Wb, alone[1]) <= 1e-13
