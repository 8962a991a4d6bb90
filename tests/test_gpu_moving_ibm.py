"""Moving Lagrangian points on the GPU: `ibm_set_velocities` with non-zero, per-step-changing v_p (PAPER.md:160,
Eq. 11: the force is proportional to v_p - U_p; :171-175 the passes repeat it until |v_p - U_f| is small).
The (v_p - U_p) term of the spreading kernel and the slip norm of the multi-pass stop rule are compared with the
oracle element by element, single pass and several passes, on one domain and cut into x-slabs."""
import numpy as np
import pytest

from conftest import rel_linf
from paper_2603_11102_b200 import slab, workloads as wl

pytestmark = pytest.mark.gpu

TOL1, TOL10 = 1e-11, 1e-9


def rigid_velocities(pos, step):
    """rigid-body motion of the point cloud that changes every step: a translation that turns with the step number
    plus a rotation about the z axis through the cloud's centre (speeds of the order of U_inf / 2)"""
    c = pos.mean(axis=0)
    vt = 0.04 * np.array([np.cos(0.9 * step), np.sin(0.9 * step), 0.3])
    om = 0.08 * (1.0 + 0.5 * np.sin(1.3 * step))
    r = pos - c
    return np.ascontiguousarray(vt[None, :] + om * np.stack([-r[:, 1], r[:, 0], np.zeros(len(r))], axis=1))


@pytest.mark.parametrize("passes", [1, 5])
@pytest.mark.parametrize("name", ["C3", "C5"])
def test_moving_points_match_the_oracle(name, passes):
    """small cylinder (C3) and turbine (C5: rotor + nacelle + tower) boxes, v_p re-set before every step:
    1e-11 after one step, 1e-9 after ten"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=True)
    pos, vol = w.ibm
    o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg)
    for s in (o, g):
        s.ibm_set_points(pos, vol)
        s.ibm_set_iterations(passes, 0.0)
        s.set_state(w.W0)
    for k in range(10):
        v = rigid_velocities(pos, k)
        for s in (o, g):
            s.ibm_set_velocities(v)
            if w.alm is not None:
                s.alm_set_points(*w.alm(k))
            s.step(w.dt)
        if k == 0:
            W1 = g.get_state()
            e1 = rel_linf(W1, o.get_state())
            assert e1 <= TOL1, (name, passes, e1)
    e10 = rel_linf(g.get_state(), o.get_state())
    assert e10 <= TOL10, (name, passes, e10)
    g.close()
    o.close()
    # the velocities did enter: the first step differs from the one of the body at rest
    g0 = gks.Gks(w.cfg)
    g0.ibm_set_points(pos, vol)
    g0.ibm_set_iterations(passes, 0.0)
    g0.set_state(w.W0)
    if w.alm is not None:
        g0.alm_set_points(*w.alm(0))
    g0.step(w.dt)
    assert rel_linf(g0.get_state(), W1) > 1e-4
    g0.close()


def test_stop_rule_measures_the_slip_against_the_moving_points():
    """tolerance semantics with v_p != 0 (S25: the passes stop once max_p |v_p - U_p| < tol): a tolerance between
    the oracle's slips after 2 and after 3 passes ends the passes of both sides at the same pass"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C3", small=True)
    pos, vol = w.ibm
    v = rigid_velocities(pos, 2)
    slips = []
    for k in (2, 3):
        o = ob.Oracle(w.cfg)
        o.ibm_set_points(pos, vol)
        o.ibm_set_iterations(k)
        o.ibm_set_velocities(v)
        o.set_state(w.W0)
        o.step(w.dt)
        slips.append(np.linalg.norm(v - o.ibm_interpolate(), axis=1).max())
        o.close()
    assert slips[1] < slips[0]
    tol = 0.5 * (slips[0] + slips[1])
    res = {}
    for passes, t in ((8, tol), (3, 0.0), (8, 0.0)):
        o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg)
        for s in (o, g):
            s.ibm_set_points(pos, vol)
            s.ibm_set_iterations(passes, t)
            s.ibm_set_velocities(v)
            s.set_state(w.W0)
            s.step(w.dt)
        res[(passes, t)] = g.get_state()
        assert rel_linf(res[(passes, t)], o.get_state()) <= TOL1, (passes, t)
        g.close()
        o.close()
    # slip after 2 passes > tol > slip after 3: the third pass still spreads, the fourth does not
    assert rel_linf(res[(8, tol)], res[(3, 0.0)]) <= 1e-14
    assert rel_linf(res[(8, tol)], res[(8, 0.0)]) > 1e-9


def test_device_pointer_null_reset_and_a_body_moving_with_the_stream():
    import torch
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C3", small=True)
    pos, vol = w.ibm
    v = rigid_velocities(pos, 1)
    out = []
    for kind in ("host", "device", "reset"):
        g = gks.Gks(w.cfg)
        g.ibm_set_points(pos, vol)
        g.set_state(w.W0)
        if kind == "device":
            with torch.cuda.stream(g.stream):
                vd = torch.from_numpy(v).to("cuda:0")
            g.stream.synchronize()
            g.ibm_set_velocities(vd)
        else:
            g.ibm_set_velocities(v)
        if kind == "reset":
            g.ibm_set_velocities(None)                          # NULL: the body is at rest again
        g.step(w.dt)
        out.append(g.get_state())
        g.close()
    assert rel_linf(out[0], out[1]) <= 1e-14                     # the spreading adds with fp64 atomics: order only
    at_rest = gks.run_workload(w, steps=1)
    assert rel_linf(out[2], at_rest) <= 1e-14                   # fp64 atomics: order only
    assert rel_linf(out[0], at_rest) > 1e-4
    # a body that moves with a uniform stream exerts no force (v_p - U_p = 0): the stream stays uniform
    g = gks.Gks(w.cfg)
    g.ibm_set_points(pos, vol)
    g.ibm_set_iterations(3, 0.0)
    g.set_state(w.W0)                                           # uniform (1, U_inf, 0, 0)
    g.ibm_set_velocities(np.tile(np.array([wl.U_INF, 0.0, 0.0]), (len(pos), 1)))
    for _ in range(2):
        g.step(w.dt)
    W = g.get_state()
    g.close()
    assert np.abs(W - w.W0).max() <= 1e-15


@pytest.mark.parametrize("passes", [1, 3])
def test_moving_points_across_slab_cuts(passes):
    """the small cylinder cut through by an x-slab boundary, moving points: every sub-domain is handed the velocities
    of the points it knows (`SlabDecomposition.ibm_velocities`); equal to the single-domain run and to the oracle"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C3", small=True)
    pos, vol = w.ibm
    for world in range(2, 9):                                 # the first decomposition that cuts through the body
        d = slab.SlabDecomposition(w.cfg, world)
        cuts = w.cfg.origin[0] + d.x_lo[1:-1] * w.cfg.spacing[0]
        if np.abs(pos[:, :1] - cuts[None, :]).min() < 0.5 * w.cfg.spacing[0]:
            break
    assert sum(len(d.ibm_select(r, pos)[0]) for r in range(world)) > len(pos)
    steps = 3
    solvers = [gks.Gks(d.local_cfg(r)) for r in range(world)]
    for r, s in enumerate(solvers):
        s.ibm_set_points(*d.ibm_points(r, pos, vol))
        s.ibm_set_iterations(passes, 0.0)
        s.set_state(d.scatter(w.W0, r))
    st = slab.SlabStepper(slab.LocalTransport(d), solvers, slab.BufferPool("cuda:0"))
    for k in range(steps):
        v = rigid_velocities(pos, k)
        for r, s in enumerate(solvers):
            s.ibm_set_velocities(d.ibm_velocities(r, pos, v))
        st.step(w.dt, ibm=True, ibm_passes=passes)
    Ws = d.gather([s.get_state() for s in solvers])
    for s in solvers:
        s.close()
    o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg)
    for s in (o, g):
        s.ibm_set_points(pos, vol)
        s.ibm_set_iterations(passes, 0.0)
        s.set_state(w.W0)
        for k in range(steps):
            s.ibm_set_velocities(rigid_velocities(pos, k))
            s.step(w.dt)
    assert rel_linf(Ws, g.get_state()) <= 1e-13
    assert rel_linf(Ws, o.get_state()) <= 3e-11
    g.close()
    o.close()
