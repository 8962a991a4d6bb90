"""Parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (persistent fused sweeps,
one CTA per SM, whole-column waves + split remainder), north_star tolerance 1e-11 after one step.

The oracle cannot run 256^3 ... 512x256x256 in seconds, so it computes SAMPLED outputs one sub-box at a time:
one S2O4 step has a finite domain of dependence (3 cells per stage and axis: normal stencil -3..+2, the two
tangential passes +-2 each; two stages -> 6 cells; IBM interpolation + spreading add 3), so the oracle run
on a sub-box cut out of the same initial state, with any boundary condition on the cut faces, reproduces
the cells further than MARGIN = 10 cells from every cut face exactly.  Sub-box faces that coincide with a
non-periodic domain face keep the domain's boundary condition (margin 0 there); periodic axes wrap.
The small full configurations (C2, C3) are compared cell for cell over the whole grid."""
import numpy as np
import pytest

from conftest import rel_linf
from paper_2603_11102_b200 import workloads as wl
from paper_2603_11102_b200.workloads import GridConfig

pytestmark = pytest.mark.gpu

TOL1 = 1e-11
MARGIN = 10
EX = wl.BC_EXTRAPOLATE


def oracle_step_on_subbox(w, lo, size, steps=1, margin=MARGIN):
    """Oracle result on the sub-box [lo, lo+size) of workload w and the slices of its trusted core."""
    from oracle import binding as ob
    cfg = w.cfg
    assert all(f is None for f in cfg.faces), "sub-boxes are cut from uniform grids"
    n = (cfg.n[0], cfg.n[1], cfg.n[2])
    bc = list(cfg.bc)
    sub_bc, core = [], []
    for a in range(3):
        periodic = bc[2 * a] == wl.BC_PERIODIC
        if not periodic:
            assert 0 <= lo[a] and lo[a] + size[a] <= n[a]
        at_lo = (not periodic) and lo[a] == 0
        at_hi = (not periodic) and lo[a] + size[a] == n[a]
        sub_bc += [bc[2 * a] if at_lo else EX, bc[2 * a + 1] if at_hi else EX]
        core.append(slice(0 if at_lo else margin, size[a] if at_hi else size[a] - margin))
    idx = [np.arange(lo[a], lo[a] + size[a]) % n[a] for a in range(3)]
    W0 = w.W0[:, idx[2]][:, :, idx[1]][:, :, :, idx[0]].copy()
    origin = tuple(cfg.origin[a] + lo[a] * cfg.spacing[a] for a in range(3))
    sub = GridConfig(n=tuple(size), origin=origin, spacing=cfg.spacing, RT=cfg.RT, nu=cfg.nu, rho_ref=cfg.rho_ref,
                     bc=tuple(sub_bc), inflow=cfg.inflow, weno_eps=cfg.weno_eps)
    o = ob.Oracle(sub)
    seen = {"ibm": 0, "alm": 0}
    hi = [origin[a] + size[a] * cfg.spacing[a] for a in range(3)]
    if w.ibm is not None:
        pos, vol = w.ibm
        inside = np.all([(pos[:, a] > origin[a]) & (pos[:, a] < hi[a]) for a in range(3)], axis=0)
        # a point whose 3-point support is cut by a sub-box face is only seen by cells outside the core
        o.ibm_set_points(pos[inside], vol[inside])
        seen["ibm"] = int(inside.sum())
    o.set_state(W0)
    for s in range(steps):
        if w.alm is not None:
            pos, force, eps = w.alm(s)
            near = np.all([(pos[:, a] > origin[a] - 3.5 * eps) & (pos[:, a] < hi[a] + 3.5 * eps) for a in range(3)], axis=0)
            o.alm_set_points(pos[near], force[near], eps)
            seen["alm"] = int(near.sum())
        o.step(w.dt)
    W = o.get_state()
    o.close()
    return W, idx, (core[2], core[1], core[0]), seen


def check_samples(w, Wg, boxes, size=(28, 28, 28), need=(), steps=1, tol=TOL1, margin=MARGIN):
    """need: per box, the forcing kinds ('alm', 'ibm') that must act inside the sub-box (the sample is then a
    test of that forcing, not only of the fluid step)"""
    scale_rho = np.abs(Wg[0]).max()
    scale_m = np.sqrt((Wg[1:] ** 2).sum(0)).max()
    worst = 0.0
    for b, lo in enumerate(boxes):
        Wo, idx, core, seen = oracle_step_on_subbox(w, lo, size, steps, margin)
        for kind in (need[b] if b < len(need) else ()):
            assert seen[kind] > 0, (w.name, lo, kind)
        G = Wg[:, idx[2]][:, :, idx[1]][:, :, :, idx[0]]
        d = np.abs(G - Wo)[(slice(None),) + core]
        assert d.size > 0
        err = max(d[0].max() / scale_rho, d[1:].max() / scale_m)   # norm S24 with the full field's scales
        worst = max(worst, err)
        assert err <= tol, (w.name, lo, err)
    return worst


def box_around(w, x, size=28):
    """sub-box origin that puts the physical point x at the centre of the trusted core"""
    lo = []
    for a in range(3):
        i = int(np.floor((x[a] - w.cfg.origin[a]) / w.cfg.spacing[a])) - size // 2
        if w.cfg.bc[2 * a] != wl.BC_PERIODIC:
            i = min(max(i, 0), w.cfg.n[a] - size)
        lo.append(i)
    return tuple(lo)


def test_M0_metric_box_256_sampled():
    """the box bench.py times: 256^3 periodic Taylor-Green; sub-boxes in the interior, across the periodic
    seam of every axis, in the remainder columns of the persistent schedule and at tile corners"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("M0")
    Wg = gks.run_workload(w, steps=1)
    boxes = [(100, 117, 3), (-14, -14, -14), (242, 5, 120), (57, 240, 243), (120, 120, 120), (7, 250, 64)]
    check_samples(w, Wg, boxes)
    # properties that hold at any size: conservation on the periodic box (P7) and finiteness
    mscale = float(np.abs(w.W0[1:]).sum(dtype=np.longdouble))
    for c in range(4):
        s0, s1 = w.W0[c].sum(dtype=np.longdouble), Wg[c].sum(dtype=np.longdouble)
        ref = abs(float(s0)) if c == 0 else 1e-3 * mscale
        assert abs(float(s1 - s0)) <= 1e-12 * ref, (c, float(s1 - s0), ref)
    assert np.isfinite(Wg).all()


def test_M0_metric_box_256_ten_steps_sampled():
    """north_star's second bar at the full size: 1e-9 after ten steps.  The domain of dependence grows by 6 cells
    per step, so the oracle runs a 136^3 sub-box (across the periodic seam) and its central 8^3 cells count"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("M0")
    Wg = gks.run_workload(w, steps=10)
    check_samples(w, Wg, [(-70, 60, 190)], size=(136, 136, 136), steps=10, tol=1e-9, margin=64)


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_full_channel_and_cylinder_cell_for_cell(name):
    """C2 128x96x64 (stretched walls, bulk-flux forcing) and C3 256x128x64 (IBM cylinder, inflow / convective
    outflow): the oracle runs the whole grid"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name)
    Wg = gks.run_workload(w, steps=1)
    o = ob.Oracle(w.cfg)
    if w.bulk_flux is not None:
        o.set_bulk_flux(*w.bulk_flux)
    if w.ibm is not None:
        o.ibm_set_points(*w.ibm)
    o.set_state(w.W0)
    o.step(w.dt)
    err = rel_linf(Wg, o.get_state())
    o.close()
    assert err <= TOL1, err


def test_C4_rotor_384x192x192_sampled():
    """ALM rotor: sub-boxes through the rotor disc (hub, blade tips), at the inflow face, on the slip wall,
    across the periodic y seam and at the convective outflow"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C4")
    Wg = gks.run_workload(w, steps=1)
    pos = w.alm(0)[0]                        # 3 blades x 64 points, root to tip
    boxes = [box_around(w, pos[0]), box_around(w, pos[63]), box_around(w, pos[64 + 63]), (0, 90, 90), (200, 96, 0),
             (150, -14, 80), (356, 80, 80), (356, 164, 164)]
    check_samples(w, Wg, boxes, need=[("alm",), ("alm",), ("alm",)])


def test_C5_turbine_512x256x256_sampled():
    """ALM rotor + IBM nacelle and tower: sub-boxes at the hub / nacelle, along the tower, at the tower foot
    on the ground (slip wall), in the wake, at inflow and outflow"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C5")
    Wg = gks.run_workload(w, steps=1)
    boxes = [(116, 114, 86), (124, 114, 40), (122, 114, 0), (116, 114, 120), (300, 100, 100), (0, 120, 90),
             (484, 120, 90), (250, -14, 228)]
    check_samples(w, Wg, boxes, need=[("alm", "ibm"), ("ibm",), ("ibm",), ("alm",)])


@pytest.mark.parametrize("name", ["C2", "C3"])
def test_full_channel_and_cylinder_ten_steps(name):
    """north_star's second bar (1e-9 after ten steps) at the stated sizes of configs 2 and 3, whole grid, cell for cell"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name)
    Wg = gks.run_workload(w, steps=10)
    o = ob.Oracle(w.cfg)
    if w.bulk_flux is not None:
        o.set_bulk_flux(*w.bulk_flux)
    if w.ibm is not None:
        o.ibm_set_points(*w.ibm)
    o.set_state(w.W0)
    for _ in range(10):
        o.step(w.dt)
    err = rel_linf(Wg, o.get_state())
    o.close()
    assert err <= 1e-9, err


def test_C4_rotor_ten_steps_sampled():
    """config 4 at 384x192x192, ten steps with the blades turning (`alm_set_points` re-issued every step on both
    sides): the oracle runs a 144^3 sub-box that holds the whole rotor disc; its trusted core (64 cells from every
    cut: 6 per step and a margin) is the 16^3 cells around the inner half of blade 0 in the rotor plane"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C4")
    Wg = gks.run_workload(w, steps=10)
    lo, size = (24, 34, 26), (144, 144, 144)
    for s in (0, 9):                                   # every actuator point acts inside the sub-box, at both ends of the run
        p = w.alm(s)[0] / w.cfg.spacing[0]
        assert all((p[:, a] > lo[a] + 8).all() and (p[:, a] < lo[a] + size[a] - 8).all() for a in range(3))
        r0 = p[4:36]                                   # stations of blade 0 at 2.25 .. 17.75 cells from the hub: inside the core
        assert all((r0[:, a] > lo[a] + 64).all() and (r0[:, a] < lo[a] + size[a] - 64).all() for a in range(3))
    check_samples(w, Wg, [lo], size=size, need=[("alm",)], steps=10, tol=1e-9, margin=64)


def test_C5_turbine_ten_steps_sampled():
    """config 5 at 512x256x256, ten steps, rotor turning: a 152 x 152 x 172 sub-box standing on the ground (the slip wall
    keeps its boundary condition, margin 0 there) that holds the rotor disc, the nacelle and the whole tower; trusted core
    = 24 x 24 cells around the tower axis from the ground up to the nacelle (z < 108).  The cuts are 64 cells from the
    core and more than 60 from the body: in ten steps their influence (6 cells per step) reaches neither, so the IBM
    (which couples cells 3 apart through a Lagrangian point) cannot carry it further"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C5")
    Wg = gks.run_workload(w, steps=10)
    lo, size = (60, 52, 0), (152, 152, 172)
    q = w.ibm[0] / w.cfg.spacing[0]
    for a in range(3):                                 # the whole body is further than 60 + 3 cells from every cut
        assert (q[:, a] > lo[a] + (64 if lo[a] > 0 else 0)).all() and (q[:, a] < lo[a] + size[a] - 64).all()
    for s in (0, 9):
        p = w.alm(s)[0] / w.cfg.spacing[0]
        assert all((p[:, a] > lo[a] + 8).all() and (p[:, a] < lo[a] + size[a] - 8).all() for a in range(3))
    check_samples(w, Wg, [lo], size=size, need=[("alm", "ibm")], steps=10, tol=1e-9, margin=64)


def test_maximum_size_box_beyond_32_bit_indices():
    """768 x 640 x 576 = 283 M cells (84 GB of workspace of the 180 GB): the padded field has 2.9e8 doubles, so the
    flux arrays (8 fields) and the state are indexed beyond 2^31 - every index must be 64-bit.  One step on a
    periodic box: conservation to round-off (P7 holds at any size), finiteness, and parity with the oracle on
    sub-boxes at the origin, in the middle and at the far corner (the largest indices), where a wrapped index would
    read or write the wrong cell"""
    from paper_2603_11102_b200 import gks
    n = (768, 640, 576)
    L = 2.0 * np.pi
    cfg = GridConfig(n=n, spacing=tuple(L / m for m in n), nu=1e-4, bc=(wl.BC_PERIODIC,) * 6)
    x, y, z = [cfg.centres(a) for a in range(3)]
    sx, cx, sy, cy, sz, cz = np.sin(x), np.cos(x), np.sin(y), np.cos(y), np.sin(z), np.cos(z)
    W0 = np.empty((4, n[2], n[1], n[0]))
    W0[0] = 1.0 + 0.01 * (np.cos(2 * z)[:, None, None] * cy[None, :, None] * sx[None, None, :])
    W0[1] = 0.1 * (cz[:, None, None] * cy[None, :, None] * sx[None, None, :])
    W0[2] = -0.1 * (cz[:, None, None] * sy[None, :, None] * cx[None, None, :])
    W0[3] = 0.02 * (sz[:, None, None] * np.sin(2 * y)[None, :, None] * np.cos(3 * x)[None, None, :])
    W0[1:] *= W0[0]
    w = wl.Workload("max_size", cfg, W0, 0.4 * min(cfg.spacing) / 1.15, 1)
    g = gks.Gks(cfg)
    assert g.workspace_bytes > 8 * 2 ** 31                     # 8 flux fields alone pass 2^31 doubles
    g.set_state(W0)
    g.step(w.dt)
    Wg = g.get_state()
    g.close()
    assert np.isfinite(Wg).all()
    mscale = float(np.abs(W0[1:]).sum(dtype=np.longdouble))
    for c in range(4):
        s0, s1 = W0[c].sum(dtype=np.longdouble), Wg[c].sum(dtype=np.longdouble)
        ref = abs(float(s0)) if c == 0 else 1e-3 * mscale
        assert abs(float(s1 - s0)) <= 1e-12 * ref, (c, float(s1 - s0), ref)
    boxes = [(-14, -14, -14), (370, 300, 280), (n[0] - 20, n[1] - 20, n[2] - 20), (n[0] - 30, 5, n[2] - 40)]
    check_samples(w, Wg, boxes)
