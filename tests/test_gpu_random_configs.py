"""Parity of the CUDA path with the oracle on SEEDED RANDOM configurations: sizes 6..29 per axis (ragged against every
tile shape), any pair of boundary kinds per axis, stretched non-periodic axes, both RT, three viscosities, and any
mix of ALM points or an on-line rotor, IBM points with one or several forcing passes, body force, bulk-flux forcing
and the linear-weight tangential variant.  Two steps, north_star tolerance 1e-11.
Whatever the oracle accepts the library must accept, and the other way round."""
from dataclasses import replace

import numpy as np
import pytest

from conftest import rel_linf
from paper_2603_11102_b200.workloads import GridConfig, synthetic_rotor

pytestmark = pytest.mark.gpu

P, NS, SL, IN, OUT, EX = range(6)
KINDS = [(P, P), (NS, NS), (SL, SL), (NS, SL), (EX, EX), (IN, OUT), (OUT, IN), (IN, EX), (EX, NS), (SL, EX)]


def random_case(seed, wide=False, anywhere=False):
    rng = np.random.default_rng(seed)
    n = tuple(int(v) for v in rng.integers(6, 30, 3))
    if wide:        # two long axes and a short one: more tile columns than SMs, so whole-column waves AND a remainder
        n = [int(rng.integers(120, 200)), int(rng.integers(120, 200)), int(rng.integers(6, 12))]
        n = tuple(n[i] for i in rng.permutation(3))
    bc, inflow = [], [1.0, 0.0, 0.0, 0.0]
    for a in range(3):
        lo, hi = KINDS[rng.integers(len(KINDS))]
        bc += [lo, hi]
        if IN in (lo, hi) or OUT in (lo, hi):
            inflow[1 + a] = 0.1 if (lo == IN or hi == OUT) else -0.1
    sp = tuple(float(v) for v in rng.uniform(0.05, 0.15, 3))
    faces = [None] * 3
    for a in range(3):
        if bc[2 * a] != P and rng.random() < 0.4:
            faces[a] = np.cumsum(np.r_[0.0, rng.uniform(0.7, 1.3, n[a])]) * sp[a]
    cfg = GridConfig(n=n, faces=tuple(faces), spacing=sp, nu=float(rng.choice([0.0, 1e-3, 1e-2])), bc=tuple(bc),
                     inflow=tuple(inflow), RT=float(rng.choice([1.0, 0.7])))
    W0 = np.zeros((4, n[2], n[1], n[0]))
    W0[0] = 1 + 0.02 * rng.standard_normal(W0[0].shape)
    for c in range(3):
        W0[1 + c] = W0[0] * (inflow[1 + c] + 0.02 * rng.standard_normal(W0[0].shape))
    x0 = [cfg.face_coords(a)[0] for a in range(3)]
    length = [cfg.face_coords(a)[-1] - x0[a] for a in range(3)]
    alm = ibm = body = bulk = None
    if rng.random() < 0.6:
        k = int(rng.integers(1, 12))
        eps = float(rng.uniform(1.0, 2.0) * max(sp))
        if all(6 * eps < length[a] for a in range(3) if bc[2 * a] == P):
            inside = (0.0, 1.0) if anywhere else (0.1, 0.9)       # anywhere: supports cut by walls and faces
            pos = np.column_stack([x0[a] + rng.uniform(-0.2, 1.2, k) * length[a] if bc[2 * a] == P
                                   else x0[a] + rng.uniform(*inside, k) * length[a] for a in range(3)])
            alm = (pos, 0.05 * rng.standard_normal((k, 3)), eps)
    if all(f is None for f in faces) and rng.random() < 0.6:
        k = int(rng.integers(1, 30))
        inside = (0.0, 1.0) if anywhere else (0.3, 0.7)       # anywhere: next to walls, across periodic seams
        pos = np.column_stack([x0[a] + rng.uniform(*inside, k) * length[a] for a in range(3)])
        ibm = (pos, np.full(k, sp[0] * sp[1] * sp[2]) * rng.uniform(0.3, 1.0, k))
    if rng.random() < 0.3:
        body = tuple(0.01 * rng.standard_normal(3))
    if rng.random() < 0.2:
        bulk = (int(rng.integers(3)), 0.1)
    dt = 0.3 * min(cfg.widths(a).min() for a in range(3)) / 1.3
    extras = {"linear": rng.random() < 0.25, "passes": int(rng.integers(2, 6)) if ibm and rng.random() < 0.4 else 0,
              "rotor": None}
    if alm is None and rng.random() < 0.5:          # a small rotor about the middle of the box, axis +x
        R = 0.3 * min(length[1], length[2])
        eps = float(1.5 * max(sp))
        if all(6 * eps < length[a] for a in range(3) if bc[2 * a] == P):
            hub = tuple(x0[a] + 0.5 * length[a] for a in range(3))
            extras["rotor"] = synthetic_rotor(hub, R, eps, u_ref=0.1, tsr=5.0, nblades=int(rng.integers(2, 4)), npts=8,
                                              seed=seed, freestream_correction=bool(rng.integers(2)),
                                              tip_correction=bool(rng.integers(2)))
    # (drawn last, so that the cases above stay what they were) moving Lagrangian points; a rotor with stations refined at
    # root and tip and three airfoil sections (reading S28)
    extras["ibm_vel"] = 0.05 * rng.standard_normal((len(ibm[0]), 3)) if ibm and rng.random() < 0.5 else None
    if extras["rotor"] is not None and rng.random() < 0.5:
        r0 = extras["rotor"]
        extras["rotor"] = synthetic_rotor(r0.hub, r0.R, r0.eps, u_ref=0.1, tsr=5.0, nblades=r0.nblades, npts=8, seed=seed,
                                          refine=True, nsections=3, freestream_correction=r0.freestream_correction,
                                          tip_correction=r0.tip_correction)
    return cfg, W0, alm, ibm, body, bulk, dt, extras


def two_steps(solver, cfg, W0, alm, ibm, body, bulk, dt, extras):
    s = solver(cfg)
    try:
        if extras["linear"]:
            s.set_reconstruction(1)
        if alm:
            s.alm_set_points(*alm)
        if extras["rotor"] is not None:
            s.alm_set_rotor(extras["rotor"])
        if ibm:
            s.ibm_set_points(*ibm)
            if extras["passes"]:
                s.ibm_set_iterations(extras["passes"], 0.0)
            if extras["ibm_vel"] is not None:
                s.ibm_set_velocities(extras["ibm_vel"])
        if body:
            s.set_body_force(*body)
        if bulk:
            s.set_bulk_flux(*bulk)
        s.set_state(W0)
        for _ in range(2):
            s.step(dt)
        return s.get_state(), s.cfl_dt(0.4)
    finally:
        s.close()


@pytest.mark.parametrize("first", [0, 20, 40, 60, 80])
def test_twenty_random_configurations(first):
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    forced = 0
    for seed in range(first, first + 20):
        case = random_case(seed)
        try:
            Wo, dto = two_steps(ob.Oracle, *case)
        except ob.OracleError:
            with pytest.raises(gks.GksError):
                two_steps(gks.Gks, *case)
            continue
        Wg, dtg = two_steps(gks.Gks, *case)
        err = rel_linf(Wg, Wo)
        assert err <= 1e-11, (seed, case[0].n, case[0].bc, err)
        assert dtg == pytest.approx(dto, rel=1e-12)          # the CFL time step of the state after the two steps
        forced += any(c is not None for c in case[2:6]) or case[7]["rotor"] is not None
    assert forced >= 5


def slab_case(seed):
    """a random case whose x axis can be cut: uniform x, at least 6 cells per slab, periodic or closed or
    inflow/outflow x; forcing of every kind"""
    rng = np.random.default_rng(10_000 + seed)
    for trial in range(100):
        case = random_case(int(rng.integers(1 << 30)))
        cfg = case[0]
        world = int(rng.integers(2, 5))
        if cfg.faces[0] is None and cfg.n[0] // world >= 6 and OUT not in cfg.bc[2:]:   # include/gks.h: outflow on the cut axis only
            return case, world
    raise AssertionError("no cuttable case")


def slab_two_steps(case, world, mode="plain"):
    """mode: plain (exchange through buffers), overlap (the step in parts), push (neighbours write the ghosts directly)"""
    from paper_2603_11102_b200 import gks, slab
    cfg, W0, alm, ibm, body, bulk, dt, extras = case
    d = slab.SlabDecomposition(cfg, world)
    solvers = [gks.Gks(d.local_cfg(r)) for r in range(world)]
    try:
        for r, s in enumerate(solvers):
            if extras["linear"]:
                s.set_reconstruction(1)
            if ibm:
                s.ibm_set_points(*d.ibm_points(r, *ibm))
                if extras["passes"]:
                    s.ibm_set_iterations(extras["passes"], 0.0)
                if extras["ibm_vel"] is not None:
                    s.ibm_set_velocities(d.ibm_velocities(r, ibm[0], extras["ibm_vel"]))
            if body:
                s.set_body_force(*body)
            if bulk:
                s.set_bulk_flux(*bulk)
            s.set_state(d.scatter(W0, r))
        stepper = slab.SlabStepper(slab.LocalTransport(d), solvers, slab.BufferPool("cuda:0"))
        rot = slab.RotorDriver(d, extras["rotor"], "cuda:0") if extras["rotor"] is not None else None
        for _ in range(2):
            stepper.step(dt, before_forcing=(lambda s: s.alm_set_points(*d.alm_points(solvers.index(s), *alm))) if alm else None,
                         ibm=bool(ibm),
                         bulk=bool(bulk), rotor=rot, ibm_passes=max(extras["passes"], 1), overlap=mode == "overlap",
                         push=mode == "push")
        return d.gather([s.get_state() for s in solvers])
    finally:
        for s in solvers:
            s.close()


@pytest.mark.parametrize("first", [0, 15])
def test_fifteen_random_configurations_cut_into_x_slabs(first):
    """the x-slab path (f3) on random configurations, 2-4 sub-domains in this process: equal to the single-domain run of
    the library to round-off (the arithmetic of a cell does not depend on the sub-domain it sits in, up to the
    warp-uniform series length) and to the oracle within the north_star tolerance"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    for seed in range(first, first + 15):
        case, world = slab_case(seed)
        Ws = slab_two_steps(case, world, ("plain", "overlap", "push")[seed % 3])
        W1 = two_steps(gks.Gks, *case)[0]
        assert rel_linf(Ws, W1) <= 1e-13, (seed, world, case[0].n, case[0].bc)
        assert rel_linf(Ws, two_steps(ob.Oracle, *case)[0]) <= 1e-11, (seed, world)


def test_forty_random_configurations_with_points_anywhere_in_the_domain():
    """Lagrangian and actuator points up to the boundary faces: supports cut by walls (dropped beyond them, include/gks.h),
    wrapped across periodic seams, sitting on cell faces"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    with_points = 0
    for seed in range(2000, 2040):
        case = random_case(seed, anywhere=True)
        Wo, _ = two_steps(ob.Oracle, *case)
        Wg, _ = two_steps(gks.Gks, *case)
        assert rel_linf(Wg, Wo) <= 1e-11, (seed, case[0].n, case[0].bc)
        with_points += case[2] is not None or case[3] is not None
    assert with_points >= 15


@pytest.mark.parametrize("seed", [1, 2, 3, 4, 5, 6])
def test_wide_random_configurations_fill_whole_waves_of_the_persistent_kernel(seed):
    """about 200 tile columns on 148 SMs for the sweeps whose tile lies in the two long axes (whole-column waves plus an
    evenly cut remainder) and a few long columns for the others"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    case = random_case(1000 + seed, wide=True)
    err = rel_linf(two_steps(gks.Gks, *case)[0], two_steps(ob.Oracle, *case)[0])
    assert err <= 1e-11, (case[0].n, case[0].bc, err)


# ---------------------------------------------------------------- invalid input: refusal parity
def attempt(solver, cfg, W0, actions, dt):
    """'ok', or where it was refused and why"""
    try:
        s = solver(cfg)
    except Exception as e:
        return "create: " + str(e)[:70]
    try:
        for name, args in actions:
            getattr(s, name)(*args)
        s.set_state(W0)
        s.step(dt)
        return "ok" if np.isfinite(s.get_state()).all() else "nonfinite"
    except Exception as e:
        return "call: " + str(e)[:70]
    finally:
        s.close()


def defective_case(seed):
    """a random case with one random defect (or borderline value) in the configuration, the time step or a call"""
    rng = np.random.default_rng(50_000 + seed)
    cfg, W0, _, _, _, _, dt, _ = random_case(int(rng.integers(1 << 30)))
    x0 = [cfg.face_coords(a)[0] for a in range(3)]
    length = [cfg.face_coords(a)[-1] - x0[a] for a in range(3)]
    centre = np.array([[x0[a] + 0.5 * length[a] for a in range(3)]])
    actions = []
    defect, a = int(rng.integers(12)), int(rng.integers(3))
    if defect == 0:       # ALM width: zero, negative, just above / below a sixth of the shortest axis
        eps = float(rng.choice([0.0, -1.0, min(length) / 5.9, min(length) / 6.1]))
        actions.append(("alm_set_points", (centre, np.ones((1, 3)), eps)))
    elif defect == 1:     # ALM point outside the domain along axis a
        p = centre.copy()
        p[0, a] = x0[a] + float(rng.choice([-0.05, 1.05, -3.0, 4.0])) * length[a]
        actions.append(("alm_set_points", (p, np.ones((1, 3)), 1.2 * max(cfg.spacing))))
    elif defect == 2:     # IBM point near, on or beyond a boundary face of axis a
        p = centre.copy()
        p[0, a] = x0[a] + float(rng.choice([-0.01, 0.0, 0.01, 0.5, 0.99, 1.0, 1.01])) * length[a]
        actions.append(("ibm_set_points", (p, np.array([1e-3]))))
    elif defect == 3:     # IBM points on whatever grid the case has (stretched axes are refused)
        p = np.column_stack([x0[b] + rng.uniform(0.05, 0.95, 5) * length[b] for b in range(3)])
        actions.append(("ibm_set_points", (p, np.full(5, 1e-3))))
    elif defect == 4:     # periodic on one side only
        bc = list(cfg.bc)
        bc[2 * a], bc[2 * a + 1] = P, int(rng.choice([NS, EX, P]))
        cfg = replace(cfg, bc=tuple(bc), faces=(None, None, None))
    elif defect == 5:     # 1..6 cells along axis a
        n = list(cfg.n)
        n[a] = int(rng.integers(1, 7))
        cfg = replace(cfg, n=tuple(n), faces=(None, None, None))
        W0 = np.ones((4, n[2], n[1], n[0]))
        W0[1:] = 0.0
    elif defect == 6:
        dt = float(rng.choice([0.0, -1e-3, np.nan]))
    elif defect == 7:
        cfg = replace(cfg, RT=float(rng.choice([0.0, -1.0, 1.0])), nu=float(rng.choice([-1e-3, 0.0])))
    elif defect == 8:     # face coordinates that do not increase
        f = np.cumsum(np.r_[0.0, np.full(cfg.n[a], cfg.spacing[a])])
        f[3] = f[2] if rng.random() < 0.5 else f[1]
        faces, bc = list(cfg.faces), list(cfg.bc)
        faces[a] = f
        if bc[2 * a] == P:
            bc[2 * a] = bc[2 * a + 1] = EX
        cfg = replace(cfg, faces=tuple(faces), bc=tuple(bc))
    elif defect == 9:
        actions.append(("set_bulk_flux", (int(rng.choice([-1, 0, 2, 3, 7])), 0.1)))
    elif defect == 10:    # (more than 64 passes is a limit of the library only, include/gks.h)
        actions.append(("ibm_set_iterations", (int(rng.choice([0, -1, 1, 64])), float(rng.choice([0.0, -1.0, 1e-3])))))
    else:
        actions.append(("set_reconstruction", (int(rng.choice([-1, 0, 1, 2])),)))
    return cfg, W0, actions, dt


@pytest.mark.parametrize("first", [0, 50, 100])
def test_what_the_oracle_refuses_the_library_refuses(first):
    """ALM width against the periodic axes, points outside or on the boundary, IBM on stretched grids, unpaired
    periodic faces, fewer than 6 cells, dt <= 0 or NaN, RT <= 0, nu < 0, non-increasing faces, bad axis / pass count /
    variant arguments: the same accept-or-refuse decision on both sides, and a finite state wherever both accept"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    refused = 0
    for seed in range(first, first + 50):
        cfg, W0, actions, dt = defective_case(seed)
        ro, rg = attempt(ob.Oracle, cfg, W0, actions, dt), attempt(gks.Gks, cfg, W0, actions, dt)
        assert (ro == "ok") == (rg == "ok"), (seed, ro, rg)
        refused += ro != "ok"
    assert 5 <= refused <= 45
