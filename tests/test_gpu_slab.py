"""x-slab decomposition on ONE GPU: all sub-domains live in this process (slab.LocalTransport hands the packed
halo buffers over; no kernel waits on another).  The decomposed run must reproduce the single-domain run of the
same library - the arithmetic of a cell does not depend on which sub-domain it sits in - and the oracle."""
import numpy as np
import pytest
import torch

from conftest import rel_linf
from paper_2603_11102_b200 import slab, workloads as wl

pytestmark = pytest.mark.gpu


def run_slabs(w, world, steps, linear=False, overlap=False, push=False):
    from paper_2603_11102_b200 import gks
    d = slab.SlabDecomposition(w.cfg, world)
    solvers = [gks.Gks(d.local_cfg(r)) for r in range(world)]
    for r, s in enumerate(solvers):
        if linear:
            s.set_reconstruction(1)
        if w.ibm is not None:
            s.ibm_set_points(*d.ibm_points(r, *w.ibm))
        if w.bulk_flux is not None:
            s.set_bulk_flux(*w.bulk_flux)
        s.set_state(d.scatter(w.W0, r))
    newbuf = slab.BufferPool("cuda:0")
    stepper = slab.SlabStepper(slab.LocalTransport(d), solvers, newbuf)
    for k in range(steps):
        pts = w.alm(k) if w.alm is not None else None
        stepper.step(w.dt, before_forcing=(lambda s: s.alm_set_points(*pts)) if pts is not None else None,
                     ibm=w.ibm is not None, bulk=w.bulk_flux is not None, overlap=overlap, push=push)
    W = d.gather([s.get_state() for s in solvers])
    for s in solvers:
        s.close()
    return W


def run_single(w, steps, linear=False):
    from paper_2603_11102_b200 import gks
    g = gks.Gks(w.cfg)
    if linear:
        g.set_reconstruction(1)
    if w.ibm is not None:
        g.ibm_set_points(*w.ibm)
    if w.bulk_flux is not None:
        g.set_bulk_flux(*w.bulk_flux)
    g.set_state(w.W0)
    for k in range(steps):
        if w.alm is not None:
            g.alm_set_points(*w.alm(k))
        g.step(w.dt)
    W = g.get_state()
    g.close()
    return W


@pytest.mark.parametrize("world", [2, 3])
def test_periodic_box_in_slabs_equals_the_single_domain(world):
    w = wl.by_name("C1")                                     # 32^3 periodic: slabs of 16 / 11, 11, 10 cells
    Ws, W1 = run_slabs(w, world, 5), run_single(w, 5)
    # same arithmetic per cell up to the warp-uniform choice of the erf/exp series length, which depends on the
    # other faces of the tile (8 terms if all have z^2 <= 1/64, else 12/14): both are exact to 1e-17
    assert rel_linf(Ws, W1) <= 1e-13


@pytest.mark.parametrize("world", [2, 3])
def test_channel_with_bulk_flux_forcing_in_slabs(world):
    """small C2: periodic x, stretched no-slip y, bulk-flux forcing = one global sum per step, assembled from the
    sub-domains' partial sums"""
    from oracle import binding as ob
    w = wl.by_name("C2", small=True)
    Ws, W1 = run_slabs(w, world, 3), run_single(w, 3)
    assert rel_linf(Ws, W1) <= 1e-13
    o = ob.Oracle(w.cfg)
    o.set_bulk_flux(*w.bulk_flux)
    o.set_state(w.W0)
    for _ in range(3):
        o.step(w.dt)
    assert rel_linf(Ws, o.get_state()) <= 3e-11
    vol = np.einsum("k,j,i->kji", w.cfg.widths(2), w.cfg.widths(1), w.cfg.widths(0))
    assert (Ws[1] * vol).sum() / vol.sum() == pytest.approx(w.bulk_flux[1], rel=1e-12)
    o.close()


def test_rotor_box_in_four_slabs_with_the_rotor_on_a_cut():
    """small C4: inflow / convective outflow along x, periodic y, slip z, prescribed ALM points whose Gaussian
    supports straddle the cut between slab 0 and slab 1 (hub at cell 24 of 96 = the cut)"""
    from oracle import binding as ob
    w = wl.by_name("C4", small=True)
    d = slab.SlabDecomposition(w.cfg, 4)
    hub_x = w.alm(0)[0][:, 0].mean()
    assert abs(hub_x / w.cfg.spacing[0] - d.owned(1)[0]) < 1.0
    Ws, W1 = run_slabs(w, 4, 3), run_single(w, 3)
    assert rel_linf(Ws, W1) <= 1e-14
    o = ob.Oracle(w.cfg)
    o.set_state(w.W0)
    for k in range(3):
        o.alm_set_points(*w.alm(k))
        o.step(w.dt)
    assert rel_linf(Ws, o.get_state()) <= 3e-11
    o.close()


@pytest.mark.parametrize("name", ["C3", "C5"])
def test_ibm_bodies_across_cuts(name):
    """small cylinder (C3: 64 cells along x, cylinder at x = 16 = the first cut of 4 slabs) and turbine (C5: ALM
    rotor + IBM nacelle and tower) boxes: Lagrangian points next to a cut are known to both sub-domains"""
    from oracle import binding as ob
    w = wl.by_name(name, small=True)
    for world in range(2, 9):                                 # the first decomposition that cuts through the body
        d = slab.SlabDecomposition(w.cfg, world)
        cuts = w.cfg.origin[0] + d.x_lo[1:-1] * w.cfg.spacing[0]
        if np.abs(w.ibm[0][:, :1] - cuts[None, :]).min() < 0.5 * w.cfg.spacing[0]:
            break
    shared = sum(len(d.ibm_points(r, *w.ibm)[0]) for r in range(world)) - len(w.ibm[0])
    assert shared > 0                                         # the case does exercise the cut
    Ws, W1 = run_slabs(w, world, 3), run_single(w, 3)
    assert rel_linf(Ws, W1) <= 1e-13                          # fp64 atomics of the spreading: order only
    o = ob.Oracle(w.cfg)
    o.ibm_set_points(*w.ibm)
    o.set_state(w.W0)
    for k in range(3):
        if w.alm is not None:
            o.alm_set_points(*w.alm(k))
        o.step(w.dt)
    assert rel_linf(Ws, o.get_state()) <= 3e-11
    o.close()


@pytest.mark.parametrize("name,switches", [("C4", {}), ("C5", {"freestream_correction": True, "tip_correction": True})])
def test_online_rotor_on_slabs(name, switches):
    """the on-line rotor with the disc ON a cut (hub at cell 24 of 96 = the first cut of 4 slabs: the sampling of
    the owner reads its HALO ghosts), with IBM bodies for the turbine: the decomposed run reproduces the
    single-domain run with alm_set_rotor, and the oracle"""
    from oracle import binding as ob
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=True)
    pos0, _, eps = w.alm(0)
    hub = pos0.reshape(3, -1, 3).mean(axis=(0, 1))
    r = wl.synthetic_rotor(hub=hub, R=float(np.linalg.norm(pos0 - hub, axis=1).max() * 64.5 / 64.0), eps=eps, npts=40,
                           **switches)
    world, steps = 4, 3
    d = slab.SlabDecomposition(w.cfg, world)
    assert abs(hub[0] / w.cfg.spacing[0] - d.owned(1)[0]) < 0.5
    solvers = [gks.Gks(d.local_cfg(k)) for k in range(world)]
    for k, s in enumerate(solvers):
        if w.ibm is not None:
            s.ibm_set_points(*d.ibm_points(k, *w.ibm))
        s.set_state(d.scatter(w.W0, k))
    stepper = slab.SlabStepper(slab.LocalTransport(d), solvers, slab.BufferPool("cuda:0"))
    rot = slab.RotorDriver(d, r, "cuda:0")
    assert rot.owner == 1
    for _ in range(steps):
        stepper.step(w.dt, ibm=w.ibm is not None, rotor=rot)
    Ws = d.gather([s.get_state() for s in solvers])
    for s in solvers:
        s.close()
    o, g = ob.Oracle(w.cfg), gks.Gks(w.cfg)
    for s in (o, g):
        if w.ibm is not None:
            s.ibm_set_points(*w.ibm)
        s.set_state(w.W0)
        s.alm_set_rotor(r)
        for _ in range(steps):
            s.step(w.dt)
    assert rel_linf(Ws, g.get_state()) <= 1e-13
    assert rel_linf(Ws, o.get_state()) <= 3e-11
    with pytest.raises(gks.GksError):
        g.alm_rotor_points(r, 0.0)                           # refused while a rotor is set
    g.close()
    o.close()


@pytest.mark.parametrize("name", ["C3", "C5"])
def test_ibm_passes_on_slabs(name):
    """multi-direct-forcing passes with the body cut through: a fixed number of passes, and the stop rule with a
    tolerance that ends the passes early - the decision is taken from the MAX of the sub-domains' slips"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=True)
    for world in range(2, 9):
        d = slab.SlabDecomposition(w.cfg, world)
        cuts = w.cfg.origin[0] + d.x_lo[1:-1] * w.cfg.spacing[0]
        if np.abs(w.ibm[0][:, :1] - cuts[None, :]).min() < 0.5 * w.cfg.spacing[0]:
            break

    def single(passes, tol):
        g = gks.Gks(w.cfg)
        g.ibm_set_points(*w.ibm)
        g.ibm_set_iterations(passes, tol)
        g.set_state(w.W0)
        for k in range(2):
            if w.alm is not None:
                g.alm_set_points(*w.alm(k))
            g.step(w.dt)
        W = g.get_state()
        g.close()
        return W

    def slabs(passes, tol):
        solvers = [gks.Gks(d.local_cfg(r)) for r in range(world)]
        for r, s in enumerate(solvers):
            s.ibm_set_points(*d.ibm_points(r, *w.ibm))
            s.ibm_set_iterations(passes, tol)
            s.set_state(d.scatter(w.W0, r))
        st = slab.SlabStepper(slab.LocalTransport(d), solvers, slab.BufferPool("cuda:0"))
        for k in range(2):
            pts = w.alm(k) if w.alm is not None else None
            st.step(w.dt, before_forcing=(lambda s: s.alm_set_points(*pts)) if pts is not None else None, ibm=True,
                    ibm_passes=passes)
        W = d.gather([s.get_state() for s in solvers])
        for s in solvers:
            s.close()
        return W

    W1, W3, W8 = single(1, 0.0), single(3, 0.0), single(8, 0.0)
    assert rel_linf(slabs(3, 0.0), W3) <= 1e-13
    # a tolerance between the slips that stop after 3 passes: the result equals the 3-pass one, not the 8-pass one
    o_slip = []
    for k in (2, 3):
        g = gks.Gks(w.cfg)
        g.ibm_set_points(*w.ibm)
        g.ibm_set_iterations(k, 0.0)
        g.set_state(w.W0)
        if w.alm is not None:
            g.alm_set_points(np.zeros((0, 3)), np.zeros((0, 3)), 1.0)
        g.step(w.dt)
        from oracle import binding as ob
        o = ob.Oracle(w.cfg)
        o.ibm_set_points(*w.ibm)
        o.set_state(g.get_state())
        o_slip.append(np.linalg.norm(o.ibm_interpolate(), axis=1).max())
        o.close()
        g.close()
    tol = 0.5 * (o_slip[0] + o_slip[1])
    Wt = slabs(8, tol)
    assert rel_linf(Wt, single(8, tol)) <= 1e-13
    assert rel_linf(Wt, W8) > 1e-9 and rel_linf(W3, W1) > 1e-9


def test_linear_variant_and_error_paths():
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C1")
    assert rel_linf(run_slabs(w, 2, 2, linear=True), run_single(w, 2, linear=True)) <= 1e-13
    d = slab.SlabDecomposition(w.cfg, 2)
    g = gks.Gks(d.local_cfg(0))
    buf = torch.empty(g.halo_doubles(0), dtype=torch.float64, device="cuda:0")
    with pytest.raises(gks.GksError):
        g.halo_pack(0, 0, buf)                               # before set_state
    g.set_state(d.scatter(w.W0, 0))
    with pytest.raises(gks.GksError):
        g.halo_pack(1, 0, buf)                               # W* only exists inside a step
    with pytest.raises(gks.GksError):
        g.step_finish(w.dt)                                  # without begin
    g.set_bulk_flux(0, 0.1)

    def fill_halo_ghosts(which):
        # the contract of gks_step_begin / gks_step_finish: HALO ghosts in place.  Any finite data will do here:
        # the sub-domain is its own neighbour (what it packs at one face it unpacks beyond the other)
        for src, dst in ((0, 1), (1, 0)):
            g.halo_pack(which, src, buf)
            g.halo_unpack(which, dst, buf)

    fill_halo_ghosts(0)
    g.step_begin(w.dt)
    fill_halo_ghosts(1)
    g.step_finish(w.dt)
    with pytest.raises(gks.GksError):
        g.step_force(w.dt)                                   # the global bulk sum was not supplied
    part = torch.zeros(1, dtype=torch.float64, device="cuda:0")
    torch.cuda.synchronize()                                 # the fill runs on torch's stream, the solver on its own
    vol = g.bulk_partial(part)
    g.bulk_set_global(part, vol)
    g.step_force(w.dt)
    g.set_bulk_flux(-1, 0.0)
    g.halo_pack(0, 0, buf)
    host = torch.empty(g.halo_doubles(1), dtype=torch.float64)
    g.halo_pack(0, 1, host)                                  # host buffers are accepted too
    assert torch.isfinite(host).all() and torch.isfinite(buf).all()
    g.close()
    single = gks.Gks(w.cfg)
    single.set_state(w.W0)
    with pytest.raises(gks.GksError):
        single.halo_pack(0, 0, torch.empty(single.halo_doubles(0), dtype=torch.float64, device="cuda:0"))   # not a HALO face
    single.close()


def test_rotor_and_points_at_the_seam_of_a_periodic_x_axis():
    """a rotor disc and prescribed actuator points within 3 eps of the periodic seam: the slab on the far side of the seam
    meets them through their images (SlabDecomposition.alm_points, seam_shift)"""
    from paper_2603_11102_b200 import gks
    from paper_2603_11102_b200.workloads import GridConfig
    n, h = (30, 12, 12), 0.1
    cfg = GridConfig(n=n, spacing=(h, h, h), nu=1e-3, bc=(0,) * 6)
    rng = np.random.default_rng(4)
    W0 = np.zeros((4, n[2], n[1], n[0]))
    W0[0] = 1 + 0.01 * rng.standard_normal(W0[0].shape)
    W0[1] = 0.1 * W0[0]
    eps, dt, world = 0.15, 0.02, 3
    rotor = wl.synthetic_rotor(hub=(0.04, 0.6, 0.6), R=0.4, eps=eps, u_ref=0.1, tsr=5.0, npts=10)
    pos = np.column_stack([rng.uniform(-0.3, 3.3, 12), rng.uniform(0, 1.2, 12), rng.uniform(0, 1.2, 12)])
    force = 0.05 * rng.standard_normal((12, 3))
    d = slab.SlabDecomposition(cfg, world)
    for use_rotor in (True, False):
        solvers = [gks.Gks(d.local_cfg(r)) for r in range(world)]
        for r, s in enumerate(solvers):
            s.set_state(d.scatter(W0, r))
        stepper = slab.SlabStepper(slab.LocalTransport(d), solvers, slab.BufferPool("cuda:0"))
        rot = slab.RotorDriver(d, rotor, "cuda:0") if use_rotor else None
        hook = None if use_rotor else (lambda s: s.alm_set_points(*d.alm_points(solvers.index(s), pos, force, eps)))
        for _ in range(3):
            stepper.step(dt, before_forcing=hook, rotor=rot)
        Ws = d.gather([s.get_state() for s in solvers])
        for s in solvers:
            s.close()
        g = gks.Gks(cfg)
        g.set_state(W0)
        if use_rotor:
            g.alm_set_rotor(rotor)
        else:
            g.alm_set_points(pos, force, eps)
        for _ in range(3):
            g.step(dt)
        W1 = g.get_state()
        g.close()
        assert rel_linf(Ws, W1) <= 1e-13, use_rotor
        # the forcing does reach the last slab (beyond the seam)
        free = gks.Gks(cfg)
        free.set_state(W0)
        for _ in range(3):
            free.step(dt)
        assert np.abs(W1 - free.get_state())[..., -3:].max() > 1e-6
        free.close()


@pytest.mark.parametrize("name,world,small", [("C1", 2, True), ("TG160", 2, False), ("C3", 2, False), ("C4", 3, True), ("C2", 2, False)])
def test_overlapped_step_equals_the_plain_step(name, world, small):
    """gks_step_begin_part / gks_step_finish_part (interior while the halos travel, then the rim): the same tiles and
    cells in another order - bit for bit the plain decomposed step on a periodic box (no interior at 16 cells per
    slab: the rim is everything; cells 32 .. 64 of 80 on the 160^3 box), to the order of the fp64 atomics with IBM; and the call order is enforced.
    C3 at its full 256 x 128 x 64 (slabs of 128 cells: interior 32 .. 96) has inflow / outflow along x and the body
    in the rim-interior seam of slab 0; C2 at 128 x 96 x 64 adds the bulk-flux all-reduce"""
    from paper_2603_11102_b200 import gks
    w = wl.taylor_green(160) if name == "TG160" else wl.by_name(name, small=small)   # 160: slabs of 80, interior 32 .. 64
    steps = 2
    Wp, Wo = run_slabs(w, world, steps), run_slabs(w, world, steps, overlap=True)
    if w.ibm is None:
        assert np.array_equal(Wo, Wp)
    else:
        assert rel_linf(Wo, Wp) <= 1e-14
    assert rel_linf(Wo, run_single(w, steps)) <= 1e-13
    d = slab.SlabDecomposition(w.cfg, world)
    g = gks.Gks(d.local_cfg(0))
    g.set_state(d.scatter(w.W0, 0))
    with pytest.raises(gks.GksError):
        g.step_begin_part(w.dt, 1)                           # the rim before the interior
    g.step_begin_part(w.dt, 0)
    with pytest.raises(gks.GksError):
        g.step_begin_part(w.dt, 0)
    with pytest.raises(gks.GksError):
        g.step_finish(w.dt)
    g.close()


@pytest.mark.parametrize("name,world", [("C1", 3), ("C3", 4), ("C5", 3), ("C2", 2)])
def test_exchange_by_direct_push_equals_the_buffered_exchange(name, world):
    """gks_halo_push: every sub-domain writes its boundary planes straight into its neighbours' ghost layers (pack,
    transfer and unpack in one kernel; slabs of unequal width have different pitches and field strides) - the same
    bits as the exchange through buffers; refusals"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=name != "C1")
    Wb, Wp = run_slabs(w, world, 2), run_slabs(w, world, 2, push=True)
    if w.ibm is None:
        assert np.array_equal(Wp, Wb)
    else:
        assert rel_linf(Wp, Wb) <= 1e-14
    d = slab.SlabDecomposition(w.cfg, world)
    g0, g1 = gks.Gks(d.local_cfg(0)), gks.Gks(d.local_cfg(1))
    g0.set_state(d.scatter(w.W0, 0))
    g1.set_state(d.scatter(w.W0, 1))
    win = g1.halo_window(0)
    assert win.nx == d.local_cfg(1).n[0] and win.pitch_x >= win.nx + 6 and win.W
    g0.halo_push(0, 1, win)
    with pytest.raises(gks.GksError):
        g0.halo_push(0, 2, win)                              # not an x face
    with pytest.raises(gks.GksError):
        g0.halo_push(1, 1, win)                              # W* only exists inside a step
    win.ny += 1
    with pytest.raises(gks.GksError):
        g0.halo_push(0, 1, win)                              # extents differ
    g0.close()
    g1.close()


@pytest.mark.parametrize("name,world", [("C1", 2), ("C1", 3), ("C3", 4), ("C5", 3), ("C2", 2)])
def test_stage_update_that_writes_the_neighbours_ghosts_equals_the_buffered_exchange(name, world):
    """gks_step_begin_push: the stage-1 update kernel also stores the boundary planes of W* into the ghost layers of the
    sub-domains beyond its cut faces (update, pack, transfer and unpack in one kernel): the same bits as the exchange
    through buffers (two slabs on a periodic axis: the same neighbour on both sides); refusals"""
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=name != "C1")
    Wb, Wf = run_slabs(w, world, 3), run_slabs(w, world, 3, push="fused")
    if w.ibm is None:
        assert np.array_equal(Wf, Wb)
    else:
        assert rel_linf(Wf, Wb) <= 1e-14
    d = slab.SlabDecomposition(w.cfg, world)
    g0, g1 = gks.Gks(d.local_cfg(0)), gks.Gks(d.local_cfg(1))
    g0.set_state(d.scatter(w.W0, 0))
    g1.set_state(d.scatter(w.W0, 1))
    win = g1.halo_window(1)
    if d.local_cfg(0).bc[0] != slab.BC_HALO:
        with pytest.raises(gks.GksError):
            g0.step_begin_push(w.dt, win, None)              # my low face is not a cut
    win.nz += 1
    with pytest.raises(gks.GksError):
        g0.step_begin_push(w.dt, None, win)                  # extents differ
    win.nz -= 1
    with pytest.raises(gks.GksError):
        g0.step_begin_push(-1.0, None, win)
    g0.step_begin_push(w.dt, None, win)                      # accepted; the step is open now
    with pytest.raises(gks.GksError):
        g0.step_begin_push(w.dt, None, win)
    g0.close()
    g1.close()
