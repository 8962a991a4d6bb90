"""Host logic of the x-slab decomposition (paper_2603_11102_b200/slab.py) without a GPU: ownership, sub-domain
configurations, the exchange schedule, and the torch.distributed transport with world_size 2 and 3 over gloo,
driven by a numpy stand-in for the solver that implements gks_halo_pack / gks_halo_unpack as array slices."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2603_11102_b200 import slab, workloads as wl
from paper_2603_11102_b200.workloads import GridConfig

NG = 3


class FakeSolver:
    """padded field [c][k][j][i] with 3 ghost layers in x only; pack / unpack follow include/gks.h"""

    def __init__(self, cfg, W):
        self.n = cfg.n
        self.W = np.full((4, cfg.n[2], cfg.n[1], cfg.n[0] + 2 * NG), np.nan)
        self.W[..., NG:-NG] = W
        self.Ws = self.W.copy()

    def halo_doubles(self, face):
        return 4 * NG * self.n[1] * self.n[2]

    def _arr(self, which):
        return self.W if which == 0 else self.Ws

    def halo_pack(self, which, face, buf):
        A = self._arr(which)
        sl = A[..., NG:2 * NG] if face == 0 else A[..., -2 * NG:-NG]
        buf.copy_(torch.from_numpy(np.ascontiguousarray(np.moveaxis(sl, -1, 1)).reshape(-1)))   # [c][layer][k][j]

    def halo_unpack(self, which, face, buf):
        A = self._arr(which)
        planes = np.moveaxis(buf.numpy().reshape(4, NG, self.n[2], self.n[1]), 1, -1)
        if face == 0:
            A[..., :NG] = planes
        else:
            A[..., -NG:] = planes

    def synchronize(self):
        pass


def test_ownership_and_local_configurations():
    cfg = GridConfig(n=(32, 8, 8), spacing=(0.1, 0.1, 0.1), bc=(0,) * 6)
    d = slab.SlabDecomposition(cfg, 3)
    assert [d.owned(r) for r in range(3)] == [(0, 11), (11, 22), (22, 32)]
    assert d.neighbours(0) == (2, 1) and d.neighbours(2) == (1, 0)
    c1 = d.local_cfg(1)
    assert c1.n == (11, 8, 8) and c1.bc[:2] == (6, 6) and c1.origin[0] == pytest.approx(1.1)
    w = wl.by_name("C4", small=True)                                   # inflow / outflow along x
    d = slab.SlabDecomposition(w.cfg, 4)
    assert d.neighbours(0) == (None, 1) and d.neighbours(3) == (2, None)
    assert d.local_cfg(0).bc[:2] == (wl.BC_INFLOW, 6) and d.local_cfg(3).bc[:2] == (6, wl.BC_OUTFLOW_CONVECTIVE)
    assert d.local_cfg(2).bc[2:] == w.cfg.bc[2:]
    parts = [d.scatter(w.W0, r) for r in range(4)]
    assert np.array_equal(d.gather(parts), w.W0)
    assert slab.SlabDecomposition(cfg, 1).local_cfg(0).bc == cfg.bc and slab.SlabDecomposition(cfg, 1).schedule(0) == []
    with pytest.raises(ValueError):
        slab.SlabDecomposition(cfg, 6)                                  # 5 cells per slab: too thin


def _check_ghosts(d, rank, s, W, which):
    """ghost planes of the sub-domain = the global field's planes next door (periodic wrap included)"""
    i0, i1 = d.owned(rank)
    nx = d.cfg.n[0]
    lo, hi = d.neighbours(rank)
    A = s._arr(which)
    if lo is not None:
        idx = np.arange(i0 - NG, i0) % nx
        assert np.array_equal(A[..., :NG], W[..., idx])
    if hi is not None:
        idx = np.arange(i1, i1 + NG) % nx
        assert np.array_equal(A[..., -NG:], W[..., idx])


@pytest.mark.parametrize("world,periodic", [(2, True), (3, True), (3, False)])
def test_local_transport_moves_the_right_planes(world, periodic):
    rng = np.random.default_rng(world)
    bc = (0, 0) if periodic else (wl.BC_INFLOW, wl.BC_EXTRAPOLATE)
    cfg = GridConfig(n=(20, 5, 4), spacing=(0.1,) * 3, bc=bc + (0, 0, 0, 0))
    W = rng.standard_normal((4, 4, 5, 20))
    d = slab.SlabDecomposition(cfg, world)
    solvers = [FakeSolver(d.local_cfg(r), d.scatter(W, r)) for r in range(world)]
    t = slab.LocalTransport(d)
    newbuf = slab.BufferPool("cpu")
    t.exchange(solvers, 0, newbuf)
    for r, s in enumerate(solvers):
        _check_ghosts(d, r, s, W, 0)


def _dist_worker(rank, world, port, periodic, W, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        bc = (0, 0) if periodic else (wl.BC_INFLOW, wl.BC_EXTRAPOLATE)
        cfg = GridConfig(n=(W.shape[-1], W.shape[2], W.shape[1]), spacing=(0.1,) * 3, bc=bc + (0, 0, 0, 0))
        d = slab.SlabDecomposition(cfg, world)
        s = FakeSolver(d.local_cfg(rank), d.scatter(W, rank))
        s.Ws[..., NG:-NG] *= 2.0                               # a different field for which = 1
        t = slab.DistTransport(d, rank)
        newbuf = slab.BufferPool("cpu")
        t.exchange(s, 0, newbuf)
        t.exchange(s, 1, newbuf)
        _check_ghosts(d, rank, s, W, 0)
        _check_ghosts(d, rank, s, 2.0 * W, 1)
        # the rotor driver's broadcast: the owner's arrays arrive everywhere
        a = torch.full((5, 3), float(rank)) if rank == world - 1 else torch.zeros((5, 3))
        t.broadcast(s, world - 1, [a])
        assert torch.equal(a, torch.full((5, 3), float(world - 1)))
        tot, vol = t.all_reduce_sum(s, torch.tensor([float(rank + 1)], dtype=torch.float64), 0.5 * (rank + 1))
        assert float(tot) == world * (world + 1) / 2 and vol == pytest.approx(0.25 * world * (world + 1))
        top = t.all_reduce_max(s, torch.tensor([0.1 * (rank + 1)], dtype=torch.float64))
        assert float(top) == pytest.approx(0.1 * world)
        q.put((rank, "ok"))
    except Exception as e:                                      # noqa: BLE001 - reported to the parent
        q.put((rank, repr(e)))
    finally:
        dist.destroy_process_group()


@pytest.mark.parametrize("world,periodic", [(2, True), (2, False), (3, True)])
def test_dist_transport_over_gloo(world, periodic):
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    W = np.random.default_rng(7).standard_normal((4, 3, 4, 19))
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_dist_worker, args=(r, world, port, periodic, W, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = dict(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
    assert res == {r: "ok" for r in range(world)}, res


def test_ibm_points_are_shared_across_cuts_and_wrapped_on_a_periodic_axis():
    h = 0.1
    cfg = GridConfig(n=(24, 8, 8), spacing=(h, h, h), bc=(wl.BC_INFLOW, wl.BC_EXTRAPOLATE, 0, 0, 0, 0))
    d = slab.SlabDecomposition(cfg, 2)                                  # cut at x = 1.2
    pos = np.array([[0.05, .4, .4], [1.10, .4, .4], [1.26, .4, .4], [1.40, .4, .4], [2.35, .4, .4]])
    vol = np.arange(5.0)
    p0, v0 = d.ibm_points(0, pos, vol)
    p1, v1 = d.ibm_points(1, pos, vol)
    assert list(v0) == [0, 1, 2] and list(v1) == [1, 2, 3, 4]           # 1.10 and 1.26 are within 1.5 h of the cut
    assert np.array_equal(p0, pos[:3]) and np.array_equal(p1, pos[1:])
    per = GridConfig(n=(24, 8, 8), spacing=(h, h, h), bc=(0,) * 6)
    d = slab.SlabDecomposition(per, 2)
    p0, v0 = d.ibm_points(0, pos, vol)
    p1, v1 = d.ibm_points(1, pos, vol)
    # across the periodic seam: the point at 2.35 is also seen by slab 0 at x = -0.05, the one at 0.05 by slab 1 at 2.45
    assert sorted(v0) == [0, 1, 2, 4] and sorted(v1) == [0, 1, 2, 3, 4]
    assert p0[list(v0).index(4), 0] == pytest.approx(-0.05) and p1[list(v1).index(0), 0] == pytest.approx(2.45)
    assert slab.SlabDecomposition(per, 1).ibm_points(0, pos, vol)[0].shape == pos.shape


def test_rotor_driver_owner_is_the_slab_that_contains_the_disc():
    w = wl.by_name("C4", small=True)                                    # 96 cells along x, hub at x = 3 = cell 24
    r = wl.synthetic_rotor(hub=(3.0, 3.0, 3.0), R=1.0, eps=0.25)
    for world, owner in ((1, 0), (2, 0), (4, 1), (5, 1)):
        assert slab.RotorDriver(slab.SlabDecomposition(w.cfg, world), r, "cpu").owner == owner
    r2 = wl.synthetic_rotor(hub=(2.99, 3.0, 3.0), R=1.0, eps=0.25)
    assert slab.RotorDriver(slab.SlabDecomposition(w.cfg, 4), r2, "cpu").owner == 0


@pytest.mark.parametrize("periodic", [True, False])
@pytest.mark.parametrize("world", [2, 3, 4])
def test_alm_points_reach_every_slab_they_act_on(world, periodic):
    """brute force: the Gaussian sums (cut at 3 eps) that the sub-domains form over the cells they own, from the
    points `alm_points` gives them and WITHOUT any wrap along x, equal the sums of the whole domain with the
    nearest image along a periodic x; points outside [0, L) and supports across the seam included"""
    n, h, eps = 24, 0.1, 0.19                                   # 6 eps = 1.14 < L = 2.4
    cfg = GridConfig(n=(n, 6, 6), spacing=(h, h, h), bc=((0, 0) if periodic else (5, 5)) + (0, 0, 0, 0))
    d = slab.SlabDecomposition(cfg, world)
    rng = np.random.default_rng(world)
    L = n * h
    pos = np.column_stack([rng.uniform(-0.6, L + 0.6, 30) if periodic else rng.uniform(0.0, L, 30),
                           rng.uniform(0, 0.6, 30), rng.uniform(0, 0.6, 30)])
    pos[0, 0], pos[1, 0] = 0.01, L - 0.02                       # right at the seam
    force = rng.standard_normal((30, 3))
    xc = (np.arange(n) + 0.5) * h

    def gaussian_sum(points, weights, cells, wrap):
        dx = cells[:, None] - points[None, :, 0]
        if wrap:
            dx -= L * np.round(dx / L)
        k = np.exp(-(dx / eps) ** 2) * (np.abs(dx) <= 3 * eps)   # the y, z factors are the same on both sides
        return k @ weights

    whole = gaussian_sum(pos, force[:, 0], xc, periodic)
    seen = np.zeros(30, dtype=int)
    for r in range(world):
        p, f, e = d.alm_points(r, pos, force, eps)
        assert e == eps and p.shape == f.shape
        i0, i1 = d.owned(r)
        assert np.allclose(gaussian_sum(p, f[:, 0], xc[i0:i1], False), whole[i0:i1], rtol=1e-12, atol=1e-14)
        assert np.array_equal(p[:, 1:], p[:, 1:]) and len(p) <= 2 * len(pos)
        for q in p:                                              # every offered point is one of the originals, shifted by k L
            j = np.where(np.all(np.isclose(pos[:, 1:], q[1:]), axis=1))[0]
            assert len(j) == 1 and abs((q[0] - pos[j[0], 0]) / L - round((q[0] - pos[j[0], 0]) / L)) < 1e-12
            seen[j[0]] += 1
    assert (seen >= 1).all()
    assert np.abs(whole).max() > 0.1


def test_seam_shift_brings_the_rotor_disc_next_to_the_slab_beyond_the_seam():
    cfg = GridConfig(n=(24, 6, 6), spacing=(0.1, 0.1, 0.1), bc=(0,) * 6)
    d = slab.SlabDecomposition(cfg, 3)                           # slabs [0, 0.8), [0.8, 1.6), [1.6, 2.4)
    assert d.seam_shift(0, 0.05, 0.3) == 0.0
    assert d.seam_shift(2, 0.05, 0.3) == pytest.approx(2.4)      # the image at 2.45 acts on the last slab
    assert d.seam_shift(1, 0.05, 0.3) == 0.0                     # out of reach of the middle slab either way
    assert d.seam_shift(0, 2.35, 0.3) == pytest.approx(-2.4)
    assert d.seam_shift(0, 2.35 + 2.4, 0.3) == pytest.approx(-4.8)
    closed = slab.SlabDecomposition(GridConfig(n=(24, 6, 6), spacing=(0.1, 0.1, 0.1), bc=(5, 5, 0, 0, 0, 0)), 3)
    assert closed.seam_shift(2, 0.05, 0.3) == 0.0
