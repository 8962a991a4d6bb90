"""x-slab domain decomposition of the S2O4 GKS step over several GPUs ("the computational
domain is divided along the x-direction ... the ghost cells are exchanged between neighbouring GPUs").

Rank r owns the cells i in [x_lo[r], x_lo[r+1]) of the global grid; its sub-domain is an ordinary `gks.Gks`
context whose cut faces carry GKS_BC_HALO.  Per step the 3 ghost planes x 4 fields of each cut face move
twice: the state W^n before `step_begin`, the first-stage state W* before `step_finish`
(include/gks.h, "Domain decomposition").  Actuator points are given to every rank whose cells their support
reaches (`SlabDecomposition.alm_points`; images beyond the seam of a periodic x axis included): the Gaussian
gather of a rank only adds to the cells it owns, so a support that straddles a cut needs no exchange.

This module holds host logic only (who owns what, who talks to whom, in which order); every number is moved by
`gks_halo_pack` / `gks_halo_unpack` kernels and by the transport:
  * `LocalTransport`  - all sub-domains live in ONE process (one GPU): buffers are handed over directly.  This
    is how the decomposition is validated on a single-GPU box (no kernels wait on one another);
  * `DistTransport`   - one process per GPU, `torch.distributed` point-to-point (NCCL on device tensors; gloo on
    CPU tensors in the CPU tests of the plumbing).
IBM points within 1.5 cells of a cut are given to both sub-domains (`SlabDecomposition.ibm_points`); both
interpolate the same U_p after a third exchange (the un-forced W^{n+1}) and each adds to the cells it owns.
The on-line rotor is evaluated by the sub-domain that contains the disc and broadcast (`RotorDriver`).
The bulk-flux forcing adds the sub-domains' partial sums up with one scalar all-reduce; IBM passes > 1 exchange
the halo between the passes and take the MAX of the sub-domains' slips for the common stop decision.
"""
from dataclasses import replace

import numpy as np

BC_PERIODIC, BC_HALO = 0, 6
XLO, XHI = 0, 1


class SlabDecomposition:
    """Who owns which x-range of a global GridConfig, and the sub-domain configuration of every rank."""

    def __init__(self, cfg, world):
        if cfg.faces[0] is not None:
            raise ValueError("x-slabs need a uniform x axis")
        if world < 1 or cfg.n[0] // world < 6:
            raise ValueError("every slab needs at least 6 cells along x")
        self.cfg, self.world = cfg, world
        base, extra = divmod(cfg.n[0], world)
        sizes = [base + (1 if r < extra else 0) for r in range(world)]
        self.x_lo = np.concatenate([[0], np.cumsum(sizes)]).astype(int)
        self.periodic = cfg.bc[0] == BC_PERIODIC

    def owned(self, rank):
        return int(self.x_lo[rank]), int(self.x_lo[rank + 1])

    def neighbours(self, rank):
        """(rank on the low-x side, rank on the high-x side); None at a physical boundary"""
        if self.world == 1:
            return None, None
        lo = rank - 1 if rank > 0 else (self.world - 1 if self.periodic else None)
        hi = rank + 1 if rank < self.world - 1 else (0 if self.periodic else None)
        return lo, hi

    def local_cfg(self, rank):
        i0, i1 = self.owned(rank)
        lo, hi = self.neighbours(rank)
        bc = list(self.cfg.bc)
        if self.world > 1:
            bc[0] = BC_HALO if lo is not None else self.cfg.bc[0]
            bc[1] = BC_HALO if hi is not None else self.cfg.bc[1]
        origin = (self.cfg.origin[0] + i0 * self.cfg.spacing[0], self.cfg.origin[1], self.cfg.origin[2])
        return replace(self.cfg, n=(i1 - i0, self.cfg.n[1], self.cfg.n[2]), origin=origin, bc=tuple(bc))

    def scatter(self, W, rank):
        i0, i1 = self.owned(rank)
        return np.ascontiguousarray(W[..., i0:i1])

    def gather(self, parts):
        return np.concatenate(parts, axis=-1)

    def ibm_select(self, rank, pos):
        """(indices into the global point list, x shifts) of the Lagrangian points sub-domain `rank` must know:
        those inside it and those of a neighbour whose 3-point support (1.5 cells) reaches across a cut.  On a
        periodic x axis the images beyond the seam are shifted by the period so that they sit next to the slab.
        Per-point data of the global list (volumes, velocities) are taken with the same indices."""
        i0, i1 = self.owned(rank)
        h, x0 = self.cfg.spacing[0], self.cfg.origin[0]
        lo, hi = self.neighbours(rank)
        a = x0 + i0 * h - (1.5 * h if lo is not None else 0.0)
        b = x0 + i1 * h + (1.5 * h if hi is not None else 0.0)
        L = self.cfg.n[0] * h
        idx, shifts = [], []
        for shift in ((0.0, -L, L) if (self.periodic and self.world > 1) else (0.0,)):
            x = pos[:, 0] + shift
            m = (x >= a) & (x <= b)
            if shift != 0.0:                      # images only where they are NOT already inside the slab proper
                m &= (x < x0 + i0 * h) | (x > x0 + i1 * h)
            k = np.nonzero(m)[0]
            idx.append(k)
            shifts.append(np.full(len(k), shift))
        return np.concatenate(idx), np.concatenate(shifts)

    def ibm_points(self, rank, pos, vol):
        """(positions, volumes) of the Lagrangian points of `ibm_select(rank, pos)`"""
        idx, shifts = self.ibm_select(rank, pos)
        q = pos[idx].copy()
        q[:, 0] += shifts
        return q, vol[idx]

    def ibm_velocities(self, rank, pos, vel):
        """the velocities v_p of the same points, in the same order (gks `ibm_set_velocities`)"""
        idx, _ = self.ibm_select(rank, pos)
        return np.ascontiguousarray(np.asarray(vel, dtype=np.float64)[idx])

    def alm_points(self, rank, pos, force, eps):
        """Actuator points sub-domain `rank` must know: those whose Gaussian support (3 eps) reaches the cells it owns.
        A sub-domain's cut faces are not periodic, so on a periodic x axis a point acts on a slab beyond the seam
        through its image: positions are wrapped into the period and the images one period below and above are
        offered too (6 eps < period: a cell sees one image of a point at most)."""
        pos, force = np.asarray(pos, dtype=np.float64), np.asarray(force, dtype=np.float64)
        i0, i1 = self.owned(rank)
        h, x0 = self.cfg.spacing[0], self.cfg.origin[0]
        a, b = x0 + i0 * h - 3.0 * eps, x0 + i1 * h + 3.0 * eps
        L = self.cfg.n[0] * h
        wrap = self.periodic and self.world > 1
        x = x0 + np.mod(pos[:, 0] - x0, L) if wrap else pos[:, 0]
        out_p, out_f = [], []
        for shift in ((0.0, -L, L) if wrap else (0.0,)):
            m = (x + shift >= a) & (x + shift <= b)
            q = pos[m].copy()
            q[:, 0] = x[m] + shift
            out_p.append(q)
            out_f.append(force[m])
        return np.concatenate(out_p), np.concatenate(out_f), eps

    def seam_shift(self, rank, x, reach):
        """the multiple of the period that brings the plane x within `reach` of sub-domain `rank` (0.0 if it already
        is, or if x is not periodic, or if no image is)"""
        if not (self.periodic and self.world > 1):
            return 0.0
        i0, i1 = self.owned(rank)
        h, x0 = self.cfg.spacing[0], self.cfg.origin[0]
        L = self.cfg.n[0] * h
        xw = x0 + np.mod(x - x0, L)
        for shift in (0.0, -L, L):
            if x0 + i0 * h - reach <= xw + shift <= x0 + i1 * h + reach:
                return float(xw + shift - x)
        return 0.0

    def schedule(self, rank):
        """The exchange of one halo, as a list of (face to pack, destination rank, face the destination unpacks).
        Message tags are (sender's packed face), unique per (sender, receiver) pair even when world == 2 and
        periodic (the same neighbour on both sides)."""
        lo, hi = self.neighbours(rank)
        out = []
        if lo is not None:
            out.append((XLO, lo, XHI))
        if hi is not None:
            out.append((XHI, hi, XLO))
        return out


class LocalTransport:
    """All sub-domains in this process: `exchange` hands every packed buffer to the solver that unpacks it."""

    def __init__(self, decomposition):
        self.d = decomposition

    def exchange(self, solvers, which, new_buffer):
        packed = {}
        for s in solvers:                         # persistent buffers: the previous unpacks have finished
            s.synchronize()
        for r, s in enumerate(solvers):
            for face, dst, dst_face in self.d.schedule(r):
                buf = new_buffer(s, face, "send")
                s.halo_pack(which, face, buf)
                packed[(dst, dst_face)] = buf
        for s in solvers:                         # every solver has its own stream: packs before unpacks
            s.synchronize()
        for (dst, dst_face), buf in packed.items():
            solvers[dst].halo_unpack(which, dst_face, buf)


    def exchange_push(self, solvers, which):
        """the exchange without buffers: every sub-domain writes its boundary planes straight into its neighbours'
        ghost layers (gks_halo_push: pack, transfer and unpack in one kernel; peer-to-peer stores when the
        neighbour's window lives on another GPU).  Streams are ordered on the host here; a multi-GPU driver would
        record an event behind the push and let the neighbour's stream wait for it."""
        for s in solvers:                         # the neighbours have finished reading the ghosts we overwrite
            s.synchronize()
        for r, s in enumerate(solvers):
            for face, dst, dst_face in self.d.schedule(r):
                s.halo_push(which, face, solvers[dst].halo_window(which))
        for s in solvers:
            s.synchronize()

    def step_begin_push(self, solvers, dt):
        """stage 1 with the exchange of W* fused into its update kernel (gks_step_begin_push): every sub-domain's
        update also writes its boundary planes of W* into its neighbours' ghost layers"""
        for s in solvers:                         # the neighbours' W* ghosts are free (their previous stage 2 has run)
            s.synchronize()
        for r, s in enumerate(solvers):
            to = {face: solvers[dst].halo_window(1) for face, dst, dst_face in self.d.schedule(r)}
            s.step_begin_push(dt, to.get(XLO), to.get(XHI))

    def exchange_landed(self, solvers):
        for s in solvers:                         # every update (and with it every push) has run
            s.synchronize()

    # the same exchange in two halves, for the overlapped step (nothing overlaps inside one process: the hand-over
    # is a pointer; the split is what is exercised)
    def exchange_begin(self, solvers, which, new_buffer):
        for s in solvers:
            s.synchronize()
        self._packed = {}
        for r, s in enumerate(solvers):
            for face, dst, dst_face in self.d.schedule(r):
                buf = new_buffer(s, face, "send")
                s.halo_pack(which, face, buf)
                self._packed[(dst, dst_face)] = buf

    def exchange_end(self, solvers, which, new_buffer):
        for s in solvers:
            s.synchronize()
        for (dst, dst_face), buf in self._packed.items():
            solvers[dst].halo_unpack(which, dst_face, buf)
        self._packed = {}


class DistTransport:
    """One process per sub-domain; point-to-point messages through torch.distributed (nccl or gloo)."""

    def __init__(self, decomposition, rank, group=None):
        import torch.distributed as dist
        self.d, self.rank, self.dist, self.group = decomposition, rank, dist, group

    def exchange(self, solver, which, new_buffer):
        import contextlib
        import torch
        dist = self.dist
        sched = self.d.schedule(self.rank)
        recvs, ops = [], []
        cuda = False
        for face, dst, dst_face in sched:                       # sends in the order of the packed face
            sbuf = new_buffer(solver, face, "send")
            cuda = cuda or sbuf.is_cuda
            solver.halo_pack(which, face, sbuf)
            ops.append(dist.P2POp(dist.isend, sbuf, dst, group=self.group, tag=face))
        # what arrives for my face `face` was packed by `dst` at its face `dst_face`.  NCCL matches the messages
        # of a pair of ranks by order, not by tag: receives are posted in the order of the SENDER's packed face
        # (this matters when both neighbours are the same rank: two slabs on a periodic axis)
        for face, dst, dst_face in sorted(sched, key=lambda e: e[2]):
            rbuf = new_buffer(solver, face, "recv")
            recvs.append((face, rbuf))
            ops.append(dist.P2POp(dist.irecv, rbuf, dst, group=self.group, tag=dst_face))
        if ops:
            # device buffers (NCCL): issue on the solver's stream, so that the packs before and the unpacks after
            # are ordered with the transfers without a host synchronisation; host buffers (gloo): the packs have
            # synchronised already
            with (torch.cuda.stream(solver.stream) if cuda else contextlib.nullcontext()):
                for req in dist.batch_isend_irecv(ops):
                    req.wait()
        for face, rbuf in recvs:
            solver.halo_unpack(which, face, rbuf)

    def exchange_begin(self, solver, which, new_buffer):
        """pack the halos of state `which` and post the messages; returns at once.  Device buffers (NCCL): the
        messages travel on a communication stream of their own, ordered behind the packs by an event, so the kernels
        the solver enqueues next (part 0 of a stage: everything that reads no HALO ghost) run beside the transfer."""
        import torch
        dist = self.dist
        sched = self.d.schedule(self.rank)
        ops, self._recvs, cuda = [], [], False
        for face, dst, dst_face in sched:
            sbuf = new_buffer(solver, face, "send")
            cuda = cuda or sbuf.is_cuda
            solver.halo_pack(which, face, sbuf)
            ops.append(dist.P2POp(dist.isend, sbuf, dst, group=self.group, tag=face))
        for face, dst, dst_face in sorted(sched, key=lambda e: e[2]):      # receives in the SENDER's order (see exchange)
            rbuf = new_buffer(solver, face, "recv")
            self._recvs.append((face, rbuf))
            ops.append(dist.P2POp(dist.irecv, rbuf, dst, group=self.group, tag=dst_face))
        self._reqs, self._comm = [], None
        if ops:
            if cuda:
                if getattr(self, "_comm_stream", None) is None:
                    self._comm_stream = torch.cuda.Stream(device=solver.device)
                self._comm = self._comm_stream
                self._comm.wait_stream(solver.stream)                        # behind the packs
                with torch.cuda.stream(self._comm):
                    self._reqs = dist.batch_isend_irecv(ops)
            else:
                self._reqs = dist.batch_isend_irecv(ops)                     # gloo: the packs have synchronised

    def exchange_end(self, solver, which, new_buffer):
        """complete the messages posted by exchange_begin and unpack them into the HALO ghosts"""
        import torch
        if self._comm is not None:
            with torch.cuda.stream(self._comm):
                for req in self._reqs:
                    req.wait()
            solver.stream.wait_stream(self._comm)                            # the unpacks behind the transfer
        else:
            for req in self._reqs:
                req.wait()
        for face, rbuf in self._recvs:
            solver.halo_unpack(which, face, rbuf)
        self._reqs, self._recvs = [], []

    def all_reduce_sum(self, solver, scalar, volume):
        """(sum over ranks of a 1-element tensor, sum of the host number `volume`)"""
        import contextlib
        import torch
        # on the solver's stream throughout: `scalar` was written there (gks_bulk_partial) and torch's current
        # stream is not ordered against it
        with (torch.cuda.stream(solver.stream) if scalar.is_cuda else contextlib.nullcontext()):
            pair = torch.stack([scalar.reshape(()), torch.tensor(volume, dtype=torch.float64).to(scalar.device)])
            self.dist.all_reduce(pair, group=self.group)
            total = pair[:1].contiguous()
        if scalar.is_cuda:
            solver.synchronize()
        return total, float(pair[1])

    def all_reduce_max(self, solver, scalar):
        import contextlib
        import torch
        with (torch.cuda.stream(solver.stream) if scalar.is_cuda else contextlib.nullcontext()):
            self.dist.all_reduce(scalar, op=self.dist.ReduceOp.MAX, group=self.group)
        return scalar

    def broadcast(self, solver, src, tensors):
        import contextlib
        import torch
        with (torch.cuda.stream(solver.stream) if tensors[0].is_cuda else contextlib.nullcontext()):
            for t in tensors:
                self.dist.broadcast(t, src=src, group=self.group)



class IpcPushTransport(DistTransport):
    """One process per sub-domain, halos WITHOUT buffers and without messages: every rank maps the workspaces of its
    neighbours (CUDA IPC: gks_halo_export_get / _open - peer-to-peer over NVLink when the neighbour sits on another GPU)
    and writes its boundary planes straight into their ghost layers (gks_halo_push: pack, transfer and unpack in one
    kernel).  Nothing but the order travels between the processes:

        ghosts_free[r]  interprocess event, recorded on r's stream when r calls the exchange: everything r enqueued before
                        (the sweeps that read its ghosts) precedes it; a neighbour's stream waits for it before it pushes
        landed[r]       recorded on r's stream behind its pushes; a neighbour's stream waits for it before it goes on

    A stream that waits for an interprocess event waits for the LAST record the host has issued, so the waiting host must
    know that the record has been issued: one host barrier of the control group (gloo: no device work, no stream is
    synchronised) between a record and the waits for it.  Per exchange: record, barrier, waits + pushes + record,
    barrier, waits - the GPUs never idle for the host as long as the hosts run ahead of them.  No KERNEL waits for
    another rank (the waits are the stream's, cudaStreamWaitEvent), so the ranks may also share one GPU.

    Every exchange of the step goes this way (both stages, the un-forced W^{n+1} for IBM / rotor, between IBM passes);
    the scalar reductions and the rotor broadcast stay DistTransport's."""

    def __init__(self, decomposition, rank, solver, group=None, control_group=None):
        import torch
        from . import gks
        super().__init__(decomposition, rank, group)
        dist = self.dist
        if decomposition.world < 2:
            raise ValueError("IpcPushTransport needs at least two sub-domains")
        # control plane: host-only barriers and the one-off exchange of handles
        self.control = control_group if control_group is not None else (
            group if dist.get_backend(group) == "gloo" else dist.new_group(backend="gloo"))
        self.solver = solver
        self.ev_free = torch.cuda.Event(interprocess=True)
        self.ev_landed = torch.cuda.Event(interprocess=True)
        with torch.cuda.device(solver.device):
            self.ev_free.record(solver.stream)          # an event has an IPC handle once it exists on the device
            self.ev_landed.record(solver.stream)
            mine = (solver.halo_export(), self.ev_free.ipc_handle(), self.ev_landed.ipc_handle())
        everyone = [None] * decomposition.world
        dist.all_gather_object(everyone, mine, group=self.control)
        self.win, self.peer_free, self.peer_landed, self._maps = {}, {}, {}, []
        for n in sorted({dst for _, dst, _ in decomposition.schedule(rank)}):
            blob, h_free, h_landed = everyone[n]
            wins, m = gks.halo_export_open(blob, solver.device)        # once per neighbour RANK
            self.win[n] = wins
            self._maps.append(m)
            self.peer_free[n] = torch.cuda.Event.from_ipc_handle(solver.device, h_free)
            self.peer_landed[n] = torch.cuda.Event.from_ipc_handle(solver.device, h_landed)

    def exchange_push(self, solver, which):
        st = solver.stream
        self.ev_free.record(st)                          # my ghosts may be overwritten once this has passed
        self.dist.barrier(group=self.control)            # every neighbour's record has been issued
        for ev in self.peer_free.values():
            st.wait_event(ev)
        for face, dst, dst_face in self.d.schedule(self.rank):
            solver.halo_push(which, face, self.win[dst][which])
        self.ev_landed.record(st)
        self.dist.barrier(group=self.control)
        for ev in self.peer_landed.values():             # the neighbours' planes are in my ghosts
            st.wait_event(ev)

    def exchange(self, solver, which, new_buffer=None):
        self.exchange_push(solver, which)

    def step_begin_push(self, solver, dt):
        """stage 1 with the exchange of W* fused into its update kernel.  The neighbours' W* ghosts are free: they
        were last read by the neighbours' second stage of the step before, which precedes their `landed` of this
        step's first exchange - and this stream has waited for that."""
        to = {face: self.win[dst][1] for face, dst, dst_face in self.d.schedule(self.rank)}
        solver.step_begin_push(dt, to.get(XLO), to.get(XHI))

    def exchange_landed(self, solver):
        """what is left of the second exchange: the order"""
        self.ev_landed.record(solver.stream)
        self.dist.barrier(group=self.control)
        for ev in self.peer_landed.values():
            solver.stream.wait_event(ev)

    # the same in two halves for the step in parts (SlabStepper.step(overlap=True)): the pushes are enqueued ahead of
    # the interior sweeps, which read no HALO ghost; the rim waits for the neighbours' `landed` - recorded at the START
    # of their stage, so it has long passed when the interior is done
    def exchange_begin(self, solver, which, new_buffer=None):
        st = solver.stream
        self.ev_free.record(st)
        self.dist.barrier(group=self.control)
        for ev in self.peer_free.values():
            st.wait_event(ev)
        for face, dst, dst_face in self.d.schedule(self.rank):
            solver.halo_push(which, face, self.win[dst][which])
        self.ev_landed.record(st)

    def exchange_end(self, solver, which, new_buffer=None):
        self.dist.barrier(group=self.control)
        for ev in self.peer_landed.values():
            solver.stream.wait_event(ev)

    def close(self):
        """unmap the neighbours' workspaces (before they are freed): every stream idle, then a barrier"""
        from . import gks
        self.solver.synchronize()
        self.dist.barrier(group=self.control)
        for m in self._maps:
            gks.halo_export_close(m)
        self._maps = []
        self.dist.barrier(group=self.control)

class RotorDriver:
    """The on-line actuator-line rotor on sub-domains: every sub-domain is given the rotor with `alm_set_rotor` and
    keeps its clock in the library (advanced by dt in every `gks_step_force`); the disc x = hub_x lies in ONE slab
    (its owner), which evaluates the blade-element forces of all points from the un-forced field with
    `alm_rotor_eval` (trilinear sampling reads the first HALO ghost layer when the disc sits within half a cell of a
    cut); the (tiny) position and force arrays are broadcast and handed to every sub-domain with `alm_rotor_supply`,
    which spreads them onto the cells it owns."""

    def __init__(self, decomposition, rotor, device):
        import torch
        self.d, self.r = decomposition, rotor
        i = int(np.floor((rotor.hub[0] - decomposition.cfg.origin[0]) / decomposition.cfg.spacing[0]))
        i = min(max(i, 0), decomposition.cfg.n[0] - 1)
        self.owner = int(np.searchsorted(decomposition.x_lo, i, side="right") - 1)
        n = rotor.nblades * rotor.npts
        self.pos = torch.zeros((n, 3), dtype=torch.float64, device=device)
        self.force = torch.zeros((n, 3), dtype=torch.float64, device=device)
        if self.pos.is_cuda:
            torch.cuda.synchronize()               # the fills ran on torch's stream, the solvers write on their own
        self._attached = False

    def evaluate(self, transport, solvers, many):
        """between step_finish (+ exchange of the un-forced field) and step_force"""
        sols = solvers if many else [solvers]
        if not self._attached:                     # rotor description and clock (t = 0 now) live in every context
            for s in sols:
                s.alm_set_rotor(self.r)
            self._attached = True
        if many:                                   # all sub-domains in this process: the owner's arrays are everyone's
            solvers[self.owner].alm_rotor_eval(self.pos, self.force)
            solvers[self.owner].synchronize()
            targets = list(enumerate(solvers))
        else:
            if transport.rank == self.owner:
                solvers.alm_rotor_eval(self.pos, self.force)
            transport.broadcast(solvers, self.owner, [self.pos, self.force])
            targets = [(transport.rank, solvers)]
        for rank, s in targets:
            # the disc is a plane x = hub_x: beyond the seam of a periodic x axis a slab meets its image
            s.alm_rotor_supply(self.pos, self.force, self.d.seam_shift(rank, self.r.hub[0], 3.0 * self.r.eps))


class BufferPool:
    """persistent halo buffers, one per (solver, face, role): nothing is allocated inside a step"""

    def __init__(self, device):
        self.device, self.bufs = device, {}

    def __call__(self, solver, face, role):
        import torch
        key = (id(solver), face, role)
        if key not in self.bufs:
            self.bufs[key] = torch.empty(solver.halo_doubles(face), dtype=torch.float64, device=self.device)
        return self.bufs[key]


class SlabStepper:
    """The step of include/gks.h "Domain decomposition" for the sub-domain(s) of this process.

    solvers: the list of all sub-domain solvers (LocalTransport) or the single solver of this rank
    (DistTransport).  new_buffer(solver, face, role) -> a contiguous float64 torch tensor of
    solver.halo_doubles(face) elements on the device the transport moves (CUDA for nccl / local, CPU for gloo);
    role is "send" or "recv" (`BufferPool` keeps one persistent buffer per solver, face and role)."""

    def __init__(self, transport, solvers, new_buffer):
        self.t, self.solvers, self.new_buffer = transport, solvers, new_buffer
        self.many = isinstance(solvers, (list, tuple))
        self._scr, self._keep = {}, []

    def _scratch(self, name, n, dev):
        """n persistent 1-element tensors.  The solvers write and read them on their OWN streams, which are not
        ordered against torch's current stream: a fresh `torch.zeros` per step would race its fill against those
        writes, and a temporary freed at return could be reused while a solver's copy from it is still queued.
        Allocated once, filled once, with a device-wide synchronisation at that point only."""
        import torch
        key = (name, n)
        if key not in self._scr:
            self._scr[key] = [torch.zeros(1, dtype=torch.float64, device=dev) for _ in range(n)]
            if self._scr[key][0].is_cuda:
                torch.cuda.synchronize()
        return self._scr[key]

    def _each(self, fn):
        for s in (self.solvers if self.many else [self.solvers]):
            fn(s)

    def _bulk(self):
        """global sum of the bulk momentum: partial sums of the sub-domains, one scalar all-reduce"""
        import torch
        sols = self.solvers if self.many else [self.solvers]
        dev = self.new_buffer.device if hasattr(self.new_buffer, "device") else "cpu"
        parts = self._scratch("bulk", len(sols), dev)
        vols = [s.bulk_partial(p) for s, p in zip(sols, parts)]
        if self.many:
            for s in sols:
                s.synchronize()
            self._keep.clear()          # every solver stream is idle: nothing reads last step's totals any more
            total, volume = torch.stack(parts).sum(0), float(sum(vols))
            if total.is_cuda:
                torch.cuda.current_stream().synchronize()   # the solvers copy it on their own streams
        else:
            total, volume = self.t.all_reduce_sum(sols[0], parts[0], vols[0])   # synchronises the solver
            self._keep.clear()
        self._keep.append(total)        # the solvers copy from it asynchronously: alive until they were synchronised
        for s in sols:
            s.bulk_set_global(total, volume)

    def _ibm_passes(self, passes):
        """multi-direct-forcing passes on sub-domains: the neighbours' increments travel between the passes and
        the stop decision is common (MAX of the sub-domains' slips)"""
        import torch
        sols = self.solvers if self.many else [self.solvers]
        dev = self.new_buffer.device if hasattr(self.new_buffer, "device") else "cpu"
        for k in range(passes):
            if k > 0:
                self.t.exchange(self.solvers, 0, self.new_buffer)
            for s in sols:
                s.ibm_pass(k, 0)
            if k > 0:
                slips = self._scratch("slip%d" % k, len(sols), dev)
                for s, r in zip(sols, slips):
                    s.ibm_residual(k, r)
                if self.many:
                    for s in sols:
                        s.synchronize()
                    self._keep.clear()          # safe point: every solver stream is idle
                    top = torch.stack(slips).max(0).values
                    if top.is_cuda:
                        torch.cuda.current_stream().synchronize()
                    self._keep.append(top)      # copied by the solvers on their own streams after this returns
                else:
                    top = self.t.all_reduce_max(sols[0], slips[0])
                for s in sols:
                    s.ibm_residual(k, top, set=True)
            for s in sols:
                s.ibm_pass(k, 1)

    def step(self, dt, before_forcing=None, ibm=False, rotor=None, bulk=False, ibm_passes=1, overlap=False, push=False):
        """before_forcing(solver): e.g. alm_set_points for this step (replicated point list);
        ibm: Lagrangian points are set (on any rank): the un-forced W^{n+1} is exchanged before the forcing;
        rotor: a RotorDriver (on-line actuator lines), evaluated on the un-forced W^{n+1} as well;
        bulk: the bulk-flux forcing is set: its global sum is assembled before the forcing;
        ibm_passes: the max_iter given to ibm_set_iterations on every sub-domain, when > 1;
        overlap: the halos of either stage travel while the stage's interior is swept (PAPER.md:193-197 exchanges per
        flux evaluation; include/gks.h gks_step_begin_part): post, part 0, complete, part 1;
        push: (sub-domains that can address one another's memory: LocalTransport, IpcPushTransport) the two stage
        exchanges without buffers, every sub-domain writing into its neighbours' ghost layers (gks_halo_push);
        push="fused": the exchange of W* is part of the stage-1 update kernel itself (gks_step_begin_push)"""
        if before_forcing is not None:
            self._each(before_forcing)
        if overlap:
            self.t.exchange_begin(self.solvers, 0, self.new_buffer)     # ghosts of W^n on their way
            self._each(lambda s: s.step_begin_part(dt, 0))              # interior of stage 1
            self.t.exchange_end(self.solvers, 0, self.new_buffer)
            self._each(lambda s: s.step_begin_part(dt, 1))              # rim of stage 1: W* complete
            self.t.exchange_begin(self.solvers, 1, self.new_buffer)     # ghosts of W* on their way
            self._each(lambda s: s.step_finish_part(dt, 0))
            self.t.exchange_end(self.solvers, 1, self.new_buffer)
            self._each(lambda s: s.step_finish_part(dt, 1))
        elif push == "fused":
            self.t.exchange_push(self.solvers, 0)                  # ghosts of W^n, written by the neighbours
            self.t.step_begin_push(self.solvers, dt)               # the stage update writes the ghosts of W* as well
            self.t.exchange_landed(self.solvers)
            self._each(lambda s: s.step_finish(dt))
        elif push:
            self.t.exchange_push(self.solvers, 0)                  # ghosts of W^n, written by the neighbours
            self._each(lambda s: s.step_begin(dt))
            self.t.exchange_push(self.solvers, 1)                  # ghosts of W*
            self._each(lambda s: s.step_finish(dt))
        else:
            self.t.exchange(self.solvers, 0, self.new_buffer)      # ghosts of W^n
            self._each(lambda s: s.step_begin(dt))
            self.t.exchange(self.solvers, 1, self.new_buffer)      # ghosts of W*
            self._each(lambda s: s.step_finish(dt))
        if ibm or rotor is not None:
            self.t.exchange(self.solvers, 0, self.new_buffer)  # ghosts of the un-forced W^{n+1}
        if rotor is not None:
            rotor.evaluate(self.t, self.solvers, self.many)
        if bulk:
            self._bulk()
        if ibm and ibm_passes > 1:
            self._ibm_passes(ibm_passes)
        self._each(lambda s: s.step_force(dt))
