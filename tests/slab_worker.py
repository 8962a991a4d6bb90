"""One rank of a multi-process x-slab run of the REAL library (launched by tests/test_gpu_slab_multiprocess.py through
torch.distributed.run): its own `Gks` context on cuda:0, `slab.DistTransport` over gloo with host-staged halo
buffers, the scalar all-reduces (bulk flux, IBM stop rule) and the rotor broadcast.  Every rank shares the one GPU of
the box; the ranks synchronise on the host between kernels (gloo), no kernel waits on another process.

    python -m torch.distributed.run --nproc-per-node W tests/slab_worker.py CASE STEPS OUTDIR [overlap | push]

"push": no halo buffers and no messages - `slab.IpcPushTransport` maps the neighbours' workspaces with CUDA IPC and every
rank writes its boundary planes into its neighbours' ghost layers, ordered by interprocess events.
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def case_setup(name):
    """(workload, ibm passes, rotor or None) of a named case; shared with the parent test"""
    from paper_2603_11102_b200 import workloads as wl
    if name == "taylor_green":
        return wl.by_name("C1"), 1, None
    if name == "cylinder_full":                 # 256 x 128 x 64: slabs wide enough to have an interior (overlapped step)
        return wl.by_name("C3"), 1, None
    if name == "channel":                       # bulk-flux forcing: one scalar all-reduce per step
        return wl.by_name("C2", small=True), 1, None
    if name == "cylinder":                      # IBM body cut through by a slab boundary
        return wl.by_name("C3", small=True), 1, None
    if name == "cylinder_passes":               # + the common stop decision (all-reduce MAX) of the IBM passes
        return wl.by_name("C3", small=True), 3, None
    if name == "turbine":                       # prescribed rotating ALM points + IBM nacelle and tower
        return wl.by_name("C5", small=True), 1, None
    if name == "rotor_online":                  # on-line rotor: evaluated by the owner of the disc, broadcast
        w = wl.by_name("C4", small=True)
        pos0, _, eps = w.alm(0)
        hub = pos0.reshape(3, -1, 3).mean(axis=(0, 1))
        r = wl.synthetic_rotor(hub=hub, R=float(np.linalg.norm(pos0 - hub, axis=1).max() * 64.5 / 64.0), eps=eps,
                               npts=40, freestream_correction=True, tip_correction=True)
        return w, 1, r
    raise KeyError(name)


def main():
    import torch
    import torch.distributed as dist
    from paper_2603_11102_b200 import gks, slab
    case, steps, outdir = sys.argv[1], int(sys.argv[2]), sys.argv[3]
    overlap = len(sys.argv) > 4 and sys.argv[4] in ("overlap", "push-overlap")
    push = len(sys.argv) > 4 and sys.argv[4].startswith("push")   # halos written straight into the neighbour PROCESS's ghosts
    fused = len(sys.argv) > 4 and sys.argv[4].startswith("push-fused")   # W* travels inside the stage-1 update kernel
    delay = len(sys.argv) > 4 and sys.argv[4] in ("push-delay", "push-fused-delay")     # one rank's GPU work runs late: only the interprocess
                                                                  # events keep its neighbours from reading stale ghosts
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group("gloo")
    rank, world = dist.get_rank(), dist.get_world_size()
    w, passes, rotor = case_setup(case)
    d = slab.SlabDecomposition(w.cfg, world)
    g = gks.Gks(d.local_cfg(rank), device="cuda:0")
    if w.ibm is not None:
        g.ibm_set_points(*d.ibm_points(rank, *w.ibm))
        if passes > 1:
            g.ibm_set_iterations(passes, 0.0)
    if w.bulk_flux is not None:
        g.set_bulk_flux(*w.bulk_flux)
    g.set_state(d.scatter(w.W0, rank))
    transport = slab.IpcPushTransport(d, rank, g) if push else slab.DistTransport(d, rank)
    stepper = slab.SlabStepper(transport, g, slab.BufferPool("cpu"))
    rot = slab.RotorDriver(d, rotor, "cpu") if rotor is not None else None
    for k in range(steps):
        if delay and rank == k % world:
            with torch.cuda.stream(g.stream):
                torch.cuda._sleep(60_000_000)       # about 30 ms of GPU time ahead of this rank's pushes and sweeps
        hook = None
        if w.alm is not None and rotor is None:
            pts = d.alm_points(rank, *w.alm(k))
            hook = lambda s, pts=pts: s.alm_set_points(*pts)
        stepper.step(w.dt, before_forcing=hook, ibm=w.ibm is not None, rotor=rot, bulk=w.bulk_flux is not None,
                     ibm_passes=passes, overlap=overlap, push=("fused" if fused else push))
    if push:
        transport.close()
    np.save(os.path.join(outdir, "part%d.npy" % rank), g.get_state())
    launches = g.launch_count
    g.close()
    dist.barrier()
    dist.destroy_process_group()
    assert launches > 0


if __name__ == "__main__":
    main()
