"""The x-slab path as it runs on several GPUs, with the real library in every process: W ranks are
launched with torch.distributed.run, each owns one sub-domain (`Gks` on cuda:0 - the box has one GPU, the ranks share
it), halos move through `slab.DistTransport` over gloo (host-staged buffers).  This exercises what LocalTransport
cannot: message order and matching between processes (two slabs on a periodic axis have the same neighbour on both
sides), the scalar all-reduce of the bulk-flux sum, the all-reduce MAX of the IBM stop rule, the rotor broadcast -
and would hang on the deadlocks NCCL would hit too.  The gathered result equals the single-domain run."""
import os
import subprocess
import sys

import numpy as np
import pytest

from conftest import rel_linf
from slab_worker import case_setup

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
STEPS = 2


def single_domain(case):
    from paper_2603_11102_b200 import gks
    w, passes, rotor = case_setup(case)
    g = gks.Gks(w.cfg)
    if w.ibm is not None:
        g.ibm_set_points(*w.ibm)
        if passes > 1:
            g.ibm_set_iterations(passes, 0.0)
    if w.bulk_flux is not None:
        g.set_bulk_flux(*w.bulk_flux)
    g.set_state(w.W0)
    if rotor is not None:
        g.alm_set_rotor(rotor)
    for k in range(STEPS):
        if w.alm is not None and rotor is None:
            g.alm_set_points(*w.alm(k))
        g.step(w.dt)
    W = g.get_state()
    g.close()
    return W


@pytest.mark.parametrize("case,world,mode", [("taylor_green", 2, "plain"), ("taylor_green", 3, "plain"),
                                             ("cylinder", 2, "plain"), ("cylinder_passes", 3, "plain"),
                                             ("channel", 2, "plain"), ("turbine", 3, "plain"), ("rotor_online", 4, "plain"),
                                             ("cylinder_full", 2, "overlap"), ("taylor_green", 2, "overlap"),
                                             ("taylor_green", 2, "push"), ("taylor_green", 3, "push"),
                                             ("cylinder_passes", 3, "push"), ("channel", 2, "push"),
                                             ("rotor_online", 4, "push"), ("turbine", 3, "push"),
                                             ("taylor_green", 3, "push-delay"), ("cylinder_passes", 2, "push-delay"),
                                             ("cylinder_full", 2, "push-overlap"), ("taylor_green", 2, "push-overlap"),
                                             ("taylor_green", 2, "push-fused"), ("turbine", 3, "push-fused"),
                                             ("cylinder_passes", 3, "push-fused-delay"), ("rotor_online", 4, "push-fused")])
def test_ranks_with_the_real_library_reproduce_the_single_domain(case, world, mode, tmp_path):
    """mode "overlap": the step in parts (slab.SlabStepper.step(overlap=True)): messages are posted before the interior
    is swept and completed before the rim; mode "push": no buffers, no messages - every rank writes its boundary planes
    into the ghost layers of its neighbour PROCESSES through CUDA IPC mappings, ordered by interprocess events
    (slab.IpcPushTransport), in every exchange of the step; "push-delay": the same with one rank's stream held back by
    30 ms in every step (another rank each step), so that its pushes land late and its ghosts stay in use late: the
    hosts run ahead, only the events order the GPUs; "push-overlap": the step in parts with the pushes enqueued ahead of
    the interior sweeps; "push-fused": the exchange of W* is part of the stage-1 update kernel (gks_step_begin_push writes
    into the neighbour process's ghost layers as it computes), only the order is exchanged"""
    port = 29650 + (hash((case, world, mode)) % 200)
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(world),
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.join(ROOT, "tests", "slab_worker.py"),
           case, str(STEPS), str(tmp_path), mode]
    r = subprocess.run(cmd, capture_output=True, text=True, timeout=600, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    Ws = np.concatenate([np.load(os.path.join(tmp_path, "part%d.npy" % k)) for k in range(world)], axis=-1)
    W1 = single_domain(case)
    assert Ws.shape == W1.shape
    # the arithmetic of a cell does not depend on the slab it sits in; what differs: the warp-uniform choice of the
    # erf / exp series length and the order of fp64 atomics
    assert rel_linf(Ws, W1) <= 1e-13, (case, world)
