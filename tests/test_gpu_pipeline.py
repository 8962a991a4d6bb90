"""gks.HostPipeline: independent batches with host buffers through two or three contexts in rotation (the end-to-end
path of bench.py) give, batch for batch, the result of one context that does copy in, step, copy out in sequence."""
import numpy as np
import pytest

from conftest import rel_linf
from paper_2603_11102_b200 import workloads as wl

pytestmark = pytest.mark.gpu


def _setup_for(w):
    def setup(g):
        if w.bulk_flux is not None:
            g.set_bulk_flux(*w.bulk_flux)
        if w.ibm is not None:
            g.ibm_set_points(*w.ibm)
    return setup


@pytest.mark.parametrize("name,depth,steps", [("C1", 2, 1), ("C3", 2, 2), ("C2", 3, 1), ("C5", 2, 1)])
def test_pipelined_batches_equal_the_serial_path(name, depth, steps):
    import torch
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=(name != "C1"))
    rng = np.random.default_rng(20260402)
    nb = 5
    ins = [torch.from_numpy(w.W0 * (1.0 + 0.01 * rng.standard_normal(w.W0.shape))).pin_memory() for _ in range(nb)]
    outs = [torch.full(ins[0].shape, float("nan"), dtype=torch.float64).pin_memory() for _ in range(nb)]
    hook = (lambda g, s: g.alm_set_points(*w.alm(s))) if w.alm is not None else None
    # serial reference: one context
    g = gks.Gks(w.cfg)
    _setup_for(w)(g)
    ref = []
    for b in range(nb):
        g.set_state(ins[b])
        for s in range(steps):
            if hook is not None:
                hook(g, s)
            g.step(w.dt)
        ref.append(g.get_state())
    g.close()
    pipe = gks.HostPipeline(w.cfg, depth=depth, setup=_setup_for(w))
    done = []
    for b in range(nb):
        r = pipe.submit(ins[b], outs[b], w.dt, steps=steps, before_step=hook)
        if b < depth - 1:
            assert r is None
        else:
            assert r is outs[b - depth + 1]
            done.append(r)
    done += pipe.drain()
    assert len(done) == nb and all(d is o for d, o in zip(done, outs))
    assert pipe.launch_count > 0
    pipe.close()
    for b in range(nb):
        if w.ibm is None:
            assert np.array_equal(outs[b].numpy(), ref[b]), b
        else:                                   # the IBM spreading adds with fp64 atomics: order varies run to run
            assert rel_linf(outs[b].numpy(), ref[b]) <= 1e-13, b
        assert not np.array_equal(ref[b], ref[(b + 1) % nb])        # the batches differ


@pytest.mark.parametrize("name", ["C1", "C2", "C3"])
def test_a_step_can_be_captured_in_a_cuda_graph(name):
    """gks_step allocates nothing, never synchronises and reads no host memory, so a caller may capture it (stream
    capture on the context's stream, programmatic dependent launches included) and replay it: same bits as the plain
    calls where the step is deterministic, 1e-13 with the fp64 atomics of the IBM spreading"""
    import torch
    from paper_2603_11102_b200 import gks
    w = wl.by_name(name, small=(name != "C1"))
    g = gks.Gks(w.cfg)
    _setup_for(w)(g)
    g.set_state(w.W0)
    for _ in range(4):
        g.step(w.dt)
    ref = g.get_state()
    g.set_state(w.W0)
    g.step(w.dt)                      # every kernel has run once before the capture
    g.synchronize()
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=g.stream):
        g.step(w.dt)                  # captured, not executed
    with torch.cuda.stream(g.stream):
        for _ in range(3):
            graph.replay()
    out = g.get_state()
    g.close()
    if w.ibm is None:
        assert np.array_equal(out, ref)
    else:
        assert rel_linf(out, ref) <= 1e-13
