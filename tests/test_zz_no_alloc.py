"""gks_cfl_dt_noalloc (include/gks.h): the CFL time step for callers that cannot allocate device memory - no context,
no workspace, scratch in a file-scope __device__ array of the library - against the existing path gks_cfl_dt.

Collected last on purpose (file name): the suite runs with pytest -x.  Passes alone in a fresh process and after the
other tests (it touches no state of theirs: its own tensors, torch's current stream)."""
import numpy as np
import pytest

from paper_2603_11102_b200 import workloads as wl

pytestmark = pytest.mark.gpu

REL = 1e-14         # tests/test_gpu_parity.py::test_cfl_dt_matches_the_oracle: max is exact, fma may move the last bit


def _existing(w, W, cfl):
    """the existing path: a context with its workspace, gks_set_state, gks_cfl_dt"""
    from paper_2603_11102_b200 import gks
    g = gks.Gks(w.cfg)
    g.set_state(W)
    dt = g.cfl_dt(cfl)
    g.close()
    return dt


def _noalloc(w, W, cfl, out):
    import torch
    from paper_2603_11102_b200 import gks
    Wd = torch.from_numpy(np.ascontiguousarray(W)).to("cuda:0")
    dmin = min(w.cfg.widths(a).min() for a in range(3))
    gks.cfl_dt_noalloc(Wd, dmin, w.cfg.RT, cfl, out)
    torch.cuda.synchronize()
    return float(out.cpu()[0])


def test_two_calls_in_a_row_match_the_existing_path():
    """first a grid of many blocks with a fast cell in the LAST block, then a smaller, slower state: partial maxima that
    the first call left in the shared scratch array must not reach the second call's result; then the first again"""
    import torch
    out = torch.full((1,), -1.0, dtype=torch.float64, device="cuda:0")
    big = wl.by_name("C2", small=False)          # 128 x 96 x 64 stretched channel: 192 blocks, ragged widths
    Wb = big.W0.copy()
    Wb[1, -1, -1, -1] = 0.9 * Wb[0, -1, -1, -1]  # the maximum sits in the last cell of the last block
    small = wl.by_name("C1")                     # 32^3 = 8 blocks, |U| <= 0.1
    rng = np.random.default_rng(20260401)
    ragged = wl.by_name("C3", small=True)
    Wr = ragged.W0 * (1.0 + 0.05 * rng.standard_normal(ragged.W0.shape))
    for w, W, cfl in ((big, Wb, 0.4), (small, small.W0, 0.4), (big, Wb, 0.7), (ragged, Wr, 0.3)):
        assert _noalloc(w, W, cfl, out) == pytest.approx(_existing(w, W, cfl), rel=REL, abs=0)
    assert _noalloc(small, small.W0, 0.4, out) == pytest.approx(wl.cfl_dt(small.cfg, small.W0, 0.4), rel=1e-13)


def test_the_call_allocates_nothing_and_is_asynchronous():
    """free device memory is the same before and after (the module and its 512 KB array are loaded by the first call);
    back-to-back calls on one stream with no synchronisation in between are ordered and each writes its own output"""
    import torch
    from paper_2603_11102_b200 import gks
    w = wl.by_name("C1")
    Wd = torch.from_numpy(w.W0).to("cuda:0")
    W2 = Wd.clone()
    W2[1:] *= 3.0
    outs = torch.zeros(3, dtype=torch.float64, device="cuda:0")
    dmin = min(w.cfg.widths(a).min() for a in range(3))
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    gks.cfl_dt_noalloc(Wd, dmin, w.cfg.RT, 0.4, outs[0:1], stream=s)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    for k, (W, cfl) in enumerate(((Wd, 0.4), (W2, 0.4), (Wd, 0.8))):
        gks.cfl_dt_noalloc(W, dmin, w.cfg.RT, cfl, outs[k:k + 1], stream=s)
    s.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    o = outs.cpu().numpy()
    assert o[0] == pytest.approx(wl.cfl_dt(w.cfg, w.W0, 0.4), rel=1e-13)
    assert o[1] == pytest.approx(wl.cfl_dt(w.cfg, W2.cpu().numpy(), 0.4), rel=1e-13) and o[1] < o[0]
    assert o[2] == 2.0 * o[0]


def test_refusals():
    """sizes beyond the static scratch, host pointers and bad scalars are refused with a message; dt is untouched"""
    import ctypes as C
    import torch
    from paper_2603_11102_b200 import gks
    L = gks.lib()
    Wd = torch.ones((4, 8, 8, 8), dtype=torch.float64, device="cuda:0")
    out = torch.full((1,), -7.0, dtype=torch.float64, device="cuda:0")
    host = np.ones((4, 8, 8, 8))
    call = lambda W, nx, ny, nz, dmin, RT, cfl, dt: L.gks_cfl_dt_noalloc(W, nx, ny, nz, dmin, RT, cfl, dt, None)
    assert call(Wd.data_ptr(), 1024, 1024, 257, 0.1, 1.0, 0.4, out.data_ptr()) == 1       # 2^28 + 2^20 cells
    msg = L.gks_noalloc_last_error().decode()
    assert "GKS_NOALLOC_MAX_CELLS" in msg and "268435456" in msg, msg
    assert call(host.ctypes.data, 8, 8, 8, 0.1, 1.0, 0.4, out.data_ptr()) == 1
    assert "DEVICE" in L.gks_noalloc_last_error().decode()
    assert call(Wd.data_ptr(), 8, 8, 8, 0.1, 1.0, 0.4, host.ctypes.data) == 1
    assert call(None, 8, 8, 8, 0.1, 1.0, 0.4, out.data_ptr()) == 1
    assert call(Wd.data_ptr(), 0, 8, 8, 0.1, 1.0, 0.4, out.data_ptr()) == 1
    for bad in ((0.0, 1.0, 0.4), (0.1, -1.0, 0.4), (0.1, 1.0, float("nan"))):
        assert call(Wd.data_ptr(), 8, 8, 8, *bad, out.data_ptr()) == 1
    torch.cuda.synchronize()
    assert float(out.cpu()[0]) == -7.0
    with pytest.raises(gks.GksError):
        gks.cfl_dt_noalloc(Wd, -1.0, 1.0, 0.4, out)
    assert call(Wd.data_ptr(), 8, 8, 8, 0.1, 1.0, 0.4, out.data_ptr()) == 0               # and the maximum itself is a
    torch.cuda.synchronize()                                                               # size check, not a state
    assert float(out.cpu()[0]) == pytest.approx(0.4 * 0.1 / (3 ** 0.5 + 1.0), rel=1e-14)
