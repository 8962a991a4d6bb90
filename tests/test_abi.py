"""CPU-side checks of the boundary: the C-ABI library loads, exports every symbol include/gks.h
declares, and the host logic that needs no GPU (validation) answers as documented."""
import ctypes as C
import os
import re
import subprocess

import numpy as np
import pytest

from paper_2603_11102_b200 import gks, workloads as wl

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_functions(header="gks.h"):
    src = open(os.path.join(ROOT, "include", header)).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b((?:gks|alm|ibm)_[a-z0-9_]+)\s*\(", src)))


def exported_functions(path):
    out = subprocess.run(["nm", "-D", "--defined-only", path], capture_output=True, text=True, check=True).stdout
    return sorted(ln.split()[-1] for ln in out.splitlines() if " T " in ln)


def test_library_exports_every_declared_symbol():
    """the product library exports include/gks.h and nothing else; the debug library adds include/gks_debug.h"""
    from paper_2603_11102_b200 import build
    build.build()
    L = C.CDLL(gks._LIB_PATH)
    names = declared_functions()
    assert len(names) >= 15
    for n in names:
        assert hasattr(L, n), n
    assert sorted(gks.EXPORTS) == names
    assert exported_functions(gks._LIB_PATH) == names
    dbg = declared_functions("gks_debug.h")
    assert dbg == sorted(gks.DEBUG_EXPORTS) and len(dbg) >= 2
    assert exported_functions(gks._LIB_DEBUG_PATH) == sorted(names + dbg)
    for n in dbg:                           # the test hooks and their kernels do not ship in the product
        assert not hasattr(L, n), n


def test_product_workspace_does_not_carry_the_cross_check_buffers():
    """gks_workspace_bytes of the product: 3 states + 3 x 8 flux fields = 36 padded fields (+ tables, point arrays);
    the debug library adds the 32 fields of intermediates of the unfused sweep"""
    w = wl.taylor_green(64)
    c, keep = gks.make_config(w.cfg)
    padded = 72 * 70 * 70 * 8
    prod = gks.lib().gks_workspace_bytes(C.byref(c))
    dbg = gks.lib(True).gks_workspace_bytes(C.byref(c))
    assert 36 * padded <= prod <= 36 * padded + (12 << 20)
    assert dbg - prod >= 32 * padded


def test_workspace_bytes_and_validation_without_gpu():
    L = gks.lib()
    w = wl.taylor_green(32)
    c, keep = gks.make_config(w.cfg)
    nbytes = L.gks_workspace_bytes(C.byref(c))
    padded = 40 * 38 * 38              # pitch rounded up to 4
    assert nbytes >= 36 * 8 * padded and nbytes % 256 == 0
    c.nx = 5                           # too small for the 5-cell stencils and 3 ghost layers
    assert L.gks_workspace_bytes(C.byref(c)) == 0
    c.nx = 32
    c.bc[0] = wl.BC_WALL_SLIP          # unpaired periodic
    assert L.gks_workspace_bytes(C.byref(c)) == 0
    c.bc[0] = wl.BC_PERIODIC
    c.RT = 0.0
    assert L.gks_workspace_bytes(C.byref(c)) == 0


def test_create_fails_loudly_without_a_device_or_workspace():
    import torch
    L = gks.lib()
    w = wl.taylor_green(32)
    c, keep = gks.make_config(w.cfg)
    h = C.c_void_p()
    st = L.gks_create(C.byref(c), None, 0, None, C.byref(h))
    assert st != gks.GKS_OK and not h.value
    msg = L.gks_last_error(None).decode()
    if not torch.cuda.is_available():
        assert st == 3 and "no CPU fallback" in msg        # GKS_ERR_CUDA
        with pytest.raises(RuntimeError):
            gks.Gks(w.cfg)
    else:
        assert st == 2                                      # GKS_ERR_WORKSPACE


def test_workload_shapes_match_baseline_configs():
    sizes = {"C1": (32, 32, 32), "C2": (128, 96, 64), "C3": (256, 128, 64)}
    for k, n in sizes.items():
        w = wl.by_name(k)
        assert w.cfg.n == n and w.W0.shape == (4, n[2], n[1], n[0])
    c3 = wl.by_name("C3")
    assert len(c3.ibm[0]) == 64 * 64
    pos, frc, eps = wl.by_name("C4", small=True).alm(3)
    assert pos.shape == (192, 3) and frc.shape == (192, 3)
    thrust = 0.5 * 0.1 ** 2 * np.pi * 0.8
    assert frc[:, 0].sum() == pytest.approx(-thrust, rel=1e-12)
