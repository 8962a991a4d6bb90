"""Measurement helpers behind the numbers DESIGN.md section 7 and profiles/r2_microbench.md quote.

    python -m paper_2603_11102_b200.trace            phase timeline of the fused sweep (three directions, M0 256^3)
    python -m paper_2603_11102_b200.trace --probe    issue-rate probe (fp64 against integer instructions, fp64 ILP)

The timeline needs the phase timers compiled into the kernel: this module builds libgks_b200_trace.so (the debug
library with -DGKS_TRACE, paper_2603_11102_b200/build.py build_trace) on first use.  The timers cost registers and
clock reads: the instrumented kernel runs a few per cent slower than the product; shares, not absolutes, are the result.
"""
import ctypes as C
import sys

import numpy as np

PHASES = ["loop bookkeeping", "hand-over wait", "TMA issue + cursor", "stage A", "stages BC + D, arrival", "pass 2 (E)",
          "transposes, flux, store (F)"]
# fp64 warp instructions of one warp and plane per phase (static count of the source: DESIGN.md section 7)
PROBE = ["KF=8 KI=0  chains=8", "KF=8 KI=4  chains=8", "KF=8 KI=8  chains=8", "KF=8 KI=12 chains=8", "KF=8 KI=16 chains=8",
         "KF=4 KI=8  chains=8", "KF=8 KI=0  chains=1", "KF=8 KI=0  chains=2", "KF=8 KI=0  chains=4"]


def probe():
    from . import gks
    from .workloads import GridConfig
    g = gks.Gks(GridConfig(n=(8, 8, 8), spacing=(1.0, 1.0, 1.0)), debug=True)
    out = (C.c_double * 9)()
    g._c("gks_debug_issue_probe", out, 9)
    print("issue-rate probe: 512 threads per CTA, one CTA per SM = 4 warps per scheduler; per round and warp KF DFMA on")
    print("`chains` independent register chains + KI integer multiply-adds on 8 chains; cycles per round (clock64)")
    print("| case | cycles / round | fp64 pipe needs 4 warps x KF x 2 | integer pipe needs 4 x KI x 2 |")
    print("|---|---|---|---|")
    for name, c in zip(PROBE, out):
        kf, ki = int(name.split("KF=")[1].split()[0]), int(name.split("KI=")[1].split()[0])
        print("| %s | %.1f | %d | %d |" % (name, c, 8 * kf, 8 * ki))
    print("fp64 peak of this GPU by the DFMA calibration kernel: %.2f TFLOP/s" % g.debug_fp64_peak())
    g.close()


def timeline():
    import torch
    from . import build, gks, workloads as wl
    build.build_trace()
    w = wl.by_name("M0")
    g = gks.Gks(w.cfg, debug="trace")
    g.set_state(w.W0)
    g.step(w.dt)
    g.synchronize()
    n = w.cfg.n
    ticks = (C.c_ulonglong * 256)()
    for d, axis in enumerate("xyz"):
        with torch.cuda.stream(g.stream):
            F = torch.empty(4 * (n[0] + 1) * (n[1] + 1) * (n[2] + 1), dtype=torch.float64, device="cuda:0")
            dF = torch.empty_like(F)
        g._c("gks_debug_eval_flux", d, F.data_ptr(), dF.data_ptr())     # one stage-1 sweep of direction d
        g._c("gks_debug_trace", ticks)
        a = np.array(list(ticks), dtype=np.float64).reshape(32, 8)[:16, :7]
        # CTA 0 marches floor(C / 148) whole columns of 256 planes + 4 priming planes each, plus its share of the rest
        iters = a.sum(1).mean() / 1.0
        print("\n%s-faces, stage 1: clock64 ticks per warp of CTA 0, summed over the launch: %.3e" % (axis, iters))
        print("| phase | share of the warp's time | min .. max over the 16 warps |")
        print("|---|---|---|")
        tot = a.sum()
        for k, nm in enumerate(PHASES):
            col = a[:, k] / a.sum(1)
            print("| %s | %.1f %% | %.1f .. %.1f %% |" % (nm, 100 * a[:, k].sum() / tot, 100 * col.min(), 100 * col.max()))
    g.close()


if __name__ == "__main__":
    probe() if "--probe" in sys.argv else timeline()
