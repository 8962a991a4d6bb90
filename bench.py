#!/usr/bin/env python
"""bench.py — S2O4 GKS Mcell-steps/s (fp64) on the 256^3 periodic Taylor-Green box (workload M0).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload M0|C1..C5]

A "step" is one pass of the whole hot path (ghost fill, three fused sweeps, stage update, twice, then
forcing) over the whole grid.  Prints ONE JSON line (rank 0).  See DESIGN.md §Measurement for the
definitions of `roofline`, `e2e` and `cpu_baseline`.

Multi-GPU: the metric is built for one GPU (BASELINE.json north_star: no sharding, no collectives), so by default
--gpus N runs N independent replicas, one per rank ("replicas only", weak scaling).  `--decomp slab` instead cuts ONE
workload into N x-slabs with halo exchange over NCCL (paper_2603_11102_b200/slab.py; strong
scaling); that path is validated on one GPU and over gloo only - its NCCL numbers are UNVERIFIED until a box with two
or more GPUs has run it, and the JSON line says so.
"""
import argparse
import csv
import glob
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "S2O4 GKS Mcell-steps/s (fp64)"
# nominal fp64 FMA peak: 148 SMs x 64 DFMA lanes x 2 flop x 1.965 GHz
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12
UNIT = "Mcell-steps/s"
# Algorithmic fp64 flops of one cell-step (plain count of +,-,*,/ and one per
# erfc/exp/sqrt, smoothness indicators shared between the two points of a cell, Navier-Stokes closed
# form for the Gauss-point flux): per face 4726 (stage 1) + 4654 (stage 2), 3 faces per cell, + update.
FLOPS_PER_FACE = {True: 4726.0, False: 4654.0}     # need_F (stage 1) / dF only (stage 2)
# linear-weight tangential variant (--variant linear): an evaluation is 3 candidates x 5 + 5 = 20 flops per value,
# pass 1 = 8 fields x 40 + 4 slopes x 20 = 400, pass 2 = 24 x 40 + 8 x 20 = 1120, normal phase 518, flux 416 / 344
FLOPS_PER_FACE_LINEAR = {True: 2454.0, False: 2382.0}
FLOPS_PER_CELL_STEP = 3 * (FLOPS_PER_FACE[True] + FLOPS_PER_FACE[False]) + 60.0


def read_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md clocks line)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "20"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True)
            self.t.start()
        except OSError:
            self.proc = None

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smax = float(f[2])
            except ValueError:
                continue
            for nm, v in zip(names, f[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax,
                "reasons": sorted(reasons), "samples": len(sm)}


def setup_solver(w, gks, device):
    g = gks.Gks(w.cfg, device=device)
    if w.bulk_flux is not None:
        g.set_bulk_flux(*w.bulk_flux)
    if w.ibm is not None:
        g.ibm_set_points(*w.ibm)
    return g


def oracle_rate(sample_n, steps, warmup=0):
    """Mcell-steps/s of the CPU oracle, as it stands, on a Taylor-Green box of sample_n^3 cells (256 = M0 itself)."""
    from oracle import binding as ob
    from paper_2603_11102_b200 import workloads as wl
    ob.build()
    w = wl.taylor_green(sample_n)
    o = ob.Oracle(w.cfg)
    o.set_state(w.W0)
    for _ in range(warmup):
        o.step(w.dt)
    t0 = time.perf_counter()
    for _ in range(steps):
        o.step(w.dt)
    dt = time.perf_counter() - t0
    o.close()
    cores = len(os.sched_getaffinity(0))
    return w.cfg.cells * steps / dt / 1e6, dt, cores


def run_reference(args, rank, world):
    """--impl reference: the CPU oracle (the only reference this tier has), timed as it stands on the host cores ON
    THE METRIC BOX ITSELF (M0, 256^3).  One oracle step of 256^3 takes about 25 s on 16 cores, so the sample is
    bounded: min(K, 2) timed steps, no warm-up steps (the oracle has no caches to warm: its first step costs what
    every step costs); ms_per_step is the mean of the steps that were timed."""
    if rank != 0:
        return
    if args.workload != "M0":
        raise SystemExit("--impl reference times the metric workload M0")
    n = args.ref_box                      # 256 = M0 itself; smaller only for the CPU test of this arm's plumbing
    timed = max(1, min(args.steps, 2))
    rate, secs, cores = oracle_rate(n, timed, 0)
    sample = "%d of the %d steps timed (no warm-up), each one oracle step of the whole %d^3 box" % (timed, args.steps, n)
    line = {"impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": secs / timed * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic",
            "config": {"workload": "M0 taylor_green_%d %dx%dx%d" % (n, n, n, n), "sample": sample, "steps_timed": timed},
            "cpu_baseline": {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def time_workload(gks, wl, name, device, steps, warmup=3, variant="weno"):
    """Mcell-steps/s and per-class kernel times of one of the paper-shaped workloads, device-resident state,
    CUDA events on the solver's stream (the same procedure as the headline number, fewer steps)."""
    import torch
    w = wl.by_name(name)
    g = setup_solver(w, gks, device)
    if variant == "linear":
        g.set_reconstruction(1)
    g.set_state(w.W0)
    k = [0]

    def one():
        if w.alm is not None:
            g.alm_set_points(*w.alm(k[0]))
        g.step(w.dt)
        k[0] += 1

    for _ in range(warmup):
        one()
    g.synchronize()
    l0 = g.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    for _ in range(steps):
        one()
    e1.record(g.stream)
    g.synchronize()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count - l0
    g.profile_enable(True)          # the breakdown by kernel class: a second pass (see main)
    g.profile_read()
    for _ in range(steps):
        one()
    prof = g.profile_read()
    g.check_finite()
    g.close()
    return {"workload": "%s %s %dx%dx%d" % (name, w.name, *w.cfg.n), "value": w.cfg.cells * steps / (ms * 1e-3) / 1e6,
            "unit": UNIT, "steps": steps, "ms_per_step": ms / steps, "gpu_launches_per_step": launches / steps,
            "kernel_ms_per_step": {c: v[0] / steps for c, v in prof.items()}}


def run_slab_proxy(args, w, gks, device):
    """One interior sub-domain of `w` cut into N x-slabs, stepped on this GPU exactly as a rank of
    the slab driver steps it - halo pack / unpack kernels of W^n and W* included, device buffers - with its own
    opposite face as the neighbour on either side (= a periodic box of nx/N cells through the HALO path).  What it
    shows: the cost of the sub-domain shape (n+1 x-faces on tiles, fewer columns per sweep, the extra kernels)
    against 1/N of the single-domain step; the transfer itself (2 x 3 planes per stage over NVLink) is not in it."""
    import torch
    from paper_2603_11102_b200 import slab
    N = args.slab_proxy
    dec = slab.SlabDecomposition(w.cfg, N)
    r = N // 2
    cfg = dec.local_cfg(r)
    assert cfg.bc[0] == slab.BC_HALO and cfg.bc[1] == slab.BC_HALO, "the proxy wants an interior slab (N >= 3, or periodic x)"
    g = gks.Gks(cfg, device=device)
    g.set_state(dec.scatter(w.W0, r))
    with torch.cuda.stream(g.stream):
        b = [torch.empty(g.halo_doubles(f), dtype=torch.float64, device=device) for f in (0, 1)]
    g.synchronize()

    def exchange(which):
        g.halo_pack(which, 0, b[0])
        g.halo_pack(which, 1, b[1])
        g.halo_unpack(which, 0, b[1])
        g.halo_unpack(which, 1, b[0])

    def step():
        if args.overlap:      # the step in parts: pack, interior, unpack, rim (what a rank does while the halos travel)
            for which, part in ((0, g.step_begin_part), (1, g.step_finish_part)):
                g.halo_pack(which, 0, b[0])
                g.halo_pack(which, 1, b[1])
                part(w.dt, 0)
                g.halo_unpack(which, 0, b[1])
                g.halo_unpack(which, 1, b[0])
                part(w.dt, 1)
        else:
            exchange(0)
            g.step_begin(w.dt)
            exchange(1)
            g.step_finish(w.dt)
        g.step_force(w.dt)

    for _ in range(max(args.warmup, 3)):
        step()
    g.synchronize()
    l0 = g.launch_count
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    for _ in range(args.steps):
        step()
    e1.record(g.stream)
    g.synchronize()
    ms = e0.elapsed_time(e1) / args.steps
    launches = (g.launch_count - l0) / args.steps
    g.profile_enable(True)
    g.profile_read()
    for _ in range(args.steps):
        step()
    prof = g.profile_read()
    g.check_finite()
    g.close()
    # the single-domain step of the same workload, same run
    g1 = setup_solver(w, gks, device)
    g1.set_state(w.W0)
    for _ in range(3):
        g1.step(w.dt)
    g1.synchronize()
    e0.record(g1.stream)
    for _ in range(args.steps):
        g1.step(w.dt)
    e1.record(g1.stream)
    g1.synchronize()
    ms1 = e0.elapsed_time(e1) / args.steps
    g1.close()
    print(json.dumps({
        "metric": METRIC, "value": cfg.cells / (ms * 1e-3) / 1e6, "unit": UNIT, "n_gpus": 1, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True, "dtype": "f64", "data": "synthetic",
        "config": {"workload": "%s x-slab %d of %d: %dx%dx%d cells, HALO faces on both sides" % (args.workload, r, N, *cfg.n),
                   "step": "in parts (interior, then rim: gks_step_begin_part)" if args.overlap else "plain",
                   "note": "one sub-domain on one GPU, its own opposite face as the neighbours; no transfer"},
        "gpu_launches_per_step": launches,
        "single_domain_ms_per_step": ms1,
        "strong_scaling_proxy": {"ideal_ms": ms1 / N, "slab_ms": ms, "efficiency": (ms1 / N) / ms},
        "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()}}), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="M0")
    ap.add_argument("--sweep", type=int, default=0, help="0 fused (production), 1 unfused cross-check kernels")
    ap.add_argument("--variant", default="weno", choices=["weno", "linear"],
                    help="weno: the scheme as read from the paper (default, the metric); linear: linear-weight tangential passes")
    ap.add_argument("--decomp", default="replicas", choices=["replicas", "slab"],
                    help="N > 1: replicas = N independent copies of the workload (default, weak scaling); slab = ONE\n"
                         "workload cut into N x-slabs with halo exchange over NCCL (strong scaling, PAPER.md:193-197)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--ref-box", type=int, default=256,
                    help="--impl reference: cells per axis of the Taylor-Green box the oracle is timed on (256 = M0)")
    ap.add_argument("--slab-proxy", type=int, default=0,
                    help="time ONE interior x-slab of the workload cut into N slabs on this GPU: HALO faces on both sides,\n"
                         "halo pack / unpack inside the step, the slab's own opposite face standing in for the neighbours\n"
                         "(a strong-scaling proxy that needs no second GPU; prints its own JSON line)")
    ap.add_argument("--overlap", action="store_true",
                    help="--slab-proxy / --decomp slab: the step in parts (interior while the halos travel, then the rim)")
    ap.add_argument("--online-rotor", action="store_true",
                    help="workloads with an ALM rotor (C4, C5): the on-line blade-element rotor (alm_set_rotor: sampling,\n"
                         "Eq. 9, tip and free-stream corrections on the device, synthetic blade data) instead of prescribed\n"
                         "point forces re-set from the host every step")
    ap.add_argument("--no-configs", action="store_true", help="skip the C1..C5 throughput block of the JSON line")
    ap.add_argument("--ibm-passes", type=int, default=1, help="IBM multi-direct-forcing passes per step (workloads with IBM)")
    ap.add_argument("--halo", choices=["messages", "push"], default="messages",
                    help="--decomp slab: halos as NCCL messages between pack / unpack kernels, or written straight into the\n"
                         "neighbour process's ghost layers through CUDA IPC mappings (slab.IpcPushTransport)")
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--e2e-depth", type=int, default=2, help="contexts in rotation in the pipelined end-to-end leg")
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        return run_reference(args, rank, world)

    import torch
    import torch.distributed as dist
    from paper_2603_11102_b200 import gks, workloads as wl
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    device = "cuda:%d" % local_rank
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device(device))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # the library is built in-tree (git ignores the .so): a fresh checkout compiles it once, rank 0 only
    if rank == 0:
        from paper_2603_11102_b200 import build as gks_build
        gks_build.build()
    barrier()

    w = wl.by_name(args.workload)
    if args.slab_proxy > 1:
        return run_slab_proxy(args, w, gks, device)
    slab_mode = args.decomp == "slab" and world > 1
    stepper = None
    if slab_mode:
        # one workload, N x-slabs: this rank owns one sub-domain; halos move over NCCL (paper_2603_11102_b200/slab.py)
        from dataclasses import replace as dc_replace
        from paper_2603_11102_b200 import slab
        dec = slab.SlabDecomposition(w.cfg, world)
        ibm_local = dec.ibm_points(rank, *w.ibm) if w.ibm is not None else None
        w_global = w
        w = dc_replace(w, cfg=dec.local_cfg(rank), W0=dec.scatter(w.W0, rank), ibm=ibm_local)
    if args.sweep == 1:                  # the unfused cross-check kernels exist in the debug library only
        g = gks.Gks(w.cfg, device=device, debug=True)
        if w.bulk_flux is not None:
            g.set_bulk_flux(*w.bulk_flux)
        if w.ibm is not None:
            g.ibm_set_points(*w.ibm)
        g.debug_set_sweep(1)
    else:
        g = setup_solver(w, gks, device)
    if args.ibm_passes > 1 and w.ibm is not None:
        g.ibm_set_iterations(args.ibm_passes, 0.0)
    if slab_mode:
        transport = slab.IpcPushTransport(dec, rank, g) if args.halo == "push" else slab.DistTransport(dec, rank)
        stepper = slab.SlabStepper(transport, g, slab.BufferPool(device))
    if args.variant == "linear":
        g.set_reconstruction(1)
    cells = w.cfg.cells
    with torch.cuda.stream(g.stream):
        Wd = torch.from_numpy(w.W0).to(device)
    g.stream.synchronize()
    g.set_state(Wd)
    step_no = [0]
    rotor_drv = None
    if args.online_rotor:
        if w.alm is None:
            raise SystemExit("--online-rotor needs a workload with an ALM rotor (C4, C5)")
        w_ref = w_global if slab_mode else w
        pos0, _, eps = w_ref.alm(0)
        hub = pos0.reshape(3, -1, 3).mean(axis=(0, 1))          # the prescribed blades are 120 degrees apart
        rot = wl.synthetic_rotor(hub=hub, R=float(np.linalg.norm(pos0 - hub, axis=1).max() * 64.5 / 64.0), eps=eps,
                                 freestream_correction=True, tip_correction=True)
        if slab_mode:
            rotor_drv = slab.RotorDriver(dec, rot, device)
        else:
            g.alm_set_rotor(rot)
        from dataclasses import replace as _rep
        w = _rep(w, alm=None)                                   # no prescribed points any more

    def slab_step(k):
        # actuator points reach a slab through dec.alm_points (supports across cuts, images beyond a periodic seam)
        hook = (lambda s: s.alm_set_points(*dec.alm_points(rank, *w.alm(k)))) if w.alm is not None else None
        stepper.step(w.dt, before_forcing=hook, ibm=w_global.ibm is not None, bulk=w.bulk_flux is not None,
                     ibm_passes=args.ibm_passes, rotor=rotor_drv, overlap=args.overlap, push=args.halo == "push")

    def one_step():
        if stepper is not None:
            slab_step(step_no[0])
        else:
            if w.alm is not None:
                g.alm_set_points(*w.alm(step_no[0]))
            g.step(w.dt)
        step_no[0] += 1

    for _ in range(max(args.warmup, 3)):
        one_step()
    g.synchronize()
    # context figure only (the headline fraction is against the nominal unit count): DFMA throughput of this GPU
    fp64_peak = gks.fp64_peak(device) if rank == 0 else None

    # ---- timed region: exactly K steps, device-resident state, CUDA events on the solver's stream.  The per-class
    # event recorder is OFF here (its event records between the kernels would keep a kernel's launch from overlapping
    # the tail of its predecessor); the per-class breakdown comes from a second, untimed pass below.
    l0 = g.launch_count
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    for _ in range(args.steps):
        one_step()
    e1.record(g.stream)
    g.synchronize()
    barrier()
    clocks = sampler.stop()
    ms = e0.elapsed_time(e1)
    launches = g.launch_count - l0
    g.check_finite()
    # ---- per-class kernel times (CUDA events around every class of kernels), same number of steps, not timed as a whole
    g.profile_enable(True)
    g.profile_read()
    for _ in range(args.steps):
        one_step()
    prof = g.profile_read()
    g.profile_enable(False)

    # ---- end to end through the C ABI with HOST buffers (pinned): H2D + step + D2H every step
    Hin = torch.from_numpy(w.W0.copy()).pin_memory()
    Hout = torch.empty_like(Hin).pin_memory()
    nbytes = Hin.numel() * 8
    def plain_step():
        if stepper is not None:
            slab_step(step_no[0])
        else:
            g.step(w.dt)

    g.set_state(Hin)
    plain_step()
    g.get_state(Hout)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.e2e_steps):
        g.set_state(Hin)
        plain_step()
        g.get_state(Hout)          # synchronises
        Hin, Hout = Hout, Hin
    barrier()
    e2e_s = time.perf_counter() - t0

    # ---- the same with INDEPENDENT batches through two contexts in rotation (gks.HostPipeline): every batch is still
    # copied in from pinned host memory, stepped and copied back inside the timed region, but the copies of one batch
    # run on the copy engines while the other context computes.  Timed from the first submit to the last batch back in
    # host memory (pipeline fill and drain included).
    pipe_s, pipe_batches = 0.0, 0
    if stepper is None and args.sweep == 0 and not args.online_rotor:
        def setup(gp):
            if w.bulk_flux is not None:
                gp.set_bulk_flux(*w.bulk_flux)
            if w.ibm is not None:
                gp.ibm_set_points(*w.ibm)
                if args.ibm_passes > 1:
                    gp.ibm_set_iterations(args.ibm_passes, 0.0)
            if args.variant == "linear":
                gp.set_reconstruction(1)
        pipe = gks.HostPipeline(w.cfg, depth=args.e2e_depth, device=device, setup=setup)
        nd = args.e2e_depth
        Hi = [torch.from_numpy(w.W0.copy()).pin_memory() for _ in range(nd)]
        Ho = [torch.empty_like(Hi[0]).pin_memory() for _ in range(nd)]
        hook = (lambda gp, s_: gp.alm_set_points(*w.alm(0))) if w.alm is not None else None
        for b in range(nd):                                  # untimed: every context once
            pipe.submit(Hi[b], Ho[b], w.dt, before_step=hook)
        pipe.drain()
        pipe_batches = 8 * args.e2e_steps
        barrier()
        t0 = time.perf_counter()
        for b in range(pipe_batches):
            pipe.submit(Hi[b % nd], Ho[b % nd], w.dt, before_step=hook)
        pipe.drain()
        barrier()
        pipe_s = time.perf_counter() - t0
        pipe.close()
        del pipe, Hi, Ho

    t = torch.tensor([ms, e2e_s * 1e3, pipe_s * 1e3], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms, e2e_ms, pipe_ms = t.tolist()
    if rank == 0:
        peaks, peak_src = read_peaks()
        # replicas: every rank steps its own copy of the workload; slab: the ranks share ONE workload
        total_cells = w_global.cfg.cells if slab_mode else cells * world
        value = total_cells * args.steps / (ms * 1e-3) / 1e6
        e2e_value = total_cells * args.e2e_steps / (e2e_ms * 1e-3) / 1e6
        serial = {"value": e2e_value, "steps": args.e2e_steps,
                  "mode": "one context; copy in, step, copy out in sequence (each step's input is the previous output)"}
        if pipe_batches:
            e2e = {"value": total_cells * pipe_batches / (pipe_ms * 1e-3) / 1e6, "unit": UNIT,
                   "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes, "steps": pipe_batches,
                   "depth": args.e2e_depth,
                   "mode": "independent batches through %d contexts in rotation (gks.HostPipeline): every batch is copied "
                           "in from pinned host memory, stepped and copied back; the copies overlap the other context's "
                           "step; timed from the first submit to the last batch in host memory" % args.e2e_depth,
                   "serial": serial}
        else:
            e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                   "steps": args.e2e_steps, "mode": serial["mode"]}
        sweep_ms = sum(prof[k][0] for k in ("sweep_x", "sweep_y", "sweep_z"))
        sweep_n = sum(prof[k][1] for k in ("sweep_x", "sweep_y", "sweep_z"))
        faces = cells  # one face per cell and direction (+ one boundary plane, < 0.5 %)
        fpf = FLOPS_PER_FACE_LINEAR if args.variant == "linear" else FLOPS_PER_FACE
        flops_per_launch = 0.5 * (fpf[True] + fpf[False]) * faces
        ach = flops_per_launch / (sweep_ms / max(sweep_n, 1) * 1e-3) / 1e12 if sweep_ms > 0 else None
        traffic, frac_pipe = None, None
        tps = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic.csv")))
        if tps and args.workload == "M0" and args.sweep == 0 and args.variant == "weno":
            with open(tps[-1]) as f:      # latest round's ncu --set full capture (text summary, not executed)
                for row in csv.DictReader(f):
                    if row["kernel"] == "sweep_mean_of_6":
                        traffic = float(row["dram_bytes_per_launch"])
                        if row.get("fp64_pipe_active_pct"):
                            frac_pipe = float(row["fp64_pipe_active_pct"]) / 100.0
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True,
            "scaling": "strong" if slab_mode else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "%s %s %dx%dx%d" % (args.workload, w.name, *(w_global if slab_mode else w).cfg.n),
                       "sweep": "fused" if args.sweep == 0 else "unfused", "variant": args.variant,
                       "alm": ("on-line rotor (alm_set_rotor, synthetic blade data)" if args.online_rotor else
                               ("prescribed point forces" if (w_global if slab_mode else w).alm is not None else None)),
                       "multi_gpu": (("x-slabs, halos pushed into the neighbour's ghosts (CUDA IPC)" if args.halo == "push" else "x-slabs with halo exchange") if slab_mode else "replicas only") if world > 1 else "single GPU",
                       "l2": "inputs larger than L2 (state %.0f MB per field set)" % (cells * 32 / 1e6)},
            "clocks": clocks,
            "e2e": e2e,
            "gpu_launches": int(launches),
            # headline fraction: against the NOMINAL fp64 rate (unit count x clock; neither MEASURED_PEAKS.json nor the
            # profiling guide carries an fp64 figure).  frac_pipe: ncu "fp64 pipe active" of the same kernels from the
            # committed capture (profiles/), the honest utilisation figure: `achieved` counts unfused +,-,* as one flop
            # each while the peak counts two per DFMA.  peak_dfma_measured: this run's own DFMA calibration (context).
            "roofline": {"bound": "alu", "kernel": "sweep (reconstruction + flux), mean of 6 launches per step",
                         "achieved": ach, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                         "frac": (ach / FP64_NOMINAL_TFLOPS) if ach else None, "traffic": traffic,
                         "peak_source": "nominal: 148 SMs x 64 fp64 FMA lanes x 2 flop x 1.965 GHz (DESIGN.md section 8)",
                         "frac_nominal": (ach / FP64_NOMINAL_TFLOPS) if ach else None,
                         "frac_pipe": frac_pipe,
                         "frac_pipe_source": os.path.relpath(tps[-1], ROOT) if (tps and frac_pipe is not None) else None,
                         "peak_dfma_measured": fp64_peak,
                         "frac_dfma_measured": (ach / fp64_peak) if (ach and fp64_peak) else None,
                         "flops_per_launch": flops_per_launch,
                         "share_of_step": sweep_ms / ms if ms > 0 else None},
            "hbm": {"bytes_per_cell_step_algorithmic": 192,
                    "achieved_gbs": 192.0 * cells * args.steps / (ms * 1e-3) / 1e9,
                    "peak_gbs": peaks.get("hbm_gbs"), "peak_source": peak_src},
            "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
        }
        if slab_mode:
            line["config"]["note"] = "x-slab numbers over NCCL are UNVERIFIED: validated on one GPU and over gloo only"
    if slab_mode and args.halo == "push":
        transport.close()              # unmap the neighbours' workspaces before anyone frees
    g.close()
    if rank == 0:
        if not args.no_configs and world == 1 and args.workload == "M0" and args.sweep == 0:
            # north_star: throughput on the five paper-shaped workloads, same run, same procedure, 5 timed steps each
            line["configs"] = {nm: time_workload(gks, wl, nm, device, steps=5, variant=args.variant)
                               for nm in ("C1", "C2", "C3", "C4", "C5")}
        if not args.no_cpu_baseline and world == 1:
            if args.workload == "M0":       # the metric box itself: one oracle step of 256^3 (about 25 s on 16 cores)
                rate, secs, cores = oracle_rate(256, 1, warmup=0)
                sample = "1 oracle step of the whole 256^3 Taylor-Green box (the workload of `value`)"
            else:
                rate, secs, cores = oracle_rate(128, 3, warmup=1)
                sample = "3 steps (after 1 untimed) of the 128^3 Taylor-Green box"
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "seconds": secs}
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
