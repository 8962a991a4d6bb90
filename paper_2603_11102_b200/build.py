"""Builds the CUDA libraries in-tree with nvcc for sm_100a (no JIT cache; the .so files travel with the repo):

  libgks_b200.so        the product: include/gks.h and nothing else
  libgks_b200_debug.so  the same sources with -DGKS_DEBUG: adds include/gks_debug.h (the unfused cross-check sweep
                        with its workspace and the fp64 calibration kernel); loaded by tests/ and by bench.py's
                        calibration only
"""
import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libgks_b200.so")
LIB_DEBUG = os.path.join(HERE, "libgks_b200_debug.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
         "-Xcompiler", "-fPIC", "-ccbin", "/usr/bin/g++"]
# translation units that do not look at GKS_DEBUG: one object serves both libraries
SHARED_OBJECTS = ("gks_update", "gks_ghost", "gks_forcing", "gks_rotor", "gks_noalloc", "gks_ipc")


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def _run(cmd):
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        raise RuntimeError("nvcc failed: %s\n%s\n%s" % (" ".join(cmd), r.stdout, r.stderr))
    return r.stderr


def build(force=False, verbose=False, extra_flags=()):
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    hdrs = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h"))
    objdir = os.path.join(HERE, "build")
    os.makedirs(os.path.join(objdir, "debug"), exist_ok=True)
    jobs, objs, objs_debug = [], [], []
    for s in srcs:
        stem = os.path.basename(s)[:-3]
        o = os.path.join(objdir, stem + ".o")
        variants = [(o, [])]
        if stem in SHARED_OBJECTS:
            objs_debug.append(o)
        else:
            od = os.path.join(objdir, "debug", stem + ".o")
            variants.append((od, ["-DGKS_DEBUG"]))
            objs_debug.append(od)
        if stem != "gks_sweep_unfused":       # empty without GKS_DEBUG
            objs.append(o)
        else:
            variants = variants[1:]
        for obj, defs in variants:
            if force or _newer(obj, [s] + hdrs):
                jobs.append([NVCC] + FLAGS + list(extra_flags) + defs + (["-Xptxas", "-v"] if verbose else []) +
                            ["-c", s, "-o", obj])
    with ThreadPoolExecutor(max_workers=8) as ex:
        logs = list(ex.map(_run, jobs))
    if verbose:
        for l in logs:
            sys.stderr.write(l)
    vs = os.path.join(CSRC, "gks_exports.map")
    for lib, lobjs in ((LIB, objs), (LIB_DEBUG, objs_debug)):
        if force or jobs or _newer(lib, lobjs + [vs]):
            _run([NVCC, "-shared", "-o", lib] + lobjs + ["-gencode", "arch=compute_100a,code=sm_100a",
                                                         "-ccbin", "/usr/bin/g++", "-Xlinker", "--version-script=" + vs])
    return LIB


def build_trace():
    """libgks_b200_trace.so: the debug library with -DGKS_TRACE (phase timers in the fused sweep, include/gks_debug.h
    gks_debug_trace).  Built on demand by paper_2603_11102_b200/trace.py; not a product artefact."""
    lib = os.path.join(HERE, "libgks_b200_trace.so")
    srcs = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    hdrs = glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        glob.glob(os.path.join(HERE, "..", "include", "*.h"))
    objdir = os.path.join(HERE, "build", "trace")
    os.makedirs(objdir, exist_ok=True)
    jobs, objs = [], []
    for s in srcs:
        o = os.path.join(objdir, os.path.basename(s)[:-3] + ".o")
        objs.append(o)
        if _newer(o, [s] + hdrs):
            jobs.append([NVCC] + FLAGS + ["-DGKS_DEBUG", "-DGKS_TRACE", "-c", s, "-o", o])
    with ThreadPoolExecutor(max_workers=8) as ex:
        list(ex.map(_run, jobs))
    if jobs or _newer(lib, objs):
        _run([NVCC, "-shared", "-o", lib] + objs + ["-gencode", "arch=compute_100a,code=sm_100a", "-ccbin", "/usr/bin/g++",
                                                    "-Xlinker", "--version-script=" + os.path.join(CSRC, "gks_exports.map")])
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
