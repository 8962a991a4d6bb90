"""Thin Python binding of libgks_b200.so (include/gks.h).  Argument marshalling only: every step of
the path runs in the library's CUDA kernels.  PyTorch supplies device memory and the stream.

There is no CPU fallback: if the library is missing or no CUDA device is present this module raises.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libgks_b200.so")
_LIB_DEBUG_PATH = os.path.join(_HERE, "libgks_b200_debug.so")     # same sources with -DGKS_DEBUG (include/gks_debug.h)
_LIBS = {}
_dp = C.POINTER(C.c_double)

GKS_OK = 0
STATUS = {0: "GKS_OK", 1: "GKS_ERR_INVALID_ARG", 2: "GKS_ERR_WORKSPACE", 3: "GKS_ERR_CUDA",
          4: "GKS_ERR_STATE", 5: "GKS_ERR_NONFINITE"}

EXPORTS = ["gks_workspace_bytes", "gks_create", "gks_destroy", "gks_set_state", "gks_get_state", "gks_step",
           "gks_set_body_force", "gks_set_bulk_flux", "alm_set_points", "ibm_set_points", "ibm_set_velocities", "ibm_set_iterations", "gks_cfl_dt", "alm_set_rotor", "alm_rotor_eval", "alm_rotor_points", "gks_set_reconstruction", "gks_halo_doubles", "gks_halo_pack", "gks_halo_unpack", "gks_step_begin",
           "gks_step_finish", "gks_step_force", "gks_bulk_partial", "gks_bulk_set_global", "gks_ibm_pass", "gks_ibm_residual",
           "gks_debug_eval_flux", "alm_rotor_supply", "gks_step_begin_part", "gks_step_finish_part", "gks_halo_window_get", "gks_halo_push",
           "gks_profile_enable", "gks_profile_read", "gks_check_finite", "gks_launch_count", "gks_last_error",
           "gks_cfl_dt_noalloc", "gks_noalloc_last_error", "gks_halo_export_get", "gks_halo_export_open", "gks_halo_export_close", "gks_step_begin_push"]
DEBUG_EXPORTS = ["gks_debug_set_sweep", "gks_debug_fp64_peak", "gks_debug_issue_probe", "gks_debug_trace"]    # include/gks_debug.h: libgks_b200_debug.so only


class AlmRotor(C.Structure):
    _fields_ = [("nblades", C.c_int), ("npts", C.c_int), ("hub", C.c_double * 3),
                ("R", C.c_double), ("r_hub", C.c_double), ("omega", C.c_double), ("theta0", C.c_double),
                ("u_ref", C.c_double), ("eps", C.c_double), ("chord", _dp), ("twist", _dp),
                ("npolar", C.c_int), ("alpha", _dp), ("cl", _dp), ("cd", _dp),
                ("freestream_correction", C.c_int), ("tip_correction", C.c_int),
                ("radius", _dp), ("width", _dp), ("nsections", C.c_int), ("section_r", _dp)]


class HaloWindow(C.Structure):
    _fields_ = [("W", C.c_void_p), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("pitch_x", C.c_int),
                ("pitch_y", C.c_int), ("field_stride", C.c_longlong)]


class HaloExport(C.Structure):
    """gks_halo_export: a sub-domain's windows as plain bytes for another process (bytes(e) / HaloExport.from_buffer_copy)"""
    _fields_ = [("mem", C.c_ubyte * 64), ("offset", C.c_ulonglong * 2), ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("pitch_x", C.c_int), ("pitch_y", C.c_int), ("field_stride", C.c_longlong)]


class GksConfig(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xf", _dp), ("yf", _dp), ("zf", _dp),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("RT", C.c_double), ("nu", C.c_double), ("rho_ref", C.c_double),
                ("bc", C.c_int * 6), ("inflow", C.c_double * 4), ("weno_eps", C.c_double)]


class GksError(RuntimeError):
    def __init__(self, status, message):
        super().__init__("%s: %s" % (STATUS.get(status, status), message))
        self.status = status


def lib(debug=False):
    """Load libgks_b200.so - or, debug=True, libgks_b200_debug.so, the same sources with the test hooks of
    include/gks_debug.h - built in-tree by paper_2603_11102_b200/build.py.  Fails loudly if absent.
    debug="trace" loads libgks_b200_trace.so (the debug library with the phase timers of the fused sweep compiled in,
    built on demand by paper_2603_11102_b200/trace.py)."""
    if debug not in _LIBS:
        path = _LIB_DEBUG_PATH if debug else _LIB_PATH
        if debug == "trace":
            path = os.path.join(_HERE, "libgks_b200_trace.so")
        if not os.path.exists(path):
            raise ImportError("%s is not built (run `python -m paper_2603_11102_b200.build`); "
                              "there is no CPU fallback" % os.path.basename(path))
        L = C.CDLL(path)
        vp = C.c_void_p
        L.gks_workspace_bytes.argtypes = [C.POINTER(GksConfig)]
        L.gks_workspace_bytes.restype = C.c_size_t
        L.gks_create.argtypes = [C.POINTER(GksConfig), vp, C.c_size_t, vp, C.POINTER(vp)]
        L.gks_destroy.argtypes = [vp]
        L.gks_set_state.argtypes = [vp, vp]
        L.gks_get_state.argtypes = [vp, vp]
        L.gks_step.argtypes = [vp, C.c_double]
        L.gks_set_body_force.argtypes = [vp, C.c_double, C.c_double, C.c_double]
        L.gks_set_bulk_flux.argtypes = [vp, C.c_int, C.c_double]
        L.alm_set_points.argtypes = [vp, C.c_int, vp, vp, C.c_double]
        L.ibm_set_points.argtypes = [vp, C.c_int, vp, vp]
        L.ibm_set_velocities.argtypes = [vp, vp]
        L.ibm_set_iterations.argtypes = [vp, C.c_int, C.c_double]
        L.gks_cfl_dt.argtypes = [vp, C.c_double, vp]
        L.alm_set_rotor.argtypes = [vp, C.POINTER(AlmRotor)]
        L.alm_rotor_eval.argtypes = [vp, vp, vp]
        L.alm_rotor_points.argtypes = [vp, C.POINTER(AlmRotor), C.c_double, vp, vp]
        L.gks_set_reconstruction.argtypes = [vp, C.c_int]
        L.gks_halo_doubles.argtypes = [vp, C.c_int]
        L.gks_halo_doubles.restype = C.c_size_t
        L.gks_halo_pack.argtypes = [vp, C.c_int, C.c_int, vp]
        L.gks_halo_unpack.argtypes = [vp, C.c_int, C.c_int, vp]
        L.gks_halo_window_get.argtypes = [vp, C.c_int, C.POINTER(HaloWindow)]
        L.gks_halo_push.argtypes = [vp, C.c_int, C.c_int, C.POINTER(HaloWindow)]
        L.gks_step_begin.argtypes = [vp, C.c_double]
        L.gks_step_begin_push.argtypes = [vp, C.c_double, C.POINTER(HaloWindow), C.POINTER(HaloWindow)]
        L.gks_step_finish.argtypes = [vp, C.c_double]
        L.gks_step_force.argtypes = [vp, C.c_double]
        L.gks_step_begin_part.argtypes = [vp, C.c_double, C.c_int]
        L.gks_step_finish_part.argtypes = [vp, C.c_double, C.c_int]
        L.gks_bulk_partial.argtypes = [vp, vp, C.POINTER(C.c_double)]
        L.gks_bulk_set_global.argtypes = [vp, vp, C.c_double]
        L.gks_ibm_pass.argtypes = [vp, C.c_int, C.c_int]
        L.gks_ibm_residual.argtypes = [vp, C.c_int, vp, C.c_int]
        L.gks_debug_eval_flux.argtypes = [vp, C.c_int, vp, vp]
        L.alm_rotor_supply.argtypes = [vp, vp, vp, C.c_double]
        L.gks_check_finite.argtypes = [vp]
        L.gks_profile_enable.argtypes = [vp, C.c_int]
        L.gks_profile_read.argtypes = [vp, _dp, C.POINTER(C.c_longlong)]
        if debug:
            L.gks_debug_set_sweep.argtypes = [vp, C.c_int]
            L.gks_debug_fp64_peak.argtypes = [vp, _dp]
            L.gks_debug_issue_probe.argtypes = [vp, _dp, C.c_int]
            L.gks_debug_trace.argtypes = [vp, C.POINTER(C.c_ulonglong)]
        L.gks_launch_count.argtypes = [vp]
        L.gks_launch_count.restype = C.c_longlong
        L.gks_last_error.argtypes = [vp]
        L.gks_last_error.restype = C.c_char_p
        L.gks_cfl_dt_noalloc.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, C.c_double, C.c_double, vp, vp]
        L.gks_halo_export_get.argtypes = [vp, C.POINTER(HaloExport)]
        L.gks_halo_export_open.argtypes = [C.POINTER(HaloExport), C.POINTER(HaloWindow), C.POINTER(vp)]
        L.gks_halo_export_close.argtypes = [vp]
        L.gks_noalloc_last_error.argtypes = []
        L.gks_noalloc_last_error.restype = C.c_char_p
        _LIBS[debug] = L
    return _LIBS[debug]


def cfl_dt_noalloc(W, dmin, RT, cfl, out, stream=None):
    """gks_cfl_dt_noalloc (include/gks.h): the CFL time step of PAPER.md:91 of the DEVICE state W (a contiguous float64
    tensor of shape (4, nz, ny, nx)) into the one-element DEVICE tensor `out`, asynchronously on `stream` (a
    torch.cuda.Stream; None = torch's current stream).  No context, no workspace: the library allocates nothing."""
    import torch
    if not (W.is_cuda and out.is_cuda and W.dtype == torch.float64 and out.dtype == torch.float64 and W.dim() == 4
            and W.shape[0] == 4 and W.is_contiguous() and out.numel() >= 1):
        raise ValueError("W: contiguous float64 CUDA tensor (4, nz, ny, nx); out: float64 CUDA tensor")
    s = stream if stream is not None else torch.cuda.current_stream(W.device)
    with torch.cuda.device(W.device):
        st = lib().gks_cfl_dt_noalloc(W.data_ptr(), int(W.shape[3]), int(W.shape[2]), int(W.shape[1]), float(dmin),
                                      float(RT), float(cfl), out.data_ptr(), s.cuda_stream)
    if st != GKS_OK:
        raise GksError(st, lib().gks_noalloc_last_error().decode())


def halo_export_open(blob, device="cuda:0"):
    """map the workspace of a sub-domain owned by another process (blob = its Gks.halo_export()) with `device` current;
    returns ([window of W^n, window of W*], mapping) - give the mapping to halo_export_close when done"""
    import torch
    e = HaloExport.from_buffer_copy(blob)
    win = (HaloWindow * 2)()
    m = C.c_void_p()
    with torch.cuda.device(device):
        st = lib().gks_halo_export_open(C.byref(e), win, C.byref(m))
    if st != GKS_OK:
        raise GksError(st, lib().gks_last_error(None).decode())
    return [win[0], win[1]], m


def halo_export_close(mapping):
    st = lib().gks_halo_export_close(mapping)
    if st != GKS_OK:
        raise GksError(st, lib().gks_last_error(None).decode())


def make_config(cfg):
    """workloads.GridConfig -> (GksConfig, keep-alive list)"""
    c = GksConfig()
    c.nx, c.ny, c.nz = cfg.n
    keep = [None if f is None else np.ascontiguousarray(f, dtype=np.float64) for f in cfg.faces]
    c.xf, c.yf, c.zf = [None if f is None else f.ctypes.data_as(_dp) for f in keep]
    c.x0, c.y0, c.z0 = cfg.origin
    c.dx, c.dy, c.dz = cfg.spacing
    c.RT, c.nu, c.rho_ref = cfg.RT, cfg.nu, cfg.rho_ref
    c.bc = (C.c_int * 6)(*cfg.bc)
    c.inflow = (C.c_double * 4)(*cfg.inflow)
    c.weno_eps = cfg.weno_eps
    return c, keep


def _ptr(x):
    """host numpy array or torch tensor (host or device) -> (address, keep-alive)"""
    if x is None:
        return None, None
    if isinstance(x, np.ndarray):
        a = np.ascontiguousarray(x, dtype=np.float64)
        return a.ctypes.data, a
    import torch
    if isinstance(x, torch.Tensor):
        assert x.dtype == torch.float64 and x.is_contiguous()
        return x.data_ptr(), x
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    return a.ctypes.data, a


class Gks:
    """One solver context on `device`.  `stream` is a torch.cuda.Stream of that device (default: a new one).
    debug=True binds libgks_b200_debug.so, which adds the hooks of include/gks_debug.h (and their workspace)."""

    def __init__(self, cfg, stream=None, device="cuda:0", debug=False):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the gas-kinetic step has no CPU fallback")
        L = lib(debug)
        self._L, self.debug = L, bool(debug)
        self._torch = torch
        self._sync_back = False
        self.device = torch.device(device)
        self.n = tuple(cfg.n)
        c, keep = make_config(cfg)
        nbytes = L.gks_workspace_bytes(C.byref(c))
        if nbytes == 0:
            h = C.c_void_p()
            st = L.gks_create(C.byref(c), None, 0, None, C.byref(h))
            raise GksError(st, L.gks_last_error(None).decode())
        # the library works on the CURRENT device (SM count, kernel attributes, launches): every call below is made
        # with this context's device current (`_c`)
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(device=self.device)
            self.workspace = torch.empty(nbytes + 256, dtype=torch.uint8, device=self.device)
            base = self.workspace.data_ptr()
            aligned = (base + 255) // 256 * 256
            self.workspace_bytes = nbytes
            self._h = C.c_void_p()
            st = L.gks_create(C.byref(c), C.c_void_p(aligned), nbytes, C.c_void_p(self.stream.cuda_stream),
                              C.byref(self._h))
        if st != GKS_OK:
            self._h = None
            raise GksError(st, L.gks_last_error(None).decode())
        self.n_ibm = 0
        self._rotor_n = 0

    # -- helpers
    def _p(self, x):
        """_ptr, plus the ordering include/gks.h asks of the caller when x is a device tensor that torch's current
        stream produced or will consume: the solver's stream waits for torch's before the call, torch's waits for
        the solver's after it (in _check), and the caching allocator keeps the block until the solver has passed."""
        p, keep = _ptr(x)
        t = self._torch
        if isinstance(x, t.Tensor) and x.is_cuda:
            cur = t.cuda.current_stream(x.device)
            if cur != self.stream:
                self.stream.wait_stream(cur)
                x.record_stream(self.stream)
                self._sync_back = True
        return p, keep

    def _check(self, st):
        if self._sync_back:
            self._sync_back = False
            self._torch.cuda.current_stream(self.device).wait_stream(self.stream)
        if st != GKS_OK:
            raise GksError(st, self._L.gks_last_error(self._h).decode())

    def _c(self, name, *args):
        """call `name`(ctx, *args) of the C ABI with this context's device current, raise on a status other than OK"""
        with self._torch.cuda.device(self.device):
            st = getattr(self._L, name)(self._h, *args)
        self._check(st)

    def close(self):
        if getattr(self, "_h", None):
            with self._torch.cuda.device(self.device):
                self._L.gks_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def shape(self):
        nx, ny, nz = self.n
        return (4, nz, ny, nx)

    def face_shape(self, d):
        nx, ny, nz = self.n
        return (4, nz + (d == 2), ny + (d == 1), nx + (d == 0))

    # -- the C ABI, same names
    def set_state(self, W):
        p, keep = self._p(W)
        self._c("gks_set_state", p)
        if isinstance(keep, np.ndarray):
            self.synchronize()      # pageable host source: be safe before the caller frees it

    def get_state(self, out=None):
        """Returns a host numpy array, or fills `out` (numpy array or torch tensor, host or device)."""
        if out is None:
            out = np.empty(self.shape)
        p, _ = self._p(out)
        self._c("gks_get_state", p)
        return out

    def step(self, dt):
        self._c("gks_step", float(dt))

    def set_body_force(self, gx, gy, gz):
        self._c("gks_set_body_force", gx, gy, gz)

    def set_bulk_flux(self, axis, target):
        self._c("gks_set_bulk_flux", int(axis), float(target))

    def alm_set_points(self, pos, force, eps):
        n = 0 if pos is None else (pos.shape[0] if hasattr(pos, "shape") else len(pos))
        pp, k1 = self._p(pos)
        pf, k2 = self._p(force)
        self._c("alm_set_points", n, pp, pf, float(eps))

    def ibm_set_points(self, pos, weights):
        n = 0 if pos is None else (pos.shape[0] if hasattr(pos, "shape") else len(pos))
        pp, k1 = self._p(pos)
        pw, k2 = self._p(weights)
        self._c("ibm_set_points", n, pp, pw)
        self.n_ibm = n

    @staticmethod
    def _rotor_struct(r):
        keep = [np.ascontiguousarray(np.asarray(x, dtype=np.float64)) for x in (r.chord, r.twist, r.alpha, r.cl, r.cd)]
        c = AlmRotor()
        c.nblades, c.npts = r.nblades, r.npts
        c.hub = (C.c_double * 3)(*r.hub)
        c.R, c.r_hub, c.omega, c.theta0, c.u_ref, c.eps = r.R, r.r_hub, r.omega, r.theta0, r.u_ref, r.eps
        c.chord, c.twist, c.alpha, c.cl, c.cd = [x.ctypes.data_as(_dp) for x in keep]
        c.npolar = len(keep[2])
        c.freestream_correction, c.tip_correction = int(r.freestream_correction), int(r.tip_correction)
        if getattr(r, "radius", None) is not None or getattr(r, "width", None) is not None:
            for name in ("radius", "width"):             # the library refuses one without the other
                v = getattr(r, name, None)
                if v is not None:
                    keep.append(np.ascontiguousarray(np.asarray(v, dtype=np.float64)))
                    setattr(c, name, keep[-1].ctypes.data_as(_dp))
        if getattr(r, "section_r", None) is not None:
            keep.append(np.ascontiguousarray(np.asarray(r.section_r, dtype=np.float64)))
            c.nsections, c.section_r = len(keep[-1]), keep[-1].ctypes.data_as(_dp)
        return c, keep

    def alm_set_rotor(self, r):
        """r: workloads.Rotor (duck-typed) or None to clear; tables are copied by the library during the call"""
        if r is None:
            self._c("alm_set_rotor", None)
            self._rotor_n = 0
            return
        c, _keep = self._rotor_struct(r)
        self._c("alm_set_rotor", C.byref(c))
        self._rotor_n = r.nblades * r.npts

    def alm_rotor_points(self, r, t, pos=None, force=None):
        """stateless front half at rotor time t on the current state; pos / force: torch CUDA tensors (n, 3) to
        fill asynchronously, or None for host numpy arrays"""
        c, _keep = self._rotor_struct(r)
        n = r.nblades * r.npts
        if pos is None:
            pos, force = np.empty((n, 3)), np.empty((n, 3))
            self._c("alm_rotor_points", C.byref(c), float(t), pos.ctypes.data, force.ctypes.data)
        else:
            assert pos.is_contiguous() and force.is_contiguous() and pos.numel() == 3 * n == force.numel()
            self._c("alm_rotor_points", C.byref(c), float(t), pos.data_ptr(), force.data_ptr())
        return pos, force

    def alm_rotor_eval(self, pos=None, force=None):
        """positions and forces of the rotor set with alm_set_rotor at the context's rotor clock, from the current
        state: host numpy arrays (synchronises), or fills the given torch CUDA tensors asynchronously"""
        n = self._rotor_n
        if pos is None:
            pos, force = np.empty((n, 3)), np.empty((n, 3))
            self._c("alm_rotor_eval", pos.ctypes.data, force.ctypes.data)
        else:
            assert pos.is_contiguous() and force.is_contiguous() and pos.numel() == 3 * n == force.numel()
            self._c("alm_rotor_eval", pos.data_ptr(), force.data_ptr())
        return pos, force

    def alm_rotor_supply(self, pos, force, x_shift=0.0):
        """sub-domain: this step's actuator points of the rotor set with alm_set_rotor (torch tensors, CUDA or CPU)"""
        assert pos.is_contiguous() and force.is_contiguous() and pos.numel() == 3 * self._rotor_n == force.numel()
        self._c("alm_rotor_supply", pos.data_ptr(), force.data_ptr(), float(x_shift))

    def step_begin(self, dt):
        self._c("gks_step_begin", float(dt))

    def step_begin_push(self, dt, to_lo=None, to_hi=None):
        """step_begin whose stage update also writes W*'s boundary planes into the neighbours' ghost layers
        (to_lo / to_hi: the HaloWindow of state 1 of the sub-domain beyond my low / high x face, or None)"""
        self._c("gks_step_begin_push", float(dt), None if to_lo is None else C.byref(to_lo),
                None if to_hi is None else C.byref(to_hi))

    def step_finish(self, dt):
        self._c("gks_step_finish", float(dt))

    def step_force(self, dt):
        self._c("gks_step_force", float(dt))

    def step_begin_part(self, dt, part):
        """part 0: interior (reads no HALO ghost), part 1: rim (HALO ghosts of W^n in place)"""
        self._c("gks_step_begin_part", float(dt), int(part))

    def step_finish_part(self, dt, part):
        self._c("gks_step_finish_part", float(dt), int(part))

    def ibm_pass(self, k, phase):
        self._c("gks_ibm_pass", int(k), int(phase))

    def ibm_residual(self, k, tensor, set=False):
        """get / set the max slip recorded by pass k (1-element float64 torch tensor, CUDA or CPU)"""
        self._c("gks_ibm_residual", int(k), tensor.data_ptr(), 1 if set else 0)

    def bulk_partial(self, out):
        """out: 1-element float64 torch tensor (CUDA or CPU) receiving this sub-domain's sum of m_axis |Omega|;
        returns the sub-domain's volume"""
        vol = C.c_double(0.0)
        self._c("gks_bulk_partial", out.data_ptr(), C.byref(vol))
        return vol.value

    def bulk_set_global(self, total, volume):
        self._c("gks_bulk_set_global", total.data_ptr(), float(volume))

    def halo_doubles(self, face):
        return int(self._L.gks_halo_doubles(self._h, int(face)))

    def halo_pack(self, which, face, buf):
        """buf: torch tensor (CUDA or CPU, float64, contiguous) of halo_doubles(face) elements"""
        assert buf.is_contiguous() and buf.numel() == self.halo_doubles(face)
        self._c("gks_halo_pack", int(which), int(face), buf.data_ptr())

    def halo_unpack(self, which, face, buf):
        assert buf.is_contiguous() and buf.numel() == self.halo_doubles(face)
        self._c("gks_halo_unpack", int(which), int(face), buf.data_ptr())

    def halo_window(self, which):
        """where a neighbour may write this context's padded state `which` directly (gks_halo_push)"""
        w = HaloWindow()
        self._c("gks_halo_window_get", int(which), C.byref(w))
        return w

    def halo_export(self):
        """this sub-domain's windows for ANOTHER process: bytes to send; the receiver calls halo_export_open"""
        e = HaloExport()
        self._c("gks_halo_export_get", C.byref(e))
        return bytes(e)

    def halo_push(self, which, face, window):
        """my 3 interior planes next to `face` straight into the neighbour's ghost planes (its `halo_window`)"""
        self._c("gks_halo_push", int(which), int(face), C.byref(window))

    def set_reconstruction(self, tangential_linear):
        self._c("gks_set_reconstruction", int(tangential_linear))

    def cfl_dt(self, cfl, out=None):
        """dt of PAPER.md:91 for the current state; out = a 1-element torch CUDA tensor keeps the call asynchronous"""
        if out is not None:
            self._c("gks_cfl_dt", float(cfl), out.data_ptr())
            return out
        host = np.zeros(1)
        self._c("gks_cfl_dt", float(cfl), host.ctypes.data)
        return float(host[0])

    def ibm_set_iterations(self, max_iter, tol=0.0):
        self._c("ibm_set_iterations", int(max_iter), float(tol))

    def ibm_set_velocities(self, vel):
        pv, k = self._p(vel)
        self._c("ibm_set_velocities", pv)

    def debug_eval_flux(self, d):
        F, dF = np.empty(self.face_shape(d)), np.empty(self.face_shape(d))
        self._c("gks_debug_eval_flux", d, F.ctypes.data, dF.ctypes.data)
        return F, dF

    def debug_set_sweep(self, mode):
        """0 = fused production kernels, 1 = unfused cross-check kernels (debug library only: include/gks_debug.h)"""
        if not self.debug:
            raise RuntimeError("gks_debug_set_sweep is not part of libgks_b200.so: create the context with debug=True")
        self._c("gks_debug_set_sweep", int(mode))

    PROF_NAMES = ("ghost", "sweep_x", "sweep_y", "sweep_z", "update", "forcing")

    def profile_enable(self, on=True):
        self._c("gks_profile_enable", int(on))

    def profile_read(self):
        """{class: (milliseconds, intervals)} accumulated since the last read; synchronises"""
        ms = (C.c_double * 6)()
        cnt = (C.c_longlong * 6)()
        self._c("gks_profile_read", ms, cnt)
        return {n: (ms[i], cnt[i]) for i, n in enumerate(self.PROF_NAMES)}

    def debug_fp64_peak(self):
        if not self.debug:
            raise RuntimeError("gks_debug_fp64_peak is not part of libgks_b200.so: create the context with debug=True")
        v = C.c_double()
        self._c("gks_debug_fp64_peak", C.byref(v))
        return v.value

    def check_finite(self):
        self._c("gks_check_finite")

    @property
    def launch_count(self):
        return self._L.gks_launch_count(self._h)

    def synchronize(self):
        self.stream.synchronize()


def fp64_peak(device="cuda:0"):
    """sustained fp64 FMA throughput [TFLOP/s] of `device`, measured by the debug library's calibration kernel on a
    throw-away context (context for bench.py's roofline; the product library does not carry the kernel)"""
    from .workloads import GridConfig
    g = Gks(GridConfig(n=(8, 8, 8), spacing=(1.0, 1.0, 1.0)), device=device, debug=True)
    try:
        return g.debug_fp64_peak()
    finally:
        g.close()


def run_workload(w, steps=None, sweep=None):
    """Run a workloads.Workload through the C ABI; returns the final state (host numpy array).
    sweep = 1 selects the unfused cross-check kernels (debug library)."""
    g = Gks(w.cfg, debug=sweep is not None)
    if sweep is not None:
        g.debug_set_sweep(sweep)
    if w.bulk_flux is not None:
        g.set_bulk_flux(*w.bulk_flux)
    if w.ibm is not None:
        g.ibm_set_points(*w.ibm)
    g.set_state(w.W0)
    for s in range(w.steps if steps is None else steps):
        if w.alm is not None:
            g.alm_set_points(*w.alm(s))
        g.step(w.dt)
    W = g.get_state()
    g.close()
    return W


class HostPipeline:
    """Independent batches with HOST buffers through `depth` solver contexts in rotation (host logic only; every step
    runs in the library's kernels).  A batch is one state in host memory that is copied to the device, advanced `steps`
    steps and copied back; the batches do not depend on one another.  Each context has its own stream, so while one
    computes, the host->device copy of the next batch and the device->host copy of the previous one run on the copy
    engines: in steady state a batch costs max(compute, copy in, copy out) instead of their sum (depth 2), and with
    depth 3 the two copies of different batches also overlap each other.

        pipe = HostPipeline(cfg, depth=2, setup=lambda g: g.ibm_set_points(pos, vol))
        for W_in, W_out in batches:                 # pinned host arrays (torch.Tensor.pin_memory) keep the copies asynchronous
            done = pipe.submit(W_in, W_out, dt)     # returns the W_out of an EARLIER batch that is now complete, or None
        pipe.drain()                                # completes the rest, in order

    W_in must stay untouched until the batch is complete; W_out is valid once submit / drain has returned it."""

    def __init__(self, cfg, depth=2, device="cuda:0", setup=None):
        if depth < 1:
            raise ValueError("depth must be >= 1")
        self.ctx = [Gks(cfg, device=device) for _ in range(depth)]
        for g in self.ctx:
            if setup is not None:
                setup(g)
        self._pending = []      # (context index, W_out) in submission order
        self._step_done = None  # event behind the last step enqueued
        self._next = 0

    def _complete_oldest(self):
        k, out = self._pending.pop(0)
        self.ctx[k].get_state(out)          # unpack + device->host copy on that context's stream, then synchronises it
        return out

    def submit(self, W_in, W_out, dt, steps=1, before_step=None):
        """enqueue set_state(W_in), `steps` x step(dt) on the next context (asynchronous), then complete the oldest
        batch if every context is busy.  before_step(g, s): optional hook called before step s (e.g. alm_set_points)."""
        k = self._next
        assert all(p[0] != k for p in self._pending)
        g = self.ctx[k]
        g.set_state(W_in)
        # the steps of successive batches run one after the other, in submission order: without this the kernels of two
        # contexts interleave on the SMs, both batches finish late and neither copy has a step left to hide behind
        # (measured on B200, 256^3: 26 ms per batch instead of 20)
        if self._step_done is not None:
            g.stream.wait_event(self._step_done)
        for s in range(steps):
            if before_step is not None:
                before_step(g, s)
            g.step(dt)
        self._step_done = g._torch.cuda.Event()
        self._step_done.record(g.stream)
        self._pending.append((k, W_out))
        self._next = (k + 1) % len(self.ctx)
        if len(self._pending) == len(self.ctx):
            return self._complete_oldest()
        return None

    def drain(self):
        done = []
        while self._pending:
            done.append(self._complete_oldest())
        return done

    @property
    def launch_count(self):
        return sum(g.launch_count for g in self.ctx)

    def close(self):
        """batches still in flight are abandoned: their streams are drained before the workspaces go"""
        for g in self.ctx:
            g.synchronize()
            g.close()
        self.ctx, self._pending = [], []
