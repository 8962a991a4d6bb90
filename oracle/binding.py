"""ctypes binding of libgks_oracle.so (TEST INFRASTRUCTURE ONLY).

Argument marshalling only; every number comes out of oracle/gks_oracle.cpp.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = None
_dp = C.POINTER(C.c_double)


class GksoConfig(C.Structure):
    _fields_ = [("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int),
                ("xf", _dp), ("yf", _dp), ("zf", _dp),
                ("x0", C.c_double), ("y0", C.c_double), ("z0", C.c_double),
                ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
                ("RT", C.c_double), ("nu", C.c_double), ("rho_ref", C.c_double),
                ("bc", C.c_int * 6), ("inflow", C.c_double * 4), ("weno_eps", C.c_double)]


class GksoRotor(C.Structure):
    _fields_ = [("nblades", C.c_int), ("npts", C.c_int), ("hub", C.c_double * 3),
                ("R", C.c_double), ("r_hub", C.c_double), ("omega", C.c_double), ("theta0", C.c_double),
                ("u_ref", C.c_double), ("eps", C.c_double), ("chord", _dp), ("twist", _dp),
                ("npolar", C.c_int), ("alpha", _dp), ("cl", _dp), ("cd", _dp),
                ("freestream_correction", C.c_int), ("tip_correction", C.c_int),
                ("radius", _dp), ("width", _dp), ("nsections", C.c_int), ("section_r", _dp)]


def build(force=False):
    """Compile the oracle with the system g++ (make -C oracle)."""
    so = os.path.join(_HERE, "libgks_oracle.so")
    src = os.path.join(_HERE, "gks_oracle.cpp")
    if force or not os.path.exists(so) or os.path.getmtime(so) < os.path.getmtime(src):
        subprocess.check_call(["make", "-C", _HERE, "-B", "libgks_oracle.so"],
                              stdout=subprocess.DEVNULL)
    return so


def lib():
    global _LIB
    if _LIB is None:
        L = C.CDLL(build())
        vp = C.c_void_p
        L.gkso_create.argtypes = [C.POINTER(GksoConfig), C.POINTER(vp)]
        L.gkso_destroy.argtypes = [vp]
        L.gkso_destroy.restype = None
        L.gkso_set_state.argtypes = [vp, _dp]
        L.gkso_get_state.argtypes = [vp, _dp]
        L.gkso_step.argtypes = [vp, C.c_double]
        L.gkso_set_body_force.argtypes = [vp, C.c_double, C.c_double, C.c_double]
        L.gkso_set_bulk_flux.argtypes = [vp, C.c_int, C.c_double]
        L.gkso_alm_set_points.argtypes = [vp, C.c_int, _dp, _dp, C.c_double]
        L.gkso_alm_set_cut.argtypes = [vp, C.c_double]
        L.gkso_ibm_set_points.argtypes = [vp, C.c_int, _dp, _dp]
        L.gkso_ibm_set_velocities.argtypes = [vp, _dp]
        L.gkso_ibm_set_iterations.argtypes = [vp, C.c_int, C.c_double]
        L.gkso_eval_flux.argtypes = [vp, C.c_int, _dp, _dp]
        L.gkso_eval_L.argtypes = [vp, _dp, _dp]
        L.gkso_get_padded.argtypes = [vp, _dp]
        L.gkso_eval_forcing.argtypes = [vp, C.c_double, _dp]
        L.gkso_ibm_interpolate.argtypes = [vp, _dp]
        L.gkso_cfl_dt.argtypes = [vp, C.c_double, _dp]
        L.gkso_alm_set_rotor.argtypes = [vp, C.POINTER(GksoRotor)]
        L.gkso_alm_rotor_eval.argtypes = [vp, _dp, _dp]
        L.gkso_last_error.restype = C.c_char_p
        L.gkso_moments.argtypes = [C.c_double, C.c_double, C.c_int, _dp]
        L.gkso_moments.restype = None
        L.gkso_micro_solve.argtypes = [C.c_double] * 4 + [_dp, _dp]
        L.gkso_micro_solve.restype = None
        L.gkso_weno5_face.argtypes = [_dp, C.c_double]
        L.gkso_weno5_face.restype = C.c_double
        L.gkso_weno5_gauss.argtypes = [_dp, C.c_double, _dp]
        L.gkso_weno5_gauss.restype = None
        L.gkso_linear5_gauss.argtypes = [_dp, _dp]
        L.gkso_linear5_gauss.restype = None
        L.gkso_set_reconstruction.argtypes = [vp, C.c_int]
        L.gkso_quartic_slope_gauss.argtypes = [_dp, _dp]
        L.gkso_quartic_slope_gauss.restype = None
        L.gkso_normal_slope.argtypes = [_dp]
        L.gkso_normal_slope.restype = C.c_double
        L.gkso_collision.argtypes = [_dp, _dp, C.c_int, C.c_double, _dp]
        L.gkso_collision.restype = None
        L.gkso_gauss_point_flux.argtypes = [_dp, _dp, C.c_int, C.c_double, C.c_double, C.c_double, _dp, _dp]
        L.gkso_gauss_point_flux.restype = None
        L.gkso_delta3.argtypes = [C.c_double]
        L.gkso_delta3.restype = C.c_double
        L.gkso_alm_kernel.argtypes = [C.c_double, C.c_double]
        L.gkso_alm_kernel.restype = C.c_double
        _LIB = L
    return _LIB


def _p(a):
    return a.ctypes.data_as(_dp)


def _arr(x, shape=None):
    a = np.ascontiguousarray(np.asarray(x, dtype=np.float64))
    if shape is not None:
        a = a.reshape(shape)
    return a


class OracleError(RuntimeError):
    pass


def _check(rc):
    if rc != 0:
        raise OracleError(lib().gkso_last_error().decode())


class Oracle:
    """One oracle context.  `cfg` is a workloads.GridConfig (duck-typed)."""

    def __init__(self, cfg):
        L = lib()
        c = GksoConfig()
        c.nx, c.ny, c.nz = cfg.n
        self._faces = [None if f is None else _arr(f) for f in cfg.faces]
        c.xf, c.yf, c.zf = [None if f is None else _p(f) for f in self._faces]
        c.x0, c.y0, c.z0 = cfg.origin
        c.dx, c.dy, c.dz = cfg.spacing
        c.RT, c.nu, c.rho_ref = cfg.RT, cfg.nu, cfg.rho_ref
        c.bc = (C.c_int * 6)(*cfg.bc)
        c.inflow = (C.c_double * 4)(*cfg.inflow)
        c.weno_eps = cfg.weno_eps
        self.n = tuple(cfg.n)
        self._h = C.c_void_p()
        _check(L.gkso_create(C.byref(c), C.byref(self._h)))
        self.n_ibm = 0

    def close(self):
        if self._h:
            lib().gkso_destroy(self._h)
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

    def set_state(self, W):
        W = _arr(W, self.shape)
        _check(lib().gkso_set_state(self._h, _p(W)))

    def get_state(self):
        W = np.empty(self.shape)
        _check(lib().gkso_get_state(self._h, _p(W)))
        return W

    def step(self, dt):
        _check(lib().gkso_step(self._h, float(dt)))

    def set_body_force(self, gx, gy, gz):
        _check(lib().gkso_set_body_force(self._h, gx, gy, gz))

    def set_bulk_flux(self, axis, target):
        _check(lib().gkso_set_bulk_flux(self._h, int(axis), float(target)))

    def alm_set_points(self, pos, force, eps):
        pos, force = _arr(pos).reshape(-1, 3), _arr(force).reshape(-1, 3)
        _check(lib().gkso_alm_set_points(self._h, len(pos), _p(pos), _p(force), float(eps)))

    def alm_set_cut(self, cut):
        _check(lib().gkso_alm_set_cut(self._h, float(cut)))

    def ibm_set_points(self, pos, weights):
        pos, weights = _arr(pos).reshape(-1, 3), _arr(weights).reshape(-1)
        _check(lib().gkso_ibm_set_points(self._h, len(pos), _p(pos), _p(weights)))
        self.n_ibm = len(pos)

    def set_reconstruction(self, tangential_linear):
        _check(lib().gkso_set_reconstruction(self._h, int(tangential_linear)))

    def ibm_set_iterations(self, max_iter, tol=0.0):
        _check(lib().gkso_ibm_set_iterations(self._h, int(max_iter), float(tol)))

    def ibm_set_velocities(self, vel):
        if vel is None:
            _check(lib().gkso_ibm_set_velocities(self._h, None))
        else:
            vel = _arr(vel).reshape(-1, 3)
            assert len(vel) == self.n_ibm
            _check(lib().gkso_ibm_set_velocities(self._h, _p(vel)))

    def face_shape(self, d):
        nx, ny, nz = self.n
        return (4, nz + (d == 2), ny + (d == 1), nx + (d == 0))

    def eval_flux(self, d):
        F, dF = np.empty(self.face_shape(d)), np.empty(self.face_shape(d))
        _check(lib().gkso_eval_flux(self._h, d, _p(F), _p(dF)))
        return F, dF

    def eval_L(self):
        L, dL = np.empty(self.shape), np.empty(self.shape)
        _check(lib().gkso_eval_L(self._h, _p(L), _p(dL)))
        return L, dL

    def get_padded(self):
        nx, ny, nz = self.n
        Wp = np.empty((4, nz + 6, ny + 6, nx + 6))
        _check(lib().gkso_get_padded(self._h, _p(Wp)))
        return Wp

    def eval_forcing(self, dt):
        nx, ny, nz = self.n
        dM = np.empty((3, nz, ny, nx))
        _check(lib().gkso_eval_forcing(self._h, float(dt), _p(dM)))
        return dM

    def alm_set_rotor(self, r):
        """r: workloads.Rotor (duck-typed) or None to clear"""
        if r is None:
            _check(lib().gkso_alm_set_rotor(self._h, None))
            self._rotor_n = 0
            return
        keep = [_arr(x) for x in (r.chord, r.twist, r.alpha, r.cl, r.cd)]
        sec_r = getattr(r, "section_r", None)
        ns = 1 if sec_r is None else len(sec_r)
        assert len(keep[0]) == r.npts and len(keep[1]) == r.npts and keep[3].size == ns * len(keep[2]) == keep[4].size
        c = GksoRotor()
        c.nblades, c.npts = r.nblades, r.npts
        c.hub = (C.c_double * 3)(*r.hub)
        c.R, c.r_hub, c.omega, c.theta0, c.u_ref, c.eps = r.R, r.r_hub, r.omega, r.theta0, r.u_ref, r.eps
        c.chord, c.twist, c.alpha, c.cl, c.cd = [_p(x) for x in keep]
        c.npolar = len(keep[2])
        c.freestream_correction, c.tip_correction = int(r.freestream_correction), int(r.tip_correction)
        if getattr(r, "radius", None) is not None:       # S28: explicit stations, section-blended polars
            keep += [_arr(r.radius), _arr(r.width)]
            assert len(keep[-1]) == r.npts == len(keep[-2])
            c.radius, c.width = _p(keep[-2]), _p(keep[-1])
        if sec_r is not None:
            keep.append(_arr(sec_r))
            c.nsections, c.section_r = ns, _p(keep[-1])
        _check(lib().gkso_alm_set_rotor(self._h, C.byref(c)))
        self._rotor_n = r.nblades * r.npts

    def alm_rotor_eval(self):
        pos, force = np.empty((self._rotor_n, 3)), np.empty((self._rotor_n, 3))
        _check(lib().gkso_alm_rotor_eval(self._h, _p(pos), _p(force)))
        return pos, force

    def cfl_dt(self, cfl):
        out = np.zeros(1)
        _check(lib().gkso_cfl_dt(self._h, float(cfl), _p(out)))
        return float(out[0])

    def ibm_interpolate(self):
        Up = np.empty((self.n_ibm, 3))
        _check(lib().gkso_ibm_interpolate(self._h, _p(Up)))
        return Up


# ---- building blocks (for the pins) ----
def moments(U, lam, nmax):
    out = np.empty(nmax + 1)
    lib().gkso_moments(U, lam, nmax, _p(out))
    return out


def micro_solve(U, V, W, lam, d):
    d, a = _arr(d), np.empty(4)
    lib().gkso_micro_solve(U, V, W, lam, _p(d), _p(a))
    return a


def weno5_face(q, eps=1e-6):
    q = _arr(q)
    return lib().gkso_weno5_face(_p(q), eps)


def weno5_gauss(q, eps=1e-6):
    q, out = _arr(q), np.empty(2)
    lib().gkso_weno5_gauss(_p(q), eps, _p(out))
    return out


def linear5_gauss(q):
    q, out = _arr(q), np.empty(2)
    lib().gkso_linear5_gauss(_p(q), _p(out))
    return out


def quartic_slope_gauss(q):
    q, out = _arr(q), np.empty(2)
    lib().gkso_quartic_slope_gauss(_p(q), _p(out))
    return out


def normal_slope(q):
    q = _arr(q)
    return lib().gkso_normal_slope(_p(q))


def collision(Ql, Qr, d, RT):
    Ql, Qr, Q0 = _arr(Ql), _arr(Qr), np.empty(4)
    lib().gkso_collision(_p(Ql), _p(Qr), d, RT, _p(Q0))
    return Q0


def gauss_point_flux(Q0, dQ, d, RT, nu, rho_ref=1.0):
    Q0, dQ = _arr(Q0), _arr(dQ, (3, 4))
    F, dF = np.empty(4), np.empty(4)
    lib().gkso_gauss_point_flux(_p(Q0), _p(dQ), d, RT, nu, rho_ref, _p(F), _p(dF))
    return F, dF


def delta3(r):
    return lib().gkso_delta3(float(r))


def alm_kernel(r, eps):
    return lib().gkso_alm_kernel(float(r), float(eps))
