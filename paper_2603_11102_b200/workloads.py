"""Seeded synthetic workloads shaped like the paper's cases (Table 2, :228-235).

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: only grids, initial states, point clouds and point forces (numpy, host memory).
The paper's own inputs (NREL 5 MW / NTNU blade data, DNS reference data) are not available; these
inputs stand in for them with the same shapes, sizes and structure.  Recipe: DESIGN.md §"Inputs".

All workloads: RT = 1 (c_s = 1), rho_ref = 1, Mach 0.1 => U_inf = 0.1, dt from the CFL condition
of PAPER.md:91 with CFL 0.4 evaluated on the initial state.
"""
from dataclasses import dataclass, field
from typing import Callable, Optional, Sequence, Tuple

import numpy as np

BC_PERIODIC, BC_WALL_NOSLIP, BC_WALL_SLIP, BC_INFLOW, BC_OUTFLOW_CONVECTIVE, BC_EXTRAPOLATE = range(6)

U_INF = 0.1
RT = 1.0


@dataclass
class GridConfig:
    n: Tuple[int, int, int]
    faces: Sequence[Optional[np.ndarray]] = (None, None, None)  # per-axis face coordinates or None (uniform)
    origin: Tuple[float, float, float] = (0.0, 0.0, 0.0)
    spacing: Tuple[float, float, float] = (1.0, 1.0, 1.0)
    RT: float = RT
    nu: float = 0.0
    rho_ref: float = 1.0
    bc: Tuple[int, ...] = (0, 0, 0, 0, 0, 0)
    inflow: Tuple[float, float, float, float] = (1.0, 0.0, 0.0, 0.0)
    weno_eps: float = 0.0

    def face_coords(self, a):
        if self.faces[a] is not None:
            return np.asarray(self.faces[a], dtype=np.float64)
        return self.origin[a] + self.spacing[a] * np.arange(self.n[a] + 1, dtype=np.float64)

    def centres(self, a):
        if self.faces[a] is not None:
            f = self.face_coords(a)
            return 0.5 * (f[:-1] + f[1:])
        return self.origin[a] + (np.arange(self.n[a]) + 0.5) * self.spacing[a]

    def widths(self, a):
        if self.faces[a] is not None:
            return np.diff(self.face_coords(a))
        return np.full(self.n[a], self.spacing[a])

    @property
    def cells(self):
        return self.n[0] * self.n[1] * self.n[2]


@dataclass
class Workload:
    name: str
    cfg: GridConfig
    W0: np.ndarray                    # (4, nz, ny, nx) cell averages of (rho, rhoU, rhoV, rhoW)
    dt: float
    steps: int = 10
    bulk_flux: Optional[Tuple[int, float]] = None
    ibm: Optional[Tuple[np.ndarray, np.ndarray]] = None           # (pos (n,3), V_p (n,))
    alm: Optional[Callable[[int], Tuple[np.ndarray, np.ndarray, float]]] = None  # step -> (pos, force, eps)
    notes: str = ""


@dataclass
class Rotor:
    """Input data of the on-line actuator-line rotor: geometry, tabulated polar, switches.
    Axis +x; blade b at azimuth theta0 + omega t + 2 pi b / nblades; station k at r_hub + (k+1/2)(R-r_hub)/npts."""
    nblades: int
    npts: int
    hub: Tuple[float, float, float]
    R: float
    r_hub: float
    omega: float
    theta0: float
    u_ref: float
    eps: float
    chord: np.ndarray        # (npts,)
    twist: np.ndarray        # (npts,) local twist angle gamma [rad]
    alpha: np.ndarray        # (npolar,) increasing [rad]
    cl: np.ndarray
    cd: np.ndarray
    freestream_correction: bool = False
    tip_correction: bool = False
    # optional (reading S28): explicit stations - radii and element widths, (npts,) each - and airfoil sections:
    # section_r (nsec,) increasing, then cl and cd are (nsec, npolar) and are blended linearly in r
    radius: Optional[np.ndarray] = None
    width: Optional[np.ndarray] = None
    section_r: Optional[np.ndarray] = None


def synthetic_rotor(hub, R, eps, u_ref=U_INF, tsr=7.0, nblades=3, npts=64, seed=20260314, refine=False, nsections=1,
                    **switches):
    """A seeded stand-in for the paper's blade data (NREL 5 MW / NTNU tables are not available): tapered
    chord, twist falling from root to tip, and a smooth polar with a linear range, stall and a drag bucket.
    refine: stations clustered at the root and the tip instead of evenly spaced; nsections > 1:
    that many airfoil sections between root and tip, thicker (less lift slope, more drag) towards the root."""
    rng = np.random.default_rng(seed)
    r_hub = 0.05 * R
    if refine:
        edges = r_hub + (R - r_hub) * 0.5 * (1.0 - np.cos(np.pi * np.arange(npts + 1) / npts))
        radius, width = 0.5 * (edges[:-1] + edges[1:]), np.diff(edges)
        s = (radius - r_hub) / (R - r_hub)
    else:
        radius = width = None
        s = (np.arange(npts) + 0.5) / npts
    chord = R * (0.09 - 0.055 * s) * (1.0 + 0.03 * rng.standard_normal(npts))
    twist = np.deg2rad(14.0 * (1.0 - s) ** 1.5 - 1.0 + 0.2 * rng.standard_normal(npts))
    alpha = np.deg2rad(np.linspace(-30.0, 40.0, 71))
    a_st = np.deg2rad(13.0)
    cl = 2 * np.pi * 0.9 * a_st * np.tanh(alpha / a_st) * (1.0 - 0.25 * np.clip((np.abs(alpha) - a_st) / a_st, 0, 1))
    cd = 0.008 + 0.9 * np.sin(alpha) ** 2
    section_r = None
    if nsections > 1:
        section_r = r_hub + (R - r_hub) * (np.arange(nsections) + 0.5) / nsections
        thick = np.linspace(1.0, 0.0, nsections)[:, None]           # 1 at the root section, 0 at the tip section
        cl = cl[None, :] * (1.0 - 0.35 * thick)
        cd = cd[None, :] * (1.0 + 1.5 * thick) + 0.004 * thick
    return Rotor(nblades=nblades, npts=npts, hub=tuple(hub), R=R, r_hub=r_hub, omega=tsr * u_ref / R, theta0=0.1,
                 u_ref=u_ref, eps=eps, chord=chord, twist=twist, alpha=alpha, cl=cl, cd=cd, radius=radius, width=width,
                 section_r=section_r, **switches)


# ----------------------------------------------------------------------------------------------
_G3_X = np.array([-np.sqrt(3.0 / 5.0), 0.0, np.sqrt(3.0 / 5.0)]) * 0.5   # nodes on [-1/2, 1/2]
_G3_W = np.array([5.0, 8.0, 5.0]) / 18.0


def _avg1d(fn, faces):
    """3-point Gauss cell averages of a 1-D function."""
    lo, hi = faces[:-1], faces[1:]
    c, w = 0.5 * (lo + hi), hi - lo
    return sum(wq * fn(c + xq * w) for xq, wq in zip(_G3_X, _G3_W))


def _sep_sum(cfg, terms):
    """Cell averages (tensor 3-point Gauss) of sum_t coef * fx(x) fy(y) fz(z)."""
    f = [cfg.face_coords(a) for a in range(3)]
    out = np.zeros((cfg.n[2], cfg.n[1], cfg.n[0]))
    for coef, fx, fy, fz in terms:
        out += coef * np.einsum("k,j,i->kji", _avg1d(fz, f[2]), _avg1d(fy, f[1]), _avg1d(fx, f[0]))
    return out


def cfl_dt(cfg, W0, cfl=0.4):
    """dt = CFL min(dx,dy,dz)/(|U|max + c_s) on the initial state."""
    rho = W0[0]
    umax = np.sqrt((W0[1] ** 2 + W0[2] ** 2 + W0[3] ** 2) / rho ** 2).max()
    dmin = min(cfg.widths(a).min() for a in range(3))
    return cfl * dmin / (umax + np.sqrt(cfg.RT))


# ----------------------------------------------------------------------------------------------
def taylor_green(n=32, steps=10):
    """C1 (n=32) and the 256^3 metric box M0: periodic Taylor-Green vortex on [0,2pi)^3, Re = 1600."""
    L = 2.0 * np.pi
    U0 = U_INF
    cfg = GridConfig(n=(n, n, n), spacing=(L / n,) * 3, nu=U0 * 1.0 / 1600.0, bc=(BC_PERIODIC,) * 6)
    a = U0 * U0 / (16.0 * RT)
    one = lambda x: np.ones_like(x)
    c2 = lambda x: np.cos(2 * x)
    zf = lambda z: np.cos(2 * z) + 2.0
    czf = lambda z: np.cos(z) * (np.cos(2 * z) + 2.0)
    rho = _sep_sum(cfg, [(1.0, one, one, one), (a, c2, one, zf), (a, one, c2, zf)])
    mU = _sep_sum(cfg, [(U0, np.sin, np.cos, np.cos),
                        (U0 * a, lambda x: np.sin(x) * c2(x), np.cos, czf),
                        (U0 * a, np.sin, lambda y: np.cos(y) * c2(y), czf)])
    mV = _sep_sum(cfg, [(-U0, np.cos, np.sin, np.cos),
                        (-U0 * a, lambda x: np.cos(x) * c2(x), np.sin, czf),
                        (-U0 * a, np.cos, lambda y: np.sin(y) * c2(y), czf)])
    W0 = np.stack([rho, mU, mV, np.zeros_like(rho)])
    dt = 0.4 * (L / n) / 1.1
    return Workload(f"taylor_green_{n}", cfg, W0, dt, steps,
                    notes="periodic Taylor-Green vortex, Re 1600, Mach 0.1")


def channel(n=(128, 96, 64), seed=20260311, steps=10):
    """C2: turbulent-channel-shaped box, tanh-stretched walls in y, bulk-flux forcing."""
    nx, ny, nz = n
    Ub = U_INF
    j = np.arange(ny + 1, dtype=np.float64)
    yf = np.tanh(2.0 * (2.0 * j / ny - 1.0)) / np.tanh(2.0)
    yf[0], yf[-1] = -1.0, 1.0
    cfg = GridConfig(n=n, faces=(None, yf, None), origin=(0.0, -1.0, 0.0),
                     spacing=(2 * np.pi / nx, 2.0 / ny, np.pi / nz), nu=Ub / 2800.0,
                     bc=(BC_PERIODIC, BC_PERIODIC, BC_WALL_NOSLIP, BC_WALL_NOSLIP, BC_PERIODIC, BC_PERIODIC))
    rng = np.random.Generator(np.random.PCG64(seed))
    prof = _avg1d(lambda y: 1.5 * Ub * (1.0 - y * y), yf)
    rho = np.ones((nz, ny, nx))
    pert = rng.uniform(-0.1 * Ub, 0.1 * Ub, size=(3, nz, ny, nx))
    vel = pert
    vel[0] += prof[None, :, None]
    W0 = np.concatenate([rho[None], rho[None] * vel])
    return Workload("channel", cfg, W0, cfl_dt(cfg, W0), steps, bulk_flux=(0, Ub),
                    notes="Poiseuille + 10% uniform random perturbation, tanh(2) stretching, bulk flux")


def cylinder(n=(256, 128, 64), steps=10):
    """C3: cylinder (D = 20 cells, axis along z) by IBM; inflow / convective outflow / extrapolate / periodic."""
    nx, ny, nz = n
    h = 12.8 / nx                             # D = 1 = 20 cells at full size
    D = 1.0
    cfg = GridConfig(n=n, spacing=(h, h, h), nu=U_INF * D / 3900.0,
                     bc=(BC_INFLOW, BC_OUTFLOW_CONVECTIVE, BC_EXTRAPOLATE, BC_EXTRAPOLATE,
                         BC_PERIODIC, BC_PERIODIC),
                     inflow=(1.0, U_INF, 0.0, 0.0))
    W0 = np.zeros((4, nz, ny, nx))
    W0[0] = 1.0
    W0[1] = U_INF
    nth = 64
    th = 2.0 * np.pi * np.arange(nth) / nth + 0.1
    cx, cy = 0.25 * nx * h, 0.5 * ny * h
    zc = cfg.centres(2)
    pos = np.stack([np.repeat(cx + 0.5 * D * np.cos(th), nz), np.repeat(cy + 0.5 * D * np.sin(th), nz),
                    np.tile(zc, nth)], axis=1)
    vol = np.full(len(pos), h * (np.pi * D / nth) * h)
    return Workload("cylinder", cfg, W0, cfl_dt(cfg, W0), steps, ibm=(pos, vol),
                    notes="IBM cylinder, 64 points round x one per z cell, 3-point delta")


def _rotor_forces(rng, npb, R, thrust):
    """Smooth seeded radial shapes of the axial and tangential point-force magnitudes (sum over one
    blade of axial = thrust/3)."""
    s = (np.arange(npb) + 0.5) / npb
    xi_a, xi_t = rng.uniform(-1, 1, 3), rng.uniform(-1, 1, 3)
    m = np.arange(1, 4)[:, None]
    base = s * np.sqrt(1.0 - s)
    fa = base * (1.0 + 0.1 * (xi_a[:, None] * np.sin(m * np.pi * s)).sum(0))
    ft = 0.1 * base * (1.0 + 0.1 * (xi_t[:, None] * np.sin(m * np.pi * s)).sum(0))
    scale = thrust / 3.0 / fa.sum()
    return s * R, fa * scale, ft * scale


def _alm_callable(hub, R, h, dt, seed, npb=64, tsr=7.0):
    rng = np.random.Generator(np.random.PCG64(seed))
    thrust = 0.5 * 1.0 * U_INF ** 2 * np.pi * R * R * 0.8
    r, fa, ft = _rotor_forces(rng, npb, R, thrust)
    omega = tsr * U_INF / R
    hub = np.asarray(hub, dtype=np.float64)

    def alm(step):
        pos, frc = [], []
        for b in range(3):
            psi = 2.0 * np.pi * b / 3.0 + omega * step * dt + 0.1
            er = np.array([0.0, np.cos(psi), np.sin(psi)])
            et = np.array([0.0, -np.sin(psi), np.cos(psi)])      # direction of rotation
            pos.append(hub[None, :] + r[:, None] * er[None, :])
            f = -fa[:, None] * np.array([1.0, 0.0, 0.0])[None, :] - ft[:, None] * et[None, :]
            frc.append(f)                                         # force ON THE FLUID
        return np.concatenate(pos), np.concatenate(frc), 2.0 * h
    return alm


def rotor(n=(384, 192, 192), seed=20260312, steps=10):
    """C4: three-blade rotor by ALM, R = 32 cells, 3 x 64 points, eps = 2 dx, tip-speed ratio 7."""
    nx, ny, nz = n
    h = 12.0 / nx                             # R = 1 = 32 cells at full size
    R = 1.0
    cfg = GridConfig(n=n, spacing=(h, h, h), nu=1e-5,
                     bc=(BC_INFLOW, BC_OUTFLOW_CONVECTIVE, BC_PERIODIC, BC_PERIODIC, BC_WALL_SLIP, BC_WALL_SLIP),
                     inflow=(1.0, U_INF, 0.0, 0.0))
    W0 = np.zeros((4, nz, ny, nx))
    W0[0] = 1.0
    W0[1] = U_INF
    dt = cfl_dt(cfg, W0)
    hub = (0.25 * nx * h, 0.5 * ny * h, 0.5 * nz * h)
    return Workload("rotor", cfg, W0, dt, steps, alm=_alm_callable(hub, R, h, dt, seed),
                    notes="ALM rotor, seeded smooth radial force distributions")


def _box_points(lo, hi, sp):
    """Surface lattice (spacing sp, cell-centred) of an axis-aligned box."""
    pts = []
    ax = [lo[a] + (np.arange(int(round((hi[a] - lo[a]) / sp))) + 0.5) * sp for a in range(3)]
    for a in range(3):
        b, c = [x for x in range(3) if x != a]
        B, Cc = np.meshgrid(ax[b], ax[c], indexing="ij")
        for val in (lo[a], hi[a]):
            p = np.empty((B.size, 3))
            p[:, a] = val
            p[:, b] = B.ravel()
            p[:, c] = Cc.ravel()
            pts.append(p)
    return np.concatenate(pts)


def _tower_points(cx, cy, D, z0, z1, sp):
    nth = int(round(np.pi * D / sp))
    th = 2.0 * np.pi * (np.arange(nth) + 0.5) / nth
    z = z0 + (np.arange(int(round((z1 - z0) / sp))) + 0.5) * sp
    T, Z = np.meshgrid(th, z, indexing="ij")
    return np.stack([cx + 0.5 * D * np.cos(T).ravel(), cy + 0.5 * D * np.sin(T).ravel(), Z.ravel()], axis=1)


def turbine(n=(512, 256, 256), seed=20260313, steps=10):
    """C5: ALM rotor (R = 48 cells) + IBM nacelle box (12x8x8 cells) + IBM tower (D = 6 cells, 96 cells
    high), ~20.9 k Lagrangian points on a dx/3 lattice, 5 % seeded inflow perturbation."""
    nx, ny, nz = n
    h = (512.0 / 48.0) / nx                   # R = 1 = 48 cells at full size
    hf = 1.0 / 48.0                           # full-size cell: body dimensions are given in it
    R = 1.0
    cfg = GridConfig(n=n, spacing=(h, h, h), nu=1e-5,
                     bc=(BC_INFLOW, BC_OUTFLOW_CONVECTIVE, BC_PERIODIC, BC_PERIODIC, BC_WALL_SLIP, BC_WALL_SLIP),
                     inflow=(1.0, U_INF, 0.0, 0.0))
    rng = np.random.Generator(np.random.PCG64(seed))
    W0 = np.zeros((4, nz, ny, nx))
    W0[0] = 1.0
    vel = rng.uniform(-0.05 * U_INF, 0.05 * U_INF, size=(3, nz, ny, nx))
    vel[0] += U_INF
    W0[1:] = vel
    dt = cfl_dt(cfg, W0)
    xh, yh, zh = 0.25 * nx * h, 0.5 * ny * h, (100.0 / 256.0) * nz * h
    sp = h / 3.0
    nac = _box_points((xh + 2 * hf, yh - 4 * hf, zh - 4 * hf), (xh + 14 * hf, yh + 4 * hf, zh + 4 * hf), sp)
    tow = _tower_points(xh + 8 * hf, yh, 6 * hf, 0.0, zh - 4 * hf, sp)
    pos = np.concatenate([nac, tow])
    vol = np.full(len(pos), h * sp * sp)
    return Workload("turbine", cfg, W0, dt, steps, ibm=(pos, vol),
                    alm=_alm_callable((xh, yh, zh), R, h, dt, seed + 1000),
                    notes="ALM rotor + IBM nacelle/tower, 5% seeded perturbation")


def by_name(name, small=False):
    """Workload by name; small=True gives a reduced grid of the same structure for quick parity runs."""
    if name == "C1":
        return taylor_green(32)
    if name == "M0":
        return taylor_green(256 if not small else 48)
    if name == "C2":
        return channel((128, 96, 64) if not small else (32, 24, 16))
    if name == "C3":
        return cylinder((256, 128, 64) if not small else (64, 32, 16))
    if name == "C4":
        return rotor((384, 192, 192) if not small else (96, 48, 48))
    if name == "C5":
        return turbine((512, 256, 256) if not small else (96, 48, 48))
    raise KeyError(name)
