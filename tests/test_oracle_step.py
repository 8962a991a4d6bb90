"""Pins of the oracle's whole step against invariants, exact solutions and closed forms (P6-P12, P14-P23).

CPU only.  Sizes are chosen so that the file runs in about two minutes.
"""
import math
import os

import numpy as np
import pytest

from oracle import binding as ob
from paper_2603_11102_b200 import workloads as wl
from paper_2603_11102_b200.workloads import GridConfig

P, NS, SL, IN, OUT, EX = range(6)


# round-off bounds of the symmetry pins (P14, P23); tests/test_gpu_physics.py widens them for the CUDA path, whose
# warps pick the series length of the collision stage per warp
TOL_SYMMETRY = 5e-15
TOL_UNIFORM = 0.0


def new_solver(cfg):
    """the solver under test: the oracle here; tests/test_gpu_physics.py swaps in the CUDA library and runs the
    same exact-solution checks on it"""
    return ob.Oracle(cfg)


def run(cfg, W0, dt, steps, setup=None):
    o = new_solver(cfg)
    if setup:
        setup(o)
    o.set_state(W0)
    for _ in range(steps):
        o.step(dt)
    W = o.get_state()
    o.close()
    return W


def const_state(n, q):
    W = np.empty((4, n[2], n[1], n[0]))
    for c in range(4):
        W[c] = q[c]
    return W


# ---------------------------------------------------------------- P6 free-stream preservation
@pytest.mark.parametrize("bc,q", [
    ((P,) * 6, (1.0, 0.1, -0.05, 0.02)),
    ((EX,) * 6, (1.0, 0.1, -0.05, 0.02)),
    ((IN, EX, P, P, SL, SL), (1.0, 0.1, 0.03, 0.0)),
    ((IN, OUT, EX, EX, P, P), (1.0, 0.1, 0.0, 0.0)),
])
def test_P6_free_stream_is_preserved_bit_for_bit(bc, q):
    n = (8, 7, 9)
    yf = np.cumsum(np.r_[0.0, np.linspace(0.5, 1.5, n[1])])        # a stretched axis as well
    cfg = GridConfig(n=n, faces=(None, yf, None), spacing=(0.3, 1.0, 0.2), nu=1e-3, bc=bc, inflow=q)
    W0 = const_state(n, q)
    W = run(cfg, W0, 0.05, 2)
    assert np.array_equal(W, W0)


# ---------------------------------------------------------------- P7 conservation
def test_P7_mass_and_momentum_conserved_on_periodic_box():
    w = wl.taylor_green(12)
    W = run(w.cfg, w.W0, w.dt, 2)
    for c in range(4):
        scale = np.abs(w.W0[c]).sum() + 1.0
        assert abs(W[c].sum() - w.W0[c].sum()) / scale < 1e-13
    assert np.abs(W - w.W0).max() > 1e-6                             # it did move


def test_P7_mass_conserved_between_noslip_walls_on_stretched_grid():
    w = wl.channel((8, 12, 6))
    cfg = w.cfg
    vol = np.einsum("k,j,i->kji", cfg.widths(2), cfg.widths(1), cfg.widths(0))
    W = run(cfg, w.W0, w.dt, 2)
    m0, m1 = (w.W0[0] * vol).sum(), (W[0] * vol).sum()
    assert abs(m1 - m0) / m0 < 1e-13
    assert np.abs(W[0] - w.W0[0]).max() > 1e-9


# ---------------------------------------------------------------- P8 order of accuracy (exact simple wave)
GL4_X = np.array([-0.8611363115940526, -0.3399810435848563, 0.3399810435848563, 0.8611363115940526]) * 0.5
GL4_W = np.array([0.3478548451374538, 0.6521451548625461, 0.6521451548625461, 0.3478548451374538]) * 0.5


def simple_wave_exact(n, t, RT=1.0, amp=0.05):
    """Cell averages (4-point Gauss per axis) of the isothermal simple wave along (1,1,1)/sqrt(3):
    U = c ln(rho) along n (Riemann invariant U - c ln rho = 0), rho constant on d xi/dt = U + c."""
    c = math.sqrt(RT)
    h = 2 * math.pi / n
    x1 = ((np.arange(n) + 0.5)[:, None] + GL4_X[None, :]).ravel() * h       # n*4 nodes per axis
    w1 = np.tile(GL4_W, n)
    Z, Y, X = np.meshgrid(x1, x1, x1, indexing="ij")
    s = X + Y + Z                                                            # phase sqrt(3) xi
    k = math.sqrt(3.0)
    rho_i = lambda s0: 1.0 + amp * np.sin(s0)
    # characteristic foot: s = s0 + k (U(rho_i(s0)) + c) t ; Newton on s0
    s0 = s - k * c * t
    for _ in range(50):
        r = rho_i(s0)
        f = s0 + k * (c * np.log(r) + c) * t - s
        df = 1.0 + k * c * t * amp * np.cos(s0) / r
        step = f / df
        s0 -= step
        if np.abs(step).max() < 1e-15:
            break
    rho = rho_i(s0)
    U = c * np.log(rho) / k                                                  # each Cartesian component
    W = np.stack([rho, rho * U, rho * U, rho * U])
    Wq = W.reshape(4, n, 4, n, 4, n, 4)
    wq = GL4_W
    return np.einsum("ckajbic,a,b,c->ckji".replace("c,a", "c,a"), Wq, wq, wq, wq) if False else \
        np.einsum("zkajbic,a,b,c->zkji", Wq, wq, wq, wq)


def simple_wave_error(n):
    cfg = GridConfig(n=(n, n, n), spacing=(2 * math.pi / n,) * 3, nu=0.0, bc=(P,) * 6)
    T = 1.0
    steps = math.ceil(T / (0.4 * (2 * math.pi / n) / 1.1))
    W = run(cfg, simple_wave_exact(n, 0.0), T / steps, steps)
    ref = simple_wave_exact(n, T)
    return np.abs(W[0] - ref[0]).mean(), np.abs(W[1:] - ref[1:]).mean()


def test_P8_order_of_accuracy_on_exact_simple_wave():
    e16, m16 = simple_wave_error(16)
    e32, m32 = simple_wave_error(32)
    order_rho = math.log2(e16 / e32)
    order_m = math.log2(m16 / m32)
    assert e32 < 2e-6
    assert order_rho >= 3.5 and order_m >= 3.5, (e16, e32, m16, m32)


# ---------------------------------------------------------------- P9 viscous decay (pins tau = mu/p, S3)
@pytest.mark.parametrize("RT,rho,rho_ref", [(1.0, 1.0, 1.0), (0.64, 1.3, 1.0), (1.5, 0.8, 1.1)])
def test_P9_shear_wave_decays_at_mu_over_rho(RT, rho, rho_ref):
    """V = V0 sin(x) exp(-(mu/rho) t) is an exact solution of the isothermal Navier-Stokes equations;
    mu = tau p = rho_ref nu whatever RT is (reading S3)."""
    n = (32, 6, 6)
    nu, V0 = 0.02, 0.01
    h = 2 * math.pi / n[0]
    cfg = GridConfig(n=n, spacing=(h, h, h), RT=RT, nu=nu, rho_ref=rho_ref, bc=(P,) * 6)
    xf = cfg.face_coords(0)
    sin_avg = (np.cos(xf[:-1]) - np.cos(xf[1:])) / h
    W0 = const_state(n, (rho, 0.0, 0.0, 0.0))
    W0[2] = rho * V0 * sin_avg[None, None, :]
    dt = 0.4 * h / (math.sqrt(RT) + V0)
    steps = 20
    W = run(cfg, W0, dt, steps)
    amp = (W[2] * sin_avg[None, None, :]).sum() / (sin_avg ** 2).sum() / (n[1] * n[2]) / (rho * V0)
    rate = -math.log(amp) / (steps * dt)
    assert rate == pytest.approx(nu * rho_ref / rho, rel=2e-3)     # WENO-JS adds < 0.2 % at 32 cells per wave
    assert np.abs(W[0] - rho).max() < 1e-9                          # density stays uniform


# ---------------------------------------------------------------- P10 acoustic speed sqrt(RT)
@pytest.mark.parametrize("RT", [1.0, 0.64])
def test_P10_acoustic_wave_travels_at_sqrt_RT(RT):
    n = (32, 6, 6)
    a = 1e-4
    cs = math.sqrt(RT)
    h = 2 * math.pi / n[0]
    cfg = GridConfig(n=n, spacing=(h, h, h), RT=RT, nu=0.0, bc=(P,) * 6)
    xf = cfg.face_coords(0)
    s_avg = (np.cos(xf[:-1]) - np.cos(xf[1:])) / h
    c_avg = (np.sin(xf[1:]) - np.sin(xf[:-1])) / h
    W0 = const_state(n, (1.0, 0.0, 0.0, 0.0))
    W0[0] += a * s_avg[None, None, :]
    W0[1] = (1.0 + a * s_avg) * (a * cs * s_avg)
    period = 2 * math.pi / cs
    steps = math.ceil(period / (0.4 * h / (cs + a)))
    W = run(cfg, W0, period / steps, steps)
    d = W[0, 0, 0, :] - 1.0
    S, Cc = (d * s_avg).sum() / (s_avg ** 2).sum(), (d * c_avg).sum() / (c_avg ** 2).sum()
    # rho - 1 = a sin(x - c t): after one nominal period the phase lag is 2 pi (1 - c/c_s)
    phase = math.atan2(-Cc, S)
    assert abs(phase) / (2 * math.pi) < 1e-3
    assert math.hypot(S, Cc) == pytest.approx(a, rel=1e-3)


# ---------------------------------------------------------------- P11 ALM integral
ALM_CUT_INTEGRAL = math.erf(3.0) - 6.0 / math.sqrt(math.pi) * math.exp(-9.0)     # = 0.99956...


@pytest.mark.parametrize("offset", [(0.0, 0.0, 0.0), (0.5, 0.5, 0.5), (0.21, 0.37, 0.48)])
def test_P11_alm_spreads_the_point_force(offset):
    n = (32, 32, 32)
    h = 0.1
    cfg = GridConfig(n=n, spacing=(h, h, h), bc=(EX,) * 6)
    o = ob.Oracle(cfg)
    o.set_state(const_state(n, (1.0, 0.1, 0.0, 0.0)))
    X = np.array([16.0, 16.0, 16.0]) * h + np.array(offset) * h
    F = np.array([-0.3, 0.2, 0.05])
    dt = 0.01
    o.alm_set_points(X[None], F[None], 2 * h)
    dM = o.eval_forcing(dt)
    total = dM.reshape(3, -1).sum(1) * h ** 3 / dt
    assert np.allclose(total / F, ALM_CUT_INTEGRAL, rtol=0, atol=1e-4)
    # touched cells all lie within 3 eps, and the kernel value there is Eq. 10
    k, j, i = np.nonzero(dM[0])
    r = np.sqrt(((i + 0.5) * h - X[0]) ** 2 + ((j + 0.5) * h - X[1]) ** 2 + ((k + 0.5) * h - X[2]) ** 2)
    assert r.max() <= 3 * 2 * h and len(r) > 0.95 * 4 / 3 * math.pi * 6 ** 3
    expect = dt * F[0] * np.exp(-(r / (2 * h)) ** 2) / ((2 * h) ** 3 * math.pi ** 1.5)
    assert np.allclose(dM[0][k, j, i], expect, rtol=1e-13)
    o.alm_set_cut(0.0)                                            # no cut: the integral is 1
    total = o.eval_forcing(dt).reshape(3, -1).sum(1) * h ** 3 / dt
    assert np.allclose(total / F, 1.0, rtol=0, atol=1e-10)
    o.close()


def test_P11_alm_wraps_on_periodic_axes_and_drops_outside_walls():
    n = (16, 16, 16)
    h = 0.1
    cfg = GridConfig(n=n, spacing=(h, h, h), bc=(P, P, P, P, SL, SL))
    o = ob.Oracle(cfg)
    o.set_state(const_state(n, (1.0, 0.0, 0.0, 0.0)))
    F = np.array([[1.0, 0.0, 0.0]])
    o.alm_set_points(np.array([[0.03, 0.8, 0.8]]), F, 2 * h)      # support crosses the periodic x face
    tot = o.eval_forcing(1.0)[0].sum() * h ** 3
    assert abs(tot - ALM_CUT_INTEGRAL) < 1e-4
    o.alm_set_points(np.array([[0.8, 0.8, 0.0]]), F, 2 * h)       # centred on the slip wall: half is lost
    tot = o.eval_forcing(1.0)[0].sum() * h ** 3
    assert abs(tot - 0.5 * ALM_CUT_INTEGRAL) < 1e-3
    o.close()


# ---------------------------------------------------------------- P12 IBM
def ibm_case(vel_field=None):
    n = (12, 10, 8)
    h = 0.25
    cfg = GridConfig(n=n, spacing=(h, h, h), bc=(EX, EX, EX, EX, P, P))
    rng = np.random.default_rng(7)
    pos = np.stack([rng.uniform(2 * h, (n[0] - 2) * h, 40), rng.uniform(2 * h, (n[1] - 2) * h, 40),
                    rng.uniform(0, n[2] * h, 40)], axis=1)        # z is periodic: any z allowed
    vol = rng.uniform(0.5, 1.5, 40) * h ** 3
    return cfg, pos, vol


def test_P12_ibm_interpolates_constants_exactly_and_conserves_impulse():
    cfg, pos, vol = ibm_case()
    n = cfg.n
    o = ob.Oracle(cfg)
    rho = 1.2
    U = np.array([0.1, -0.04, 0.07])
    W0 = const_state(n, (rho, *(rho * U)))
    o.set_state(W0)
    o.ibm_set_points(pos, vol)
    Up = o.ibm_interpolate()
    assert np.allclose(Up, U[None, :], rtol=0, atol=2e-16)
    dM = o.eval_forcing(0.1)
    h3 = 0.25 ** 3
    impulse = dM.reshape(3, -1).sum(1) * h3
    expect = (rho * (0.0 - Up) * vol[:, None]).sum(0)            # sum_p rho (v_p - U_p) V_p, v_p = 0
    assert np.allclose(impulse, expect, rtol=1e-13)
    # a fluid already moving with the body gets no force
    vp = np.tile(U, (len(pos), 1))
    o.ibm_set_velocities(vp)
    assert np.abs(o.eval_forcing(0.1)).max() < 1e-16
    o.close()


def test_P12_ibm_reads_the_unforced_field_and_rejects_outside_points():
    cfg, pos, vol = ibm_case()
    o = ob.Oracle(cfg)
    with pytest.raises(ob.OracleError):
        o.ibm_set_points(np.array([[-0.1, 1.0, 1.0]]), np.array([1.0]))
    # one step with and without an (overlapping) ALM point: the IBM increment is the same (S12)
    rng = np.random.default_rng(3)
    W0 = const_state(cfg.n, (1.0, 0.1, 0.0, 0.0)) * (1 + 0.01 * rng.standard_normal((4, 8, 10, 12)))
    o.set_state(W0)
    o.ibm_set_points(pos, vol)
    d_ibm = o.eval_forcing(0.05)
    o.alm_set_points(pos[:1], np.array([[0.1, 0.0, 0.0]]), 0.3)
    d_both = o.eval_forcing(0.05)
    o.ibm_set_points(pos[:0], vol[:0])
    d_alm = o.eval_forcing(0.05)
    assert np.allclose(d_both, d_ibm + d_alm, rtol=0, atol=1e-17)
    o.close()


# ---------------------------------------------------------------- P15 IBM multi-direct-forcing passes (S25)
def test_P15_isolated_point_contracts_by_one_minus_Vp_over_8h3_per_pass():
    """One Lagrangian point in a uniform fluid: the spread increment interpolated back at the point is
    (v - U) (V_p/h^3) (sum phi^2)^3 = (v - U) V_p/(8 h^3) (P12: sum phi^2 = 1/2 per axis), so every pass
    multiplies the slip velocity by q = 1 - V_p/(8 h^3) and the impulse after S passes is the geometric sum
    rho V_p (v - U_0) (1 - q^S)/(1 - q) (Eq. 12).  V_p = 8 h^3 removes the slip in ONE pass."""
    n, h = (10, 10, 10), 0.2
    cfg = GridConfig(n=n, spacing=(h, h, h), bc=(EX,) * 6)
    rho, U0 = 1.3, np.array([0.1, -0.05, 0.02])
    X = np.array([[1.03, 0.97, 1.11]])
    v = np.array([[0.02, 0.01, -0.03]])
    for Vp, S in [(h ** 3, 1), (h ** 3, 4), (2.5 * h ** 3, 3), (8 * h ** 3, 2)]:
        o = ob.Oracle(cfg)
        o.set_state(const_state(n, (rho, *(rho * U0))))
        o.ibm_set_points(X, np.array([Vp]))
        o.ibm_set_velocities(v)
        o.ibm_set_iterations(S)
        dM = o.eval_forcing(0.1)
        q = 1.0 - Vp / (8 * h ** 3)
        gsum = S if q == 1.0 else (1 - q ** S) / (1 - q)
        impulse = dM.reshape(3, -1).sum(1) * h ** 3
        assert np.allclose(impulse, rho * Vp * (v[0] - U0) * gsum, rtol=1e-12, atol=1e-18)
        # slip after the S passes: apply the increment and interpolate again
        W = const_state(n, (rho, *(rho * U0)))
        W[1:] += dM
        o.set_state(W)
        slip = v[0] - o.ibm_interpolate()[0]
        assert np.allclose(slip, (v[0] - U0) * q ** S, rtol=1e-11, atol=1e-17)
        o.close()


def test_P15_passes_reduce_the_slip_stop_at_the_tolerance_and_default_to_one():
    cfg, pos, vol = ibm_case()
    rng = np.random.default_rng(11)
    W0 = const_state(cfg.n, (1.0, 0.1, 0.02, -0.03)) * (1 + 0.02 * rng.standard_normal((4, 8, 10, 12)))

    def slip_after(max_iter, tol=0.0):
        o = ob.Oracle(cfg)
        o.set_state(W0)
        o.ibm_set_points(pos, vol)
        if max_iter is not None:
            o.ibm_set_iterations(max_iter, tol)
        dM = o.eval_forcing(0.05)
        W = W0.copy()
        W[1:] += dM
        o.set_state(W)
        r = np.linalg.norm(o.ibm_interpolate(), axis=1).max()      # v_p = 0
        o.close()
        return r, dM

    r = [slip_after(k)[0] for k in (1, 2, 4, 8)]
    assert r[0] > r[1] > r[2] > r[3] and r[3] < 0.5 * r[0]
    assert np.array_equal(slip_after(None)[1], slip_after(1)[1])           # default = one pass (S15)
    # tolerance: the slip before pass k is r[k-1]; with tol between r after 2 and after 1 pass exactly 2 passes run
    r1, r2 = slip_after(1)[0], slip_after(2)[0]
    tol = 0.5 * (r1 + r2)
    assert np.array_equal(slip_after(50, tol)[1], slip_after(2)[1])
    assert np.array_equal(slip_after(50, 10 * r1)[1], slip_after(1)[1])    # the first pass always runs
    with pytest.raises(ob.OracleError):
        ob.Oracle(cfg).ibm_set_iterations(0)


# ---------------------------------------------------------------- bulk flux (S16) and body force
def test_bulk_flux_restores_target_and_body_force_adds_rho_g_dt():
    w = wl.channel((8, 12, 6))
    cfg = w.cfg
    vol = np.einsum("k,j,i->kji", cfg.widths(2), cfg.widths(1), cfg.widths(0))
    W = run(cfg, w.W0, w.dt, 1, setup=lambda o: o.set_bulk_flux(0, 0.1))
    assert (W[1] * vol).sum() / vol.sum() == pytest.approx(0.1, rel=1e-13)
    Wn = run(cfg, w.W0, w.dt, 1)
    Wg = run(cfg, w.W0, w.dt, 1, setup=lambda o: o.set_body_force(0.0, 0.0, 0.3))
    assert np.allclose(Wg[3] - Wn[3], w.dt * Wn[0] * 0.3, rtol=1e-12, atol=1e-18)
    assert np.array_equal(Wg[:3], Wn[:3])


# ---------------------------------------------------------------- P14 axis symmetry
def permute_axes(W):
    """relabel (x,y,z) -> (y,z,x): new field W'(x,y,z) = old field at (z,x,y) with components rotated"""
    # array axes are (c, z, y, x); new x runs over old z, new y over old x, new z over old y
    Wn = np.transpose(W, (0, 2, 3, 1))          # (c, new z=old y, new y=old x, new x=old z)
    return np.stack([Wn[0], Wn[3], Wn[1], Wn[2]])   # new U = old W, new V = old U, new W = old V


def test_P14_one_dimensional_data_gives_the_same_result_along_every_axis():
    n, h = 12, 2 * math.pi / 12
    x = (np.arange(n) + 0.5) * h
    prof_r = 1.0 + 0.05 * np.sin(x)
    prof_u = 0.1 * np.cos(x)
    res = []
    for axis in range(3):
        shape = [1, 1, 1]
        shape[2 - axis] = n
        W0 = np.zeros((4, n, n, n))
        W0[0] = prof_r.reshape(shape)
        W0[1 + axis] = (prof_r * prof_u).reshape(shape)
        cfg = GridConfig(n=(n, n, n), spacing=(h, h, h), nu=1e-3, bc=(P,) * 6)
        W = run(cfg, W0, 0.2, 2)
        idx = [0, 0, 0]
        idx[2 - axis] = slice(None)
        res.append((W[0][tuple(idx)], W[1 + axis][tuple(idx)]))
    for axis in (1, 2):
        assert np.allclose(res[axis][0], res[0][0], rtol=0, atol=5e-16)
        assert np.allclose(res[axis][1], res[0][1], rtol=0, atol=5e-16)


def test_P14_axis_permutation_commutes_up_to_the_pass_order():
    w = wl.taylor_green(12)
    W_a = permute_axes(run(w.cfg, w.W0, w.dt, 1))
    W_b = run(w.cfg, permute_axes(w.W0), w.dt, 1)
    diff = np.abs(W_a - W_b).max()
    assert diff < 1e-6                       # only S9 (order of the tangential WENO passes) differs: O(h^5)


@pytest.mark.parametrize("lo,hi", [(NS, NS), (SL, SL), (IN, OUT), (OUT, IN), (EX, EX), (IN, EX), (NS, SL)])
@pytest.mark.parametrize("stretched", [False, True])
def test_P14_every_boundary_kind_treats_the_three_axes_alike(lo, hi, stretched):
    """data that vary along ONE axis only, between any pair of boundary kinds, on a uniform or a stretched axis: the
    same numbers whichever axis it is (to round-off: only the order of the tangential passes differs, and they act
    on constants), and exactly uniform along the two periodic axes afterwards.  This is what caught the
    zero-gradient corner ghosts of the first form of S20."""
    N = 14
    x = (np.arange(N) + 0.5) / N
    rho, un, ut = 1 + 0.02 * np.sin(2 * np.pi * x + 0.3), 0.1 + 0.01 * np.cos(2 * np.pi * x), 0.02 * np.sin(4 * np.pi * x)
    sf = np.cumsum(np.r_[0.0, np.linspace(0.8, 1.3, N)]) * 0.1
    lines = []
    for a in range(3):
        n = [6, 6, 6]
        n[a] = N
        bc = [P] * 6
        bc[2 * a], bc[2 * a + 1] = lo, hi
        inflow = [1.0, 0.0, 0.0, 0.0]
        inflow[1 + a] = 0.1
        faces = [None] * 3
        if stretched:
            faces[a] = sf
        cfg = GridConfig(n=tuple(n), faces=tuple(faces), spacing=(0.1, 0.1, 0.1), nu=2e-3, bc=tuple(bc),
                         inflow=tuple(inflow))
        shape = [1, 1, 1]
        shape[2 - a] = N
        t = (a + 1) % 3
        W0 = np.zeros((4, n[2], n[1], n[0]))
        W0[0] = rho.reshape(shape)
        W0[1 + a] = (rho * un).reshape(shape)
        W0[1 + t] = (rho * ut).reshape(shape)
        W = run(cfg, W0, 0.02, 4)
        other = tuple(i for i in range(3) if i != 2 - a)
        assert max(np.ptp(W[c], axis=other).max() for c in range(4)) <= TOL_UNIFORM
        pick = [0, 0, 0]
        pick[2 - a] = slice(None)
        pick = tuple(pick)
        lines.append(np.stack([W[0][pick], W[1 + a][pick], W[1 + t][pick], W[1 + (a + 2) % 3][pick]]))
        assert np.abs(lines[-1] - np.stack([rho, rho * un, rho * ut, 0 * rho])).max() > 1e-6      # it moved
    assert np.abs(lines[0] - lines[1]).max() < TOL_SYMMETRY and np.abs(lines[0] - lines[2]).max() < TOL_SYMMETRY


# ---------------------------------------------------------------- P16 CFL time step
def test_P16_cfl_dt_closed_forms_and_invariants():
    """dt = CFL min(dx,dy,dz)/(|U|max + sqrt(RT)): numbers worked by hand on a uniform state, the global minimum
    width on a stretched axis, the largest speed wherever it sits, linear in CFL, Galilean shift of |U|max"""
    n = (6, 7, 8)
    yf = np.array([0.0, 0.3, 0.5, 0.62, 0.7, 0.9, 1.3, 1.8])            # smallest width 0.08
    cfg = GridConfig(n=n, faces=(None, yf, None), spacing=(0.25, 1.0, 0.1), RT=0.64, bc=(EX,) * 6)
    o = ob.Oracle(cfg)
    W = const_state(n, (2.0, 2.0 * 0.3, 2.0 * -0.4, 0.0))               # |U| = 0.5, c = 0.8
    o.set_state(W)
    assert o.cfl_dt(0.4) == pytest.approx(0.4 * 0.08 / (0.5 + 0.8), rel=1e-15)
    assert o.cfl_dt(0.8) == pytest.approx(2 * o.cfl_dt(0.4), rel=1e-15)
    W[:, 5, 3, 2] = (0.5, 0.0, 0.0, 0.5 * 1.2)                          # one fast cell: |U| = 1.2
    o.set_state(W)
    assert o.cfl_dt(0.4) == pytest.approx(0.4 * 0.08 / (1.2 + 0.8), rel=1e-15)
    o.close()
    cfg2 = GridConfig(n=n, spacing=(0.25, 0.2, 0.05), RT=1.0, bc=(EX,) * 6)   # uniform grid: dz is the smallest
    o = ob.Oracle(cfg2)
    o.set_state(const_state(n, (1.0, 0.0, 0.0, 0.0)))
    assert o.cfl_dt(1.0) == pytest.approx(0.05, rel=1e-15)             # fluid at rest: dt = dz / c_s
    with pytest.raises(ob.OracleError):
        o.cfl_dt(0.0)
    o.close()
    # the input recipe's dt (workloads.cfl_dt, numpy) is the same number
    w = wl.by_name("C2", small=True)
    o = ob.Oracle(w.cfg)
    o.set_state(w.W0)
    assert o.cfl_dt(0.4) == pytest.approx(w.dt, rel=1e-14)
    o.close()


# ---------------------------------------------------------------- P17 actuator-line front half (S26, S27)
def rotor_case(**kw):
    n, h = (24, 24, 24), 0.125
    cfg = GridConfig(n=n, spacing=(h, h, h), bc=(EX, EX, P, P, EX, EX))
    r = wl.synthetic_rotor(hub=(1.5, 1.5, 1.5), R=1.0, eps=2 * h, npts=16, **kw)
    return cfg, r


def rel_velocity(r, pos, U):
    """blade-relative velocity vectors of the points in a uniform flow U (geometry only: U - omega x r)"""
    d = pos - np.asarray(r.hub)
    v_blade = r.omega * np.stack([np.zeros(len(d)), -d[:, 2], d[:, 1]], axis=1)     # omega e_x x d
    return np.asarray(U)[None, :] - v_blade


def test_P17_geometry_and_trilinear_sampling():
    cfg, r = rotor_case()
    o = ob.Oracle(cfg)
    o.set_state(const_state(cfg.n, (1.0, 0.1, 0.0, 0.0)))
    o.alm_set_rotor(r)
    pos, _ = o.alm_rotor_eval()
    d = pos - np.asarray(r.hub)
    w = (r.R - r.r_hub) / r.npts
    rad = np.hypot(d[:, 1], d[:, 2]).reshape(r.nblades, r.npts)
    assert np.allclose(d[:, 0], 0) and np.allclose(rad, r.r_hub + (np.arange(r.npts) + 0.5) * w, rtol=1e-14)
    az = np.arctan2(d[:, 2], d[:, 1]).reshape(r.nblades, r.npts)
    assert np.allclose(az[0], r.theta0) and np.allclose(np.diff(np.unwrap(az[:, 0])), 2 * np.pi / r.nblades)
    # the clock advances by dt per step: after a step the azimuth has turned by omega dt
    o.step(0.01)
    pos2, _ = o.alm_rotor_eval()
    az2 = np.arctan2(pos2[0, 2] - r.hub[2], pos2[0, 1] - r.hub[1])
    assert az2 - r.theta0 == pytest.approx(r.omega * 0.01, rel=1e-12)
    o.close()
    # sampling is exact for a velocity field that is trilinear in (x, y, z): force with a pure-drag polar is
    # 1/2 rho c w cd |U_rel| U_rel with U_rel from the exact field at the point
    x, y, z = [cfg.centres(a) for a in range(3)]
    Z, Y, X = np.meshgrid(z, y, x, indexing="ij")
    U = np.stack([0.1 + 0.02 * X + 0.01 * Y * Z, 0.03 * X * Y - 0.01, 0.02 * Z + 0.01 * X * Y * Z])
    rho = 1.1
    W = np.concatenate([np.full((1,) + X.shape, rho), rho * U])
    r2 = wl.synthetic_rotor(hub=(1.5, 1.5, 1.5), R=0.8, eps=0.25, npts=12)
    r2.cl = np.zeros_like(r2.cl)
    r2.cd = np.full_like(r2.cd, 0.7)
    o = ob.Oracle(GridConfig(n=cfg.n, spacing=cfg.spacing, bc=(EX,) * 6))
    o.set_state(W)
    o.alm_set_rotor(r2)
    pos, F = o.alm_rotor_eval()
    px, py, pz = pos.T
    Uex = np.stack([0.1 + 0.02 * px + 0.01 * py * pz, 0.03 * px * py - 0.01, 0.02 * pz + 0.01 * px * py * pz], axis=1)
    d = pos - np.asarray(r2.hub)
    rad = np.hypot(d[:, 1], d[:, 2])
    et = np.stack([np.zeros(len(d)), -d[:, 2] / rad, d[:, 1] / rad], axis=1)
    # the blade element only sees the axial and rotational components (U^2D); the radial one is dropped
    U2d = Uex[:, :1] * np.array([[1.0, 0, 0]]) + (Uex * et).sum(1, keepdims=True) * et
    Urel = U2d - r2.omega * rad[:, None] * et
    w2 = (r2.R - r2.r_hub) / r2.npts
    drag_on_blade = 0.5 * rho * np.tile(r2.chord, r2.nblades)[:, None] * w2 * 0.7 * np.linalg.norm(Urel, axis=1)[:, None] * Urel
    assert np.allclose(F, -drag_on_blade, rtol=1e-12, atol=1e-18)
    o.close()


def test_P17_lift_is_normal_and_drag_parallel_to_the_relative_flow():
    """two-dimensional airfoil theory (Eq. 9): with C_D = 0 the force is perpendicular to U_rel and
    has magnitude 1/2 rho c w C_L |U_rel|^2; with C_L = 0 it is parallel; thrust on the fluid points upstream
    and the tangential reaction opposes the rotation for an attached-flow blade"""
    cfg, r = rotor_case()
    rho, U = 1.2, np.array([0.1, 0.0, 0.0])
    w = (r.R - r.r_hub) / r.npts
    chord = np.tile(r.chord, r.nblades)
    o = ob.Oracle(cfg)
    o.set_state(const_state(cfg.n, (rho, *(rho * U))))
    lift_only = wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, npts=r.npts)
    lift_only.cd = np.zeros_like(r.cd)
    o.alm_set_rotor(lift_only)
    pos, F = o.alm_rotor_eval()
    Urel = rel_velocity(r, pos, U)
    assert np.abs((F * Urel).sum(1)).max() <= 1e-15 * np.abs(F).max() * np.abs(Urel).max()
    d = pos - np.asarray(r.hub)
    rad = np.hypot(d[:, 1], d[:, 2])
    phi = np.arctan2(U[0], r.omega * rad)                      # uniform axial wind: U_theta = 0
    cl = np.interp(phi - np.tile(r.twist, r.nblades), r.alpha, lift_only.cl)
    assert np.allclose(np.linalg.norm(F, axis=1), 0.5 * rho * chord * w * np.abs(cl) * (Urel ** 2).sum(1), rtol=1e-12)
    assert (F[:, 0] < 0).all()                                 # the fluid is pushed upstream (thrust reaction)
    et = np.stack([np.zeros(len(d)), -d[:, 2] / rad, d[:, 1] / rad], axis=1)
    assert ((F * et).sum(1) < 0).all()                         # and against the rotation (torque reaction)
    drag_only = wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, npts=r.npts)
    drag_only.cl = np.zeros_like(r.cl)
    o.alm_set_rotor(drag_only)
    pos, F = o.alm_rotor_eval()
    cross = np.cross(F, rel_velocity(r, pos, U))
    assert np.abs(cross).max() <= 1e-15 * np.abs(F).max() * np.abs(Urel).max()
    assert ((F * rel_velocity(r, pos, U)).sum(1) < 0).all()    # reaction of a drag: against U_rel
    o.close()


def test_P17_corrections():
    """free-stream correction: with a constant C_D and a constant chord the forces equal those of
    the uncorrected model in a flow scaled by 1/(1 - C_D c/(4 sqrt(pi) eps)); tip correction (Eq. 14): factors in
    (0, 1], -> 1 towards the root, -> 0 at the tip, axial and tangential differ, a no-op when switched off"""
    cfg, r = rotor_case()
    rho, U = 1.0, np.array([0.1, 0.004, -0.003])
    mk = lambda **kw: wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, npts=r.npts, **kw)
    base, corr = mk(), mk(freestream_correction=True)
    for q in (base, corr):
        q.chord = np.full(r.npts, 0.08)
        q.cd = np.full_like(r.cd, 0.3)
    k = 1.0 / (1.0 - 0.3 * 0.08 / (4 * math.sqrt(math.pi) * r.eps))
    o = ob.Oracle(cfg)
    o.set_state(const_state(cfg.n, (rho, *(rho * U))))
    o.alm_set_rotor(corr)
    F_corr = o.alm_rotor_eval()[1]
    o.set_state(const_state(cfg.n, (rho, *(rho * U * k))))
    o.alm_set_rotor(base)
    F_scaled = o.alm_rotor_eval()[1]
    assert k > 1.01 and np.allclose(F_corr, F_scaled, rtol=1e-12, atol=1e-18)
    # tip correction
    o.set_state(const_state(cfg.n, (rho, 0.1, 0.0, 0.0)))
    fine = dict(npts=200)
    o.alm_set_rotor(wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, **fine))
    pos, F0 = o.alm_rotor_eval()
    o.alm_set_rotor(wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, tip_correction=True, **fine))
    F1 = o.alm_rotor_eval()[1]
    d = pos - np.asarray(r.hub)
    rad = np.hypot(d[:, 1], d[:, 2])[:200]
    et = np.stack([np.zeros(200), -d[:200, 2] / rad, d[:200, 1] / rad], axis=1)
    f_ax = F1[:200, 0] / F0[:200, 0]
    f_tan = (F1[:200] * et).sum(1) / (F0[:200] * et).sum(1)
    for f in (f_ax, f_tan):
        assert (f > 0).all() and (f <= 1.0).all() and (np.diff(f[rad > 0.3]) < 0).all()
        assert f[rad < 0.2].min() > 0.99 and f[-1] < 0.2
    assert np.abs(f_ax - f_tan).max() > 1e-3
    # worked value: N = 3, lambda = 7, r = 0.9 R, phi from a uniform wind: f = 2/pi acos(exp(-g1 N (R-r)/(2 r sin phi)))
    # with the constants the paper prints (tests/golden/paper_constants.txt), axial and tangential
    gold = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                gold[line.split()[0]] = float(line.split()[1])
    i = np.argmin(np.abs(rad - 0.9))
    sphi = math.sin(math.atan2(0.1, 0.7 * rad[i]))
    for f_meas, kind in ((f_ax, "axial"), (f_tan, "tangential")):
        g1 = math.exp(-gold["tip_c1_" + kind] * (3 * 7.0 - gold["tip_c2_" + kind])) + 0.1
        want = 2 / math.pi * math.acos(math.exp(-g1 * 3 * (1.0 - rad[i]) / (2 * rad[i] * sphi)))
        assert f_meas[i] == pytest.approx(want, rel=1e-10)
    with pytest.raises(ob.OracleError):
        bad = mk(tip_correction=True)
        bad.u_ref = 0.0
        o.alm_set_rotor(bad)
    o.close()


def test_P17_rotor_step_equals_prescribed_points_step():
    """a step with the on-line rotor = a step with alm_set_points fed with the forces the rotor evaluates on the
    un-forced field (S12, S26): here checked through the linearity of the forcing, increment by increment"""
    cfg, r = rotor_case()
    rng = np.random.default_rng(5)
    W0 = const_state(cfg.n, (1.0, 0.1, 0.0, 0.0)) * (1 + 0.01 * rng.standard_normal((4,) + cfg.n[::-1]))
    o = ob.Oracle(cfg)
    o.set_state(W0)
    o.alm_set_rotor(r)
    pos, F = o.alm_rotor_eval()
    dM_rotor = o.eval_forcing(0.02)
    o.alm_set_rotor(None)
    o.alm_set_points(pos, F, r.eps)
    assert np.array_equal(dM_rotor, o.eval_forcing(0.02))
    assert np.abs(dM_rotor).max() > 0
    o.close()


# ---------------------------------------------------------------- P18 linear-weight tangential variant (f4)
def test_P18_linear_tangential_variant():
    """the variant's operator is the quartic through the five averages: SURVEY's Gauss-point value row, exact for
    cell averages of polynomials up to degree 4 whatever their smoothness indicators, the limit eps -> large of
    WENO-JS; the step keeps the free stream, conserves, is fourth-order on the simple wave and equals the WENO
    step on data that vary along one axis only up to the normal reconstruction"""
    s3 = math.sqrt(3.0)
    row = np.array([-1 / 4320 + 7 * s3 / 432, 1 / 1080 - 25 * s3 / 216, 719 / 720, 1 / 1080 + 25 * s3 / 216,
                    -1 / 4320 - 7 * s3 / 432])
    rng = np.random.default_rng(2)
    for _ in range(5):
        q = rng.standard_normal(5)
        vm, vp = ob.linear5_gauss(q)
        assert vp == pytest.approx(row @ q, rel=1e-13, abs=1e-15) and vm == pytest.approx(row[::-1] @ q, rel=1e-13, abs=1e-15)
        assert np.allclose(ob.weno5_gauss(q, eps=1e12), [vm, vp], rtol=1e-10)
    # exact on cell averages of a quartic with an O(1) kink-free but steep profile (nonlinear weights would bias it)
    poly = np.polynomial.Polynomial(rng.standard_normal(5) * [1, 3, 5, 7, 9])
    A = poly.integ()
    q = np.array([A(m + 0.5) - A(m - 0.5) for m in range(-2, 3)])
    vm, vp = ob.linear5_gauss(q)
    assert vp == pytest.approx(poly(s3 / 6), rel=1e-12) and vm == pytest.approx(poly(-s3 / 6), rel=1e-12)
    assert abs(ob.weno5_gauss(q)[1] - poly(s3 / 6)) > 1e-6 * abs(poly(s3 / 6))
    lin = lambda o: o.set_reconstruction(1)
    # free stream and conservation
    n = (8, 7, 6)
    cfg = GridConfig(n=n, spacing=(0.1, 0.12, 0.09), nu=1e-3, bc=(P,) * 6)
    W0 = const_state(n, (1.1, 0.11, -0.05, 0.02))
    assert np.array_equal(run(cfg, W0, 0.02, 2, setup=lin), W0)
    W0 = W0 * (1 + 0.01 * rng.standard_normal(W0.shape))
    W = run(cfg, W0, 0.02, 1, setup=lin)
    assert np.allclose(W.reshape(4, -1).sum(1), W0.reshape(4, -1).sum(1), rtol=1e-13, atol=1e-13)
    assert not np.array_equal(W, run(cfg, W0, 0.02, 1))                   # it IS a different scheme
    # order of accuracy on the exact simple wave (P8's solution)
    def err(nn):
        c = GridConfig(n=(nn, nn, nn), spacing=(2 * math.pi / nn,) * 3, nu=0.0, bc=(P,) * 6)
        steps = math.ceil(1.0 / (0.4 * (2 * math.pi / nn) / 1.1))
        Wn = run(c, simple_wave_exact(nn, 0.0), 1.0 / steps, steps, setup=lin)
        return np.abs(Wn[0] - simple_wave_exact(nn, 1.0)[0]).mean()
    e16, e32 = err(16), err(32)
    assert math.log2(e16 / e32) >= 3.5 and e32 < 2e-6
    with pytest.raises(ob.OracleError):
        ob.Oracle(cfg).set_reconstruction(2)


# ---------------------------------------------------------------- P19 stretched-grid metrics (reading S10)
def exp_faces(N, ratio=3.0):
    """smooth one-sided stretching of [0, 1]: the last cell is `ratio` times as wide as the first; one-sided, so that
    a first-order metric error cannot cancel between the two ends"""
    b = math.log(ratio)
    return (np.exp(b * np.arange(N + 1) / N) - 1.0) / (math.exp(b) - 1.0)


def couette_stress_errors(N, s, m, nu=0.05, a=0.02):
    """rho = 1, velocity component m = a x_s (plane Couette flow), axis s stretched.  Navier-Stokes: the flux of
    momentum m through faces normal to s and the flux of momentum s through faces normal to m are both -mu a,
    everywhere.  Returns the two relative errors away from the (non-linear) boundary ghosts."""
    sf = exp_faces(N)
    n = [6, 6, 6]
    n[s] = N
    faces = [None, None, None]
    faces[s] = sf
    bc = [P] * 6
    bc[2 * s] = bc[2 * s + 1] = EX
    cfg = GridConfig(n=tuple(n), faces=tuple(faces), spacing=(0.1, 0.1, 0.1), RT=1.0, nu=nu, bc=tuple(bc))
    W0 = const_state(n, (1.0, 0.0, 0.0, 0.0))
    shape = [1, 1, 1]
    shape[2 - s] = N
    W0[1 + m] = a * (0.5 * (sf[1:] + sf[:-1])).reshape(shape)      # the cell average of a linear profile
    o = new_solver(cfg)
    o.set_state(W0)
    Fs, _ = o.eval_flux(s)
    Fm, _ = o.eval_flux(m)
    o.close()
    core = [slice(None)] * 3
    core[2 - s] = slice(4, N - 4)
    core = tuple(core)
    return np.abs(Fs[1 + m][core] / (-nu * a) - 1).max(), np.abs(Fm[1 + s][core] / (-nu * a) - 1).max()


@pytest.mark.parametrize("s,m", [(0, 1), (0, 2), (1, 0), (1, 2), (2, 0), (2, 1)])
def test_P19_couette_stress_on_a_stretched_axis_is_second_order(s, m):
    """S10 divides index-space slopes by the centre distance (normal) or the cell width (tangential, both passes).
    Either is a second-order approximation of the metric; taking the other one is first order (3 % at 16 cells).
    The six (s, m) pairs reach the normal slope of every sweep and the t1 and t2 slopes of every sweep."""
    n16, t16 = couette_stress_errors(16, s, m)
    n32, t32 = couette_stress_errors(32, s, m)
    assert n32 < 1.5e-4 and t32 < 1.5e-4
    assert n16 / n32 > 3.5 and t16 / t32 > 3.5


def vortex_decay_rate_error(N, nu=0.05, U0=0.01, T=0.1):
    """u = U0 sin(kx) cos(ky), v = -U0 cos(kx) sin(ky) between slip walls at y = 0, 1 (k = pi) decays at 2 nu k^2
    (incompressible Navier-Stokes; the compressible correction is O(Ma^2) = 1e-4); x uniform, y stretched"""
    k = math.pi
    yf, xf = exp_faces(N), 2.0 * np.arange(N + 1) / N
    avg = lambda F, f: (F(f[1:]) - F(f[:-1])) / np.diff(f)
    sx, cx = avg(lambda x: -np.cos(k * x) / k, xf), avg(lambda x: np.sin(k * x) / k, xf)
    sy, cy = avg(lambda y: -np.cos(k * y) / k, yf), avg(lambda y: np.sin(k * y) / k, yf)
    cfg = GridConfig(n=(N, N, 6), faces=(None, yf, None), spacing=(2.0 / N, 1.0, 0.1), RT=1.0, nu=nu,
                     bc=(P, P, SL, SL, P, P))
    W0 = const_state((N, N, 6), (1.0, 0.0, 0.0, 0.0))
    W0[1] = U0 * (cy[:, None] * sx[None, :])[None]
    W0[2] = -U0 * (sy[:, None] * cx[None, :])[None]
    hmin = min(np.diff(yf).min(), 2.0 / N)
    steps = math.ceil(T / min(0.3 * hmin, 0.15 * hmin ** 2 / nu))
    W = run(cfg, W0, T / steps, steps)
    wy, mode = np.diff(yf), cy[:, None] * sx[None, :]
    amp = (W[1].mean(0) * mode * wy[:, None]).sum() / (mode ** 2 * wy[:, None]).sum() / U0
    return -math.log(amp) / T / (2 * nu * k * k) - 1.0


def test_P19_vortex_between_slip_walls_on_a_stretched_axis_decays_at_2_nu_k2():
    """the whole step on a stretched axis: normal slope / centre distance, flux difference / cell width, mirrored
    ghost widths at the walls.  A metric that is off by one cell is first order: 1.4 % at 32 cells"""
    e16, e32 = vortex_decay_rate_error(16), vortex_decay_rate_error(32)
    assert abs(e32) < 1.5e-3 and abs(e16 / e32) > 3.0


# ---------------------------------------------------------------- P20 inflow (reading S19): the piston problem
@pytest.mark.parametrize("axis,side", [(0, 0), (1, 1)])
def test_P20_impulsive_inflow_drives_the_rankine_hugoniot_shock(axis, side):
    """Gas at rest, inflow face switched on at U_b = 0.1 c_s: a piston.  Exact solution of the isothermal Euler
    equations: a shock with (r - 1)^2 = r M^2, r = rho_1 / rho_0, M = U_b / c_s, speed r U_b / (r - 1); behind it
    rho_1 and U_b; the mass that entered is rho_1 U_b t.  The ghost density of S19 (outgoing invariant) meets all
    three; its sign flipped, a Dirichlet density or a zero-gradient density each miss at least one by > 5x."""
    N, M, RT, T = 200, 0.1, 1.0, 0.8
    cs = math.sqrt(RT)
    Ub, h = M * cs, 2.0 / N
    n = [6, 6, 6]
    n[axis] = N
    bc = [P] * 6
    bc[2 * axis + side], bc[2 * axis + 1 - side] = IN, EX
    inflow = [1.0, 0.0, 0.0, 0.0]
    inflow[1 + axis] = Ub if side == 0 else -Ub
    cfg = GridConfig(n=tuple(n), spacing=(h, h, h), RT=RT, nu=0.0, bc=tuple(bc), inflow=tuple(inflow))
    steps = math.ceil(T / (0.3 * h / (cs + Ub)))
    W = run(cfg, const_state(n, (1.0, 0.0, 0.0, 0.0)), T / steps, steps)
    line = [0, 0, 0]
    line[2 - axis] = slice(None)
    rho, mom = W[0][tuple(line)], W[1 + axis][tuple(line)]
    if side == 1:
        rho, mom = rho[::-1], -mom[::-1]
    r = 1 + M * M / 2 + M * math.sqrt(1 + M * M / 4)
    assert (r - 1) ** 2 == pytest.approx(r * M * M, rel=1e-12)
    speed = r * Ub / (r - 1)
    x = (np.arange(N) + 0.5) * h
    plateau = (x > 0.1) & (x < speed * T - 0.15)
    assert plateau.sum() > 50
    assert np.abs(rho[plateau] - r).max() < 3e-4                       # the jump itself is 0.105
    assert np.abs(mom[plateau] / rho[plateau] - Ub).max() < 2e-3 * Ub
    assert (rho - 1).sum() * h == pytest.approx(r * Ub * T, rel=1e-3)  # mass through the inflow face
    ahead = x > speed * T + 0.15
    assert np.abs(rho[ahead] - 1).max() < 1e-5                          # nothing outruns the shock


# ---------------------------------------------------------------- P21 convective outflow (reading S20)
@pytest.mark.parametrize("axis,side", [(0, 1), (1, 0), (2, 1)])
def test_P21_vortical_pulse_leaves_through_the_convective_outflow(axis, side):
    """rho = 1, normal velocity U0, a transverse velocity A exp(-(x - x0 - U0 t)^2 / 2 sigma^2): an exact solution of
    the isothermal Euler equations (rho and the normal velocity stay uniform, the transverse momentum is advected).
    The pulse crosses the outflow face at t = 4/3; the interior must follow the exact solution while it leaves and
    be quiet afterwards.  S20's ghost update does (0.9 % of A at 4 cells per sigma); frozen ghosts give 18 % and more,
    the sign of C flipped blows up, C doubled gives 3.4 %."""
    N, U0, A, sig, x0 = 40, 0.3, 0.01, 0.1, 0.6
    h = 1.0 / N
    t_axis = (axis + 1) % 3                     # direction of the transverse velocity
    n = [6, 6, 6]
    n[axis] = N
    bc = [P] * 6
    bc[2 * axis + side], bc[2 * axis + 1 - side] = OUT, IN
    inflow = [1.0, 0.0, 0.0, 0.0]
    inflow[1 + axis] = U0 if side == 1 else -U0
    cfg = GridConfig(n=tuple(n), spacing=(h, h, h), RT=1.0, nu=0.0, bc=tuple(bc), inflow=tuple(inflow))
    xf = np.arange(N + 1) * h

    def exact(t):                               # cell averages, in the coordinate that runs towards the outflow
        F = A * sig * math.sqrt(math.pi / 2) * np.array([math.erf((v - x0 - U0 * t) / (sig * math.sqrt(2))) for v in xf])
        return np.diff(F) / h

    def along(v):                               # lay a 1-D profile along `axis`, flipped if the flow runs down the axis
        shape = [1, 1, 1]
        shape[2 - axis] = N
        return (v if side == 1 else v[::-1]).reshape(shape)

    W0 = const_state(n, inflow)
    W0[1 + t_axis] = along(exact(0.0))
    o = new_solver(cfg)
    o.set_state(W0)
    t, dt = 0.0, 0.3 * h / (1.0 + U0)
    for T in (1.1, 4.0 / 3.0, 1.6, 2.8):
        steps = math.ceil((T - t) / dt - 1e-9)
        for _ in range(steps):
            o.step((T - t) / steps)
        t = T
        W = o.get_state()
        err = np.abs(W[1 + t_axis] - along(exact(T))).max() / A
        assert err < 0.015, T
        assert np.abs(W[0] - 1).max() < 1e-12 and np.abs(W[1 + axis] - inflow[1 + axis]).max() < 1e-12
    o.close()
    assert np.abs(exact(2.8)).max() < 1e-4 * A   # by then the pulse is gone


# ---------------------------------------------------------------- P22 no-slip wall (reading S17) and the uniform body force
def wall_channel(N, axis):
    """6 x N x 6 cells (N along `axis`) between no-slip walls at 0 and 1, flow along the next axis"""
    h = 1.0 / N
    n = [6, 6, 6]
    n[axis] = N
    bc = [P] * 6
    bc[2 * axis] = bc[2 * axis + 1] = NS
    shape = [1, 1, 1]
    shape[2 - axis] = N
    other = tuple(i for i in range(3) if i != 2 - axis)
    return h, n, tuple(bc), (axis + 1) % 3, shape, other


@pytest.mark.parametrize("axis", [1, 2])
def test_P22_shear_mode_between_noslip_walls_decays_at_nu_k2(axis):
    """u = U0 sin(pi y) exp(-nu pi^2 t) vanishes on both walls: exact.  The mirror ghosts of S17 put the wall on the
    face to second order; a slip wall or a wall half a cell off would change the rate by O(1) / O(h)."""
    nu, U0, T, k = 0.05, 0.01, 0.2, math.pi
    err = []
    for N in (12, 24):
        h, n, bc, m, shape, other = wall_channel(N, axis)
        yf = np.arange(N + 1) * h
        savg = (np.cos(k * yf[:-1]) - np.cos(k * yf[1:])) / (k * h)
        cfg = GridConfig(n=tuple(n), spacing=(h, h, h), RT=1.0, nu=nu, bc=bc)
        W0 = const_state(n, (1.0, 0.0, 0.0, 0.0))
        W0[1 + m] = U0 * savg.reshape(shape)
        steps = math.ceil(T / min(0.3 * h, 0.15 * h * h / nu))
        u = run(cfg, W0, T / steps, steps)[1 + m].mean(axis=other)
        amp = (u * savg).sum() / (savg ** 2).sum() / U0
        assert np.abs(u / U0 - amp * savg).max() < 1e-6            # it stays the mode it was
        err.append(-math.log(amp) / T / (nu * k * k) - 1.0)
    assert abs(err[1]) < 2e-3 and err[0] / err[1] > 3.5


def test_P22_poiseuille_profile_is_steady_under_the_body_force():
    """g y (1 - y) / (2 nu) between no-slip walls balances the uniform acceleration g exactly (Navier-Stokes); started
    from its cell averages the step must keep it: the drift after half a viscous time is second order in h"""
    nu, g = 0.05, 0.01
    drift = []
    for N in (12, 24):
        h, n, bc, m, shape, other = wall_channel(N, 1)
        yf = np.arange(N + 1) * h
        uavg = np.diff(g / (2 * nu) * (yf ** 2 / 2 - yf ** 3 / 3)) / h
        cfg = GridConfig(n=tuple(n), spacing=(h, h, h), RT=1.0, nu=nu, bc=bc)
        W0 = const_state(n, (1.0, 0.0, 0.0, 0.0))
        W0[1 + m] = uavg.reshape(shape)
        acc = [0.0, 0.0, 0.0]
        acc[m] = g
        T = 0.5 / (nu * math.pi ** 2)
        steps = math.ceil(T / min(0.3 * h, 0.15 * h * h / nu))
        W = run(cfg, W0, T / steps, steps, setup=lambda o: o.set_body_force(*acc))
        drift.append(np.abs(W[1 + m].mean(axis=other) - uavg).max() / uavg.max())
        assert np.abs(W[0] - 1).max() < 1e-9
    assert drift[1] < 2e-3 and drift[0] / drift[1] > 3.5


# ---------------------------------------------------------------- P23 mirror symmetry (low side / high side of every boundary kind)
@pytest.mark.parametrize("bc", [(IN, OUT, P, P, SL, NS), (NS, SL, IN, OUT, P, P), (P, P, EX, NS, OUT, IN),
                                (EX, IN, SL, SL, NS, EX)])
@pytest.mark.parametrize("with_ibm", [False, True])
def test_P23_the_mirrored_problem_gives_the_mirrored_result(bc, with_ibm):
    """reflect the grid, the state, the boundary kinds, the inflow velocity and the actuator / immersed points about
    the mid-plane of an axis: the step must return the reflection (WENO, the collision and both forcing kernels are
    mirror-symmetric; round-off only).  Catches anything that treats the low and the high side of an axis
    differently.  Without IBM points the y axis is stretched."""
    n, sp = (10, 9, 8), (0.1, 0.1, 0.12)
    z, y, x = np.meshgrid(*[(np.arange(m) + 0.5) / m for m in (n[2], n[1], n[0])], indexing="ij")
    W0 = np.zeros((4,) + x.shape)
    W0[0] = 1 + 0.02 * np.sin(2 * np.pi * x + 1) * np.cos(2 * np.pi * y) + 0.01 * np.sin(2 * np.pi * z + 0.5)
    W0[1] = W0[0] * (0.1 + 0.02 * np.cos(2 * np.pi * y + 0.3) * np.sin(2 * np.pi * z))
    W0[2] = W0[0] * (0.03 * np.sin(2 * np.pi * x + 0.2) + 0.01 * np.cos(2 * np.pi * z))
    W0[3] = W0[0] * (0.02 * np.cos(2 * np.pi * x) * np.sin(2 * np.pi * y + 0.7))
    inflow = [1.0, 0.0, 0.0, 0.0]
    for ax in range(3):
        if IN in bc[2 * ax:2 * ax + 2]:
            inflow[1 + ax] = 0.1 if bc[2 * ax] == IN else -0.1
    yf = np.arange(n[1] + 1) * sp[1] if with_ibm else np.cumsum(np.r_[0.0, np.linspace(0.7, 1.4, n[1])]) * 0.1
    length = [n[0] * sp[0], yf[-1], n[2] * sp[2]]
    alm_pos = np.array([[0.42, 0.40, 0.5], [0.61, 0.33, 0.41]])
    alm_force = np.array([[0.01, 0.02, -0.01], [-0.02, 0.0, 0.01]])
    ibm_pos = np.array([[0.5, 0.45, 0.48], [0.52, 0.47, 0.5], [0.3, 0.6, 0.36]])
    ibm_vol = np.full(3, 0.5 * sp[0] * sp[1] * sp[2])

    def solve(faces_y, bcs, infl, state, apos, aforce, ipos):
        def setup(o):
            o.alm_set_points(apos, aforce, 0.08)
            if with_ibm:
                o.ibm_set_points(ipos, ibm_vol)
        cfg = GridConfig(n=n, faces=(None, faces_y, None), spacing=sp, nu=2e-3, bc=tuple(bcs), inflow=tuple(infl))
        return run(cfg, state, 0.01, 3, setup=setup)

    Wa = solve(yf, bc, inflow, W0, alm_pos, alm_force, ibm_pos)
    assert np.abs(Wa - W0).max() > 1e-4
    for a in range(3):
        sign = np.ones(4)
        sign[1 + a] = -1.0
        flip = lambda W: np.ascontiguousarray(np.flip(W, axis=3 - a) * sign[:, None, None, None])
        bcm = list(bc)
        bcm[2 * a], bcm[2 * a + 1] = bc[2 * a + 1], bc[2 * a]
        inflm = list(inflow)
        inflm[1 + a] = -inflow[1 + a]
        mirror = lambda pts: np.where(np.arange(3) == a, length[a] - pts, pts)
        Wb = flip(solve((yf[-1] - yf)[::-1] if a == 1 else yf, bcm, inflm, flip(W0), mirror(alm_pos),
                        alm_force * sign[1:], mirror(ibm_pos)))
        assert np.abs(Wa - Wb).max() < TOL_SYMMETRY, a


# ---------------------------------------------------------------- P24 stations and airfoil sections (reading S28)
def test_P24_explicit_stations_and_section_blended_polars():
    """PAPER.md:376 (actuator points refined at tip and root) and :127 (lift and drag tables interpolated between nearby
    airfoil sections).  Pinned on special cases that reduce to the single-table, evenly spaced rotor of P17 and on the
    linearity of Eq. 9 in the element width and in the tabulated coefficients."""
    from dataclasses import replace
    cfg, r = rotor_case()
    rng = np.random.default_rng(5)
    W = const_state(cfg.n, (1.05, 0.1, 0.01, -0.02))
    W += 1e-3 * rng.standard_normal(W.shape) * np.array([1.0, 0.1, 0.1, 0.1])[:, None, None, None]

    def forces(rot):
        o = ob.Oracle(cfg)
        o.set_state(W)
        o.alm_set_rotor(rot)
        out = o.alm_rotor_eval()
        o.close()
        return out

    p0, f0 = forces(r)
    w = (r.R - r.r_hub) / r.npts
    even_r, even_w = r.r_hub + (np.arange(r.npts) + 0.5) * w, np.full(r.npts, w)
    # (i) the default stations given explicitly: the same bits
    p1, f1 = forces(replace(r, radius=even_r, width=even_w))
    assert np.array_equal(p1, p0) and np.array_equal(f1, f0)
    # (ii) Eq. 9 is linear in the element width w: doubling the width of station 5 doubles its force and no other
    w2 = even_w.copy()
    w2[5] *= 2.0
    _, f2 = forces(replace(r, radius=even_r, width=w2))
    f0b, f2b = f0.reshape(r.nblades, r.npts, 3), f2.reshape(r.nblades, r.npts, 3)
    assert np.array_equal(f2b[:, 5], 2.0 * f0b[:, 5]) and np.array_equal(np.delete(f2b, 5, 1), np.delete(f0b, 5, 1))
    # (iii) the points sit at the given radii on the blade's azimuth (refined stations of the synthetic recipe)
    rr = wl.synthetic_rotor(hub=r.hub, R=r.R, eps=r.eps, npts=r.npts, refine=True)
    assert rr.width.sum() == pytest.approx(r.R - r.r_hub, rel=1e-14) and rr.width[0] < 0.3 * rr.width[r.npts // 2]
    p3, _ = forces(rr)
    d = p3 - np.asarray(r.hub)
    assert np.allclose(np.hypot(d[:, 1], d[:, 2]).reshape(r.nblades, r.npts), rr.radius[None, :], rtol=1e-14)
    assert np.allclose(np.arctan2(d[:, 2], d[:, 1]).reshape(r.nblades, r.npts)[0], r.theta0)
    # (iv) airfoil sections.  Two identical sections are the single table ...
    two = replace(r, cl=np.stack([r.cl, r.cl]), cd=np.stack([r.cd, r.cd]), section_r=np.array([0.3, 0.8]))
    assert np.array_equal(forces(two)[1], f0)
    # ... inside the first / outside the last section their own tables act, and between them C_L and C_D are linear in
    # r, i.e. (both look-ups being linear in the table values) the force of a station is the one a single table
    # blended with the same weight gives
    clb, cdb = 0.6 * r.cl + 0.1, 1.7 * r.cd + 0.01
    sec = np.array([even_r[4], even_r[10]])                                  # sections AT stations 4 and 10
    mixed = replace(r, cl=np.stack([r.cl, clb]), cd=np.stack([r.cd, cdb]), section_r=sec)
    fm = forces(mixed)[1].reshape(r.nblades, r.npts, 3)
    fa = f0b
    fb = forces(replace(r, cl=clb, cd=cdb))[1].reshape(r.nblades, r.npts, 3)
    assert np.array_equal(fm[:, :5], fa[:, :5]) and np.array_equal(fm[:, 10:], fb[:, 10:])
    for k in range(5, 10):
        t = (even_r[k] - sec[0]) / (sec[1] - sec[0])
        fk = forces(replace(r, cl=(1 - t) * r.cl + t * clb, cd=(1 - t) * r.cd + t * cdb))[1].reshape(r.nblades, r.npts, 3)
        assert np.abs(fm[:, k] - fk[:, k]).max() <= 1e-14 * np.abs(fk[:, k]).max(), k
    assert np.abs(fm[:, 7] - fa[:, 7]).max() > 1e-3 * np.abs(fa[:, 7]).max()     # the blend does change the force
    # refusals: radius without width, decreasing section radii, a station beyond the tip
    o = ob.Oracle(cfg)
    o.set_state(W)
    for bad in (replace(r, radius=even_r), replace(mixed, section_r=sec[::-1].copy()),
                replace(r, radius=even_r * 2.0, width=even_w)):
        with pytest.raises(Exception):
            o.alm_set_rotor(bad)
    o.close()


# ---------------------------------------------------------------- P25 ghost cells by their definitions (S17, S18, S21)
def test_P25_ghost_cells_by_definition():
    """the ghost fill read back (`get_padded`) against the definitions of DESIGN.md, written out with numpy on the input
    array: extrapolation = the nearest interior cell in all three layers (S21: zero gradient, NOT a linear
    extrapolation - the data below have a gradient, so any other constant or linear rule fails), no-slip wall = mirror
    image with all momenta odd (S17), slip wall = mirror image with the normal momentum odd (S18), periodic = image;
    pass order x, y, z: an edge ghost is the y-rule applied to the x-ghost"""
    rng = np.random.default_rng(31)
    n = (7, 8, 9)
    W = np.empty((4, n[2], n[1], n[0]))
    x, y, z = np.meshgrid(np.arange(n[2]), np.arange(n[1]), np.arange(n[0]), indexing="ij")
    W[0] = 1.0 + 0.01 * z + 0.02 * y + 0.015 * x + 1e-3 * rng.standard_normal(W[0].shape)
    W[1:] = 0.1 + 0.01 * rng.standard_normal(W[1:].shape) + 0.005 * (x + 2 * y - z)
    cfg = GridConfig(n=n, spacing=(0.1, 0.1, 0.1), bc=(EX, EX, NS, SL, P, P))
    o = ob.Oracle(cfg)
    o.set_state(W)
    G = o.get_padded()                                          # (4, nz+6, ny+6, nx+6)
    o.close()
    I = G[:, 3:-3, 3:-3, 3:-3]
    assert np.array_equal(I, W)
    # x faces: extrapolation, both sides, all three layers = the first / last interior cell
    for g in range(1, 4):
        assert np.array_equal(G[:, 3:-3, 3:-3, 3 - g], W[..., 0]) and np.array_equal(G[:, 3:-3, 3:-3, 2 + n[0] + g], W[..., -1])
    # y low: no-slip wall (rho even, momenta odd); y high: slip wall (rho, tangential momenta even, normal momentum odd)
    for g in range(1, 4):
        lo, hi = G[:, 3:-3, 3 - g, 3:-3], G[:, 3:-3, 2 + n[1] + g, 3:-3]
        assert np.array_equal(lo[0], W[0, :, g - 1, :]) and np.array_equal(lo[1:], -W[1:, :, g - 1, :])
        assert np.array_equal(hi[[0, 1, 3]], W[[0, 1, 3]][:, :, n[1] - g, :]) and np.array_equal(hi[2], -W[2, :, n[1] - g, :])
    # z: periodic image
    for g in range(1, 4):
        assert np.array_equal(G[:, 3 - g, 3:-3, 3:-3], W[:, n[2] - g]) and np.array_equal(G[:, 2 + n[2] + g, 3:-3, 3:-3], W[:, g - 1])
    # an x-y edge: the y-rule (no-slip mirror) applied to the x-ghost column (pass order x, then y)
    assert np.array_equal(G[0, 3:-3, 2, 1], W[0, :, 0, 0]) and np.array_equal(G[2, 3:-3, 1, 3 + n[0]], -W[2, :, 1, -1])
