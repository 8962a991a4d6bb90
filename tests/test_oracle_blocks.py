"""Pins of the oracle's building blocks against what the paper and the mathematics fix (P1-P5, P11-P13).

Every expected value here is built independently of oracle/gks_oracle.cpp: quadrature of the
Maxwellian, polynomial fits by numpy, textbook Navier-Stokes fluxes.  CPU only.
"""
import os

import numpy as np
import pytest
from numpy.polynomial import Polynomial as Poly
from numpy.polynomial.hermite import hermgauss

from oracle import binding as ob

RNG = np.random.default_rng(1234)


# ---------------------------------------------------------------- P1: moment recursion
@pytest.mark.parametrize("U,lam", [(0.0, 0.5), (0.1, 0.5), (-0.37, 0.5), (1.3, 2.0), (-0.05, 50.0)])
def test_P1_moment_recursion_vs_quadrature(U, lam):
    """<u^n> = (1/rho) int u^n g du by Gauss-Hermite quadrature, n <= 6."""
    x, w = hermgauss(24)
    u = U + x / np.sqrt(lam)
    ref = np.array([(w * u ** n).sum() / np.sqrt(np.pi) for n in range(7)])
    got = ob.moments(U, lam, 6)
    assert np.allclose(got, ref, rtol=1e-13, atol=1e-15)
    assert got[0] == 1.0 and got[1] == U


# ---------------------------------------------------------------- P2: reconstruction operators
def cell_averages(poly, centres, width=1.0):
    P = poly.integ()
    return np.array([(P(c + width / 2) - P(c - width / 2)) / width for c in centres])


def fit_from_averages(q, centres):
    """polynomial of degree len(q)-1 whose cell averages (unit cells at `centres`) equal q"""
    n = len(q)
    A = np.array([[((c + .5) ** (p + 1) - (c - .5) ** (p + 1)) / (p + 1) for p in range(n)] for c in centres])
    return Poly(np.linalg.solve(A, q))


CENTRES = np.arange(-2, 3, dtype=float)
GP = np.sqrt(3.0) / 6.0


def js_beta_from_definition(q):
    """Jiang-Shu: beta_k = sum_{l=1,2} int_{-1/2}^{1/2} (d^l p_k/dx^l)^2 dx on the middle cell"""
    betas, cands = [], []
    for k in range(3):
        p = fit_from_averages(q[k:k + 3], CENTRES[k:k + 3])
        b = 0.0
        for l in (1, 2):
            d2 = (p.deriv(l) ** 2).integ()
            b += d2(0.5) - d2(-0.5)
        betas.append(b)
        cands.append(p)
    return np.array(betas), cands


def weno_from_definition(q, x, eps):
    """WENO5-JS built from its definition at point x of the middle cell: candidates = quadratic fits,
    linear weights = those that reproduce the quartic fit, alpha_k = d_k/(eps+beta_k)^2."""
    betas, cands = js_beta_from_definition(q)
    # linear weights from the definition: sum_k d_k p_k(x) = p_quartic(x) for every data set
    rows, rhs = [], []
    for _ in range(3):
        qq = RNG.standard_normal(5)
        _, cc = js_beta_from_definition(qq)
        rows.append([c(x) for c in cc])
        rhs.append(fit_from_averages(qq, CENTRES)(x))
    d = np.linalg.solve(np.array(rows), np.array(rhs))
    assert abs(d.sum() - 1) < 1e-10 and (d > 0).all()
    alpha = d / (eps + betas) ** 2
    wgt = alpha / alpha.sum()
    return sum(wk * c(x) for wk, c in zip(wgt, cands))


@pytest.mark.parametrize("deg", range(5))
def test_P2_linear_weights_reproduce_polynomials(deg):
    """with the nonlinear weights switched off (eps huge) every operator is exact for degree <= 4"""
    poly = Poly(RNG.standard_normal(deg + 1))
    q = cell_averages(poly, CENTRES)
    big = 1e20
    assert abs(ob.weno5_face(q, big) - poly(0.5)) < 1e-12
    assert abs(ob.weno5_face(q[::-1], big) - poly(-0.5)) < 1e-12          # mirrored = left edge
    v = ob.weno5_gauss(q, big)
    assert abs(v[0] - poly(-GP)) < 1e-12 and abs(v[1] - poly(GP)) < 1e-12
    s = ob.quartic_slope_gauss(q)
    assert abs(s[0] - poly.deriv()(-GP)) < 1e-12 and abs(s[1] - poly.deriv()(GP)) < 1e-12


@pytest.mark.parametrize("deg", range(3))
def test_P2_nonlinear_weno_exact_for_quadratics(deg):
    """all three candidates are exact for degree <= 2, so any weights give the exact value"""
    poly = Poly(RNG.standard_normal(deg + 1))
    q = cell_averages(poly, CENTRES)
    assert abs(ob.weno5_face(q) - poly(0.5)) < 1e-13
    v = ob.weno5_gauss(q)
    assert abs(v[0] - poly(-GP)) < 1e-13 and abs(v[1] - poly(GP)) < 1e-13


def test_P2_linear_weight_rows():
    """the coefficient rows SURVEY.md P2 states for the linear-weight operators"""
    s3 = np.sqrt(3.0)
    face_row = np.array([1 / 30, -13 / 60, 47 / 60, 9 / 20, -1 / 20])
    gp_row = np.array([-1 / 4320 + 7 * s3 / 432, 1 / 1080 - 25 * s3 / 216, 719 / 720,
                       1 / 1080 + 25 * s3 / 216, -1 / 4320 - 7 * s3 / 432])
    I = np.eye(5)
    got_face = np.array([ob.weno5_face(I[m], 1e20) for m in range(5)])
    got_gp = np.array([ob.weno5_gauss(I[m], 1e20)[1] for m in range(5)])
    assert np.allclose(got_face, face_row, atol=1e-14)
    assert np.allclose(got_gp, gp_row, atol=1e-14)


def test_P2_normal_slope_exact_for_cubics():
    for deg in range(4):
        poly = Poly(RNG.standard_normal(deg + 1))
        q = cell_averages(poly, np.array([-1.5, -0.5, 0.5, 1.5]))
        assert abs(ob.normal_slope(q) - poly.deriv()(0.0)) < 1e-12


def test_P2_weno_constant_data_exact():
    for c in (1.0, 0.1, -3.7, 1e-8):
        q = np.full(5, c)
        assert ob.weno5_face(q) == pytest.approx(c, rel=4e-16)
        v = ob.weno5_gauss(q)
        assert v[0] == pytest.approx(c, rel=4e-16) and v[1] == pytest.approx(c, rel=4e-16)
        assert np.abs(ob.quartic_slope_gauss(q)).max() <= 1e-15 * abs(c)


@pytest.mark.parametrize("trial", range(6))
def test_P2_weno_js_against_definition(trial):
    """random (non-smooth) data: value = definition of WENO5-JS (smoothness integrals, fitted
    candidates, derived linear weights) at the face and both Gauss points"""
    q = RNG.standard_normal(5) * (10.0 ** RNG.integers(-3, 1))
    eps = 1e-6
    assert ob.weno5_face(q, eps) == pytest.approx(weno_from_definition(q, 0.5, eps), rel=1e-11, abs=1e-14)
    v = ob.weno5_gauss(q, eps)
    assert v[1] == pytest.approx(weno_from_definition(q, GP, eps), rel=1e-11, abs=1e-14)
    assert v[0] == pytest.approx(weno_from_definition(q, -GP, eps), rel=1e-11, abs=1e-14)


def test_P2_weno_picks_smooth_stencil_at_a_jump():
    """essentially non-oscillatory: a jump inside the right sub-stencils leaves the left candidate"""
    q = np.array([1.0, 1.0, 1.0, 5.0, 5.0])
    assert abs(ob.weno5_face(q) - 1.0) < 1e-6
    assert abs(ob.weno5_gauss(q)[1] - 1.0) < 1e-6


# ---------------------------------------------------------------- P3: Appendix solve
def appendix_matrix(U, V, W, lam):
    """the 4x4 matrix printed at PAPER.md:537"""
    h = 1.0 / (2.0 * lam)
    return np.array([[1, U, V, W],
                     [U, U * U + h, U * V, U * W],
                     [V, U * V, V * V + h, V * W],
                     [W, U * W, V * W, W * W + h]])


@pytest.mark.parametrize("trial", range(5))
def test_P3_micro_solve_inverts_appendix_matrix(trial):
    U, V, W = RNG.uniform(-0.5, 0.5, 3)
    lam = RNG.uniform(0.3, 3.0)
    d = RNG.standard_normal(4)
    a = ob.micro_solve(U, V, W, lam, d)
    assert np.allclose(appendix_matrix(U, V, W, lam) @ a, d, rtol=0, atol=1e-13)


def test_P3_micro_coefficients_are_log_derivatives_of_g():
    """a = d(ln g)/dx: a^2 = 2 lam U_x, a^3 = 2 lam V_x, a^4 = 2 lam W_x,
    a^1 = rho_x/rho - 2 lam (U U_x + V V_x + W W_x)   (differentiate Eq. 2)"""
    rho, U, V, W, lam = 1.3, 0.2, -0.1, 0.05, 0.7
    rx, Ux, Vx, Wx = 0.4, -0.3, 0.25, 0.11
    dQ = np.array([rx, rx * U + rho * Ux, rx * V + rho * Vx, rx * W + rho * Wx])
    a = ob.micro_solve(U, V, W, lam, dQ / rho)
    ref = np.array([rx / rho - 2 * lam * (U * Ux + V * Vx + W * Wx), 2 * lam * Ux, 2 * lam * Vx, 2 * lam * Wx])
    assert np.allclose(a, ref, atol=1e-14)


# ---------------------------------------------------------------- P4: collision
def half_moments_quadrature(Q, d, RT, sign):
    """int_{sign*u_n>0} psi g dXi by 1-D numerical quadrature along the normal velocity"""
    from scipy.integrate import quad
    lam = 1 / (2 * RT)
    rho = Q[0]
    vel = Q[1:] / rho
    Un = vel[d]
    g1 = lambda u: np.sqrt(lam / np.pi) * np.exp(-lam * (u - Un) ** 2)
    lo, hi = (0, np.inf) if sign > 0 else (-np.inf, 0)
    m0 = quad(g1, lo, hi, epsabs=1e-14, epsrel=1e-13)[0]
    m1 = quad(lambda u: u * g1(u), lo, hi, epsabs=1e-14, epsrel=1e-13)[0]
    out = np.empty(4)
    out[0] = rho * m0
    for c in range(3):
        out[1 + c] = rho * (m1 if c == d else vel[c] * m0)
    return out


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P4_collision_is_sum_of_half_maxwellian_moments(d):
    RT = 1.0
    Ql = np.array([1.05, 0.12, -0.03, 0.07])
    Qr = np.array([0.97, 0.08, 0.02, -0.05])
    ref = half_moments_quadrature(Ql, d, RT, +1) + half_moments_quadrature(Qr, d, RT, -1)
    assert np.allclose(ob.collision(Ql, Qr, d, RT), ref, rtol=1e-12, atol=1e-14)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_P4_collision_identity_and_mirror(d):
    Q = np.array([1.1, 0.13, -0.2, 0.05])
    assert np.allclose(ob.collision(Q, Q, d, 1.0), Q, rtol=0, atol=3e-16)
    Ql = np.array([1.05, 0.12, -0.03, 0.07])
    Qr = np.array([0.97, 0.08, 0.02, -0.05])
    flip = np.ones(4)
    flip[1 + d] = -1.0
    a = ob.collision(Ql, Qr, d, 0.8)
    b = ob.collision(Qr * flip, Ql * flip, d, 0.8)
    assert np.allclose(a, b * flip, rtol=0, atol=3e-16)


# ---------------------------------------------------------------- P5: Navier-Stokes flux identity
def primitive_gradients(Q0, dQ):
    rho = Q0[0]
    vel = Q0[1:] / rho
    drho = dQ[:, 0]
    dvel = (dQ[:, 1:] - vel[None, :] * drho[:, None]) / rho      # dvel[s][i] = d_s U_i
    return rho, vel, drho, dvel


def euler_flux(Q, d, RT):
    rho, vel = Q[0], Q[1:] / Q[0]
    F = Q * vel[d]
    F[1 + d] += rho * RT
    return F


def test_P5_flux_is_isothermal_navier_stokes_flux():
    """Eq. 7 moments with A from compatibility = Euler flux - mu (d_i U_j + d_j U_i), mu = tau p = rho_ref nu;
    dF/dt = (dF_Euler/dQ) . Q_t with Q_t = -div F_Euler (chain rule through the slopes)."""
    RT, nu, rho_ref = 0.9, 0.013, 1.2
    for trial in range(5):
        Q0 = np.array([1.0 + 0.1 * RNG.standard_normal(), *(0.2 * RNG.standard_normal(3))])
        dQ = 0.3 * RNG.standard_normal((3, 4))
        rho, vel, drho, dvel = primitive_gradients(Q0, dQ)
        mu = rho_ref * nu
        # Q_t = -sum_s dF_Euler^s/dQ . d_s Q  by finite-difference-free chain rule (Jacobian by complex step)
        def jac(d):
            J = np.empty((4, 4))
            for m in range(4):
                Qc = Q0.astype(complex)
                Qc[m] += 1e-30j
                J[:, m] = euler_flux(Qc, d, RT).imag / 1e-30
            return J
        Qt = -sum(jac(s) @ dQ[s] for s in range(3))
        for d in range(3):
            F, dF = ob.gauss_point_flux(Q0, dQ, d, RT, nu, rho_ref)
            ref = euler_flux(Q0.copy(), d, RT)
            for i in range(3):
                ref[1 + i] -= mu * (dvel[d, i] + dvel[i, d])
            assert np.allclose(F, ref, rtol=0, atol=2e-15), (d, F - ref)
            assert np.allclose(dF, jac(d) @ Qt, rtol=0, atol=5e-15)


# ---------------------------------------------------------------- P13: brute-force velocity-space quadrature
def test_P13_flux_by_direct_quadrature_of_eq7():
    """int psi u_d f dXi with f of Eq. 7 on a tensor Gauss-Hermite velocity grid; a_s and A obtained by
    numpy.linalg.solve on quadrature-built moment matrices (no use of the Appendix formulas)."""
    RT, nu, rho_ref = 1.0, 0.02, 1.0
    lam = 1 / (2 * RT)
    x, w = hermgauss(12)
    Q0 = np.array([1.07, 0.11, -0.06, 0.09])
    dQ = np.array([[0.2, -0.1, 0.05, 0.3], [-0.15, 0.25, 0.1, -0.2], [0.05, 0.12, -0.3, 0.08]])
    rho = Q0[0]
    vel = Q0[1:] / rho
    u, v, ww = np.meshgrid(vel[0] + x / np.sqrt(lam), vel[1] + x / np.sqrt(lam), vel[2] + x / np.sqrt(lam), indexing="ij")
    wt = np.einsum("i,j,k->ijk", w, w, w) / np.pi ** 1.5 * rho        # quadrature weights of g0 dXi
    psi = np.stack([np.ones_like(u), u, v, ww])
    mom = lambda f: np.array([(wt * f * p).sum() for p in psi])       # int psi f g0 dXi
    M = np.array([mom(p) for p in psi])                               # M[m][n] = int psi_n psi_m g0
    a = [np.linalg.solve(M.T, dQ[s]) for s in range(3)]               # <a_s psi> rho = d_s Q0  (Eq. 8)
    apoly = [sum(a[s][m] * psi[m] for m in range(4)) for s in range(3)]
    adv = apoly[0] * u + apoly[1] * v + apoly[2] * ww
    A = np.linalg.solve(M.T, -mom(adv))                               # compatibility
    Apoly = sum(A[m] * psi[m] for m in range(4))
    tau = rho_ref * nu / (rho * RT)
    for d, un in enumerate((u, v, ww)):
        F_ref = mom(un * (1 - tau * (adv + Apoly)))
        dF_ref = mom(un * Apoly)
        F, dF = ob.gauss_point_flux(Q0, dQ, d, RT, nu, rho_ref)
        assert np.allclose(F, F_ref, rtol=0, atol=1e-13)
        assert np.allclose(dF, dF_ref, rtol=0, atol=1e-13)


# ---------------------------------------------------------------- P11 (kernel part) / paper constants
def golden():
    out = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "paper_constants.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()[:2]
                out[k] = float(v)
    return out


def test_P11_gaussian_kernel_paper_values():
    g = golden()
    eps = 0.37
    ratio = ob.alm_kernel(g["gauss_1pct_radius_in_eps"] * eps, eps) / ob.alm_kernel(0.0, eps)
    assert abs(ratio - 0.01) < 5e-4                                     # "1 %" at r = 2.15 eps
    assert ob.alm_kernel(0.0, eps) == pytest.approx(1 / (eps ** 3 * np.pi ** 1.5), rel=1e-15)
    # normalisation: int_0^inf 4 pi r^2 K(r) dr = 1 (Eq. 10 conserves the point force)
    from scipy.integrate import quad
    val = quad(lambda r: 4 * np.pi * r * r * ob.alm_kernel(r, eps), 0, 20 * eps, epsabs=1e-13)[0]
    assert abs(val - 1) < 1e-11


# ---------------------------------------------------------------- P12: discrete delta
def test_P12_delta3_identities():
    for r in np.linspace(-0.5, 0.5, 41):
        ph = np.array([ob.delta3(r - i) for i in (-2, -1, 0, 1, 2)])
        off = np.array([r - i for i in (-2, -1, 0, 1, 2)])
        assert abs(ph.sum() - 1) < 1e-14
        assert abs((off * ph).sum()) < 1e-14
        assert abs((ph ** 2).sum() - 0.5) < 1e-14
    assert ob.delta3(1.5) == 0.0 and ob.delta3(1.7) == 0.0 and ob.delta3(-2.0) == 0.0
    assert ob.delta3(0.0) == pytest.approx(2.0 / 3.0)
