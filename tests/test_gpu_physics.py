"""The exact-solution checks that pin the oracle (tests/test_oracle_step.py: P8-P10, P19-P22), run on the CUDA
library itself through the C ABI.  They need no oracle and hold at any size, so the two finest ones go beyond
what the oracle can afford on the CPU: the order of accuracy is also measured 32^3 -> 64^3, the stretched vortex at
64 cells, a Taylor-Green vortex on 128^3.

The scenario functions are the CPU suite's own; only the solver factory is swapped."""
import math

import numpy as np
import pytest

import test_oracle_step as tos

pytestmark = pytest.mark.gpu


class CudaSolver:
    """the names the scenario functions use (those of oracle/binding.py) on paper_2603_11102_b200.gks.Gks"""

    def __init__(self, cfg):
        from paper_2603_11102_b200 import gks
        self._g = gks.Gks(cfg)

    def __getattr__(self, name):
        return getattr(self._g, name)

    def eval_flux(self, d):
        return self._g.debug_eval_flux(d)


@pytest.fixture(autouse=True)
def cuda_solver(monkeypatch):
    monkeypatch.setattr(tos, "new_solver", CudaSolver)
    monkeypatch.setattr(tos, "TOL_SYMMETRY", 1e-13)
    monkeypatch.setattr(tos, "TOL_UNIFORM", 1e-13)


def test_order_of_accuracy_on_the_exact_simple_wave_up_to_64_cubed():
    """PAPER.md:89 'two-stage fourth-order': the L1 error of the isothermal simple wave along (1,1,1) falls 16x per
    refinement (P8's exact solution by Newton on the characteristics)"""
    tos.test_P8_order_of_accuracy_on_exact_simple_wave()
    e32, e64 = tos.simple_wave_error(32), tos.simple_wave_error(64)
    assert math.log2(e32[0] / e64[0]) >= 3.7 and math.log2(e32[1] / e64[1]) >= 3.7, (e32, e64)
    assert e64[0] < 1.5e-7


@pytest.mark.parametrize("RT,rho,rho_ref", [(1.0, 1.0, 1.0), (0.64, 1.3, 1.0)])
def test_viscous_decay_rate(RT, rho, rho_ref):
    tos.test_P9_shear_wave_decays_at_mu_over_rho(RT, rho, rho_ref)


def test_acoustic_speed():
    tos.test_P10_acoustic_wave_travels_at_sqrt_RT(0.64)


@pytest.mark.parametrize("s,m", [(0, 1), (1, 2), (2, 0)])
def test_couette_stress_on_a_stretched_axis(s, m):
    tos.test_P19_couette_stress_on_a_stretched_axis_is_second_order(s, m)


def test_vortex_decay_on_a_stretched_axis_third_level():
    """P19's vortex, one refinement further than the CPU suite goes"""
    tos.test_P19_vortex_between_slip_walls_on_a_stretched_axis_decays_at_2_nu_k2()
    e32, e64 = tos.vortex_decay_rate_error(32), tos.vortex_decay_rate_error(64)
    assert abs(e64) < 3e-4 and abs(e32 / e64) > 2.0, (e32, e64)


@pytest.mark.parametrize("axis,side", [(0, 0), (1, 1), (2, 0)])
def test_piston_problem(axis, side):
    tos.test_P20_impulsive_inflow_drives_the_rankine_hugoniot_shock(axis, side)


@pytest.mark.parametrize("axis,side", [(0, 1), (0, 0), (1, 0), (1, 1), (2, 0), (2, 1)])
def test_pulse_through_the_convective_outflow(axis, side):
    tos.test_P21_vortical_pulse_leaves_through_the_convective_outflow(axis, side)


@pytest.mark.parametrize("axis", [1, 2])
def test_noslip_walls(axis):
    tos.test_P22_shear_mode_between_noslip_walls_decays_at_nu_k2(axis)
    if axis == 1:
        tos.test_P22_poiseuille_profile_is_steady_under_the_body_force()


def test_taylor_green_kinetic_energy_decays_at_2_nu_k2_on_the_metric_box_shape():
    """the 2-D Taylor-Green vortex extended along z on a 128^3 periodic box (the shape of BASELINE.json's metric box
    at a quarter of its cells): kinetic energy decays at 4 nu k^2, velocity amplitude at 2 nu k^2"""
    from paper_2603_11102_b200.workloads import GridConfig
    N, nu, U0, k = 128, 0.02, 0.02, 1.0
    h = 2 * math.pi / N
    cfg = GridConfig(n=(N, N, N), spacing=(h, h, h), RT=1.0, nu=nu, bc=(tos.P,) * 6)
    xf = np.arange(N + 1) * h
    s = (np.cos(xf[:-1]) - np.cos(xf[1:])) / h
    c = (np.sin(xf[1:]) - np.sin(xf[:-1])) / h
    W0 = tos.const_state((N, N, N), (1.0, 0.0, 0.0, 0.0))
    W0[1] = U0 * (c[:, None] * s[None, :])[None]          # u =  U0 sin x cos y
    W0[2] = -U0 * (s[:, None] * c[None, :])[None]         # v = -U0 cos x sin y
    T = 0.5
    steps = math.ceil(T / (0.4 * h / (1.0 + U0)))
    W = tos.run(cfg, W0, T / steps, steps)
    mode = (c[:, None] * s[None, :])[None]
    amp = (W[1] * mode).sum() / (mode ** 2).sum() / N / U0
    assert -math.log(amp) / T == pytest.approx(2 * nu * k * k, rel=2e-3)   # O(Ma^2) = 4e-4 compressibility
    assert np.abs(W[3]).max() < 1e-12


@pytest.mark.parametrize("lo,hi", [(tos.NS, tos.SL), (tos.IN, tos.OUT), (tos.OUT, tos.IN), (tos.EX, tos.EX)])
@pytest.mark.parametrize("stretched", [False, True])
def test_every_boundary_kind_treats_the_three_axes_alike(lo, hi, stretched):
    """P14 on the CUDA path: three different sweep kernels (x-, y-, z-faces) and three ghost passes must agree"""
    tos.test_P14_every_boundary_kind_treats_the_three_axes_alike(lo, hi, stretched)


@pytest.mark.parametrize("bc", [(tos.IN, tos.OUT, tos.P, tos.P, tos.SL, tos.NS), (tos.P, tos.P, tos.EX, tos.NS, tos.OUT, tos.IN),
                                (tos.EX, tos.IN, tos.SL, tos.SL, tos.NS, tos.EX)])
@pytest.mark.parametrize("with_ibm", [False, True])
def test_the_mirrored_problem_gives_the_mirrored_result(bc, with_ibm):
    """P23 on the CUDA path: low and high side of every boundary kind, of the tiles' ragged edges, of IBM and ALM"""
    tos.test_P23_the_mirrored_problem_gives_the_mirrored_result(bc, with_ibm)


def test_three_hundred_steps_of_the_taylor_green_vortex_stay_conservative_and_dissipative():
    """the metric box's flow at 128^3, 300 steps (a long run for a test, a blink for the GPU): mass and momentum are
    conserved to round-off, the kinetic energy never grows (Re = 1600, early times: slow viscous decay), all finite"""
    from paper_2603_11102_b200 import gks, workloads as wl
    w = wl.taylor_green(128)
    g = gks.Gks(w.cfg)
    g.set_state(w.W0)
    ke = lambda W: 0.5 * ((W[1:] ** 2).sum(0) / W[0]).sum(dtype=np.longdouble)
    energy, sums0 = [ke(w.W0)], [w.W0[c].sum(dtype=np.longdouble) for c in range(4)]
    scale = np.abs(w.W0[1:]).sum(dtype=np.longdouble)
    for chunk in range(6):
        for _ in range(50):
            g.step(w.dt)
        W = g.get_state()
        g.check_finite()
        energy.append(ke(W))
        assert abs(W[0].sum(dtype=np.longdouble) - sums0[0]) <= 1e-12 * abs(sums0[0])
        for c in range(1, 4):
            assert abs(W[c].sum(dtype=np.longdouble) - sums0[c]) <= 1e-12 * scale
    g.close()
    drops = -np.diff(np.array(energy, dtype=np.float64))
    assert (drops > 0).all() and drops.sum() < 0.05 * float(energy[0]), energy
