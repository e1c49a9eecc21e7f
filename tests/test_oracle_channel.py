"""Pins of the adiabatic no-slip wall and the constant body force on the laminar
channel of PAPER.md:535-546, whose analytic steady solution eq. (52)-(53) the paper prints together with
T_aw = 1.155520.  Running to t = 1000 (1e7 steps) is out of reach for a test; instead:
  * the adiabatic wall temperature the boundary fill derives from the analytic interior profile is the
    printed T_aw (T is a quartic and the one-sided 4th-order stencil is exact on quartics);
  * the viscous + heat-flux + body-force part of the residual vanishes to round-off on the analytic
    solution (u quadratic, T quartic: the 4th-order stencils and closures are exact), i.e. eq. (52)-(53)
    is a steady state of the discrete momentum and energy balance -- which fixes the sign and size of the
    force terms and of every viscous / heat-flux term against the paper's own formulas;
  * the full residual (with the TENO6 / WENO-Z5 inviscid part) is at truncation level on it.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W


def make(case, **over):
    kw = case.physics()
    kw.update(over)
    return O.Oracle(**kw)


def temperature(case, Q):
    rho = Q[0]
    ke = 0.5 * (Q[1] ** 2 + Q[2] ** 2 + Q[3] ** 2) / rho
    return case.gamma * case.Minf ** 2 * (case.gamma - 1.0) * (Q[4] - ke) / rho


def test_adiabatic_wall_temperature_is_the_printed_value():
    case = W.channel()
    assert abs(case.extra["T_aw"] - 1.155520) < 5e-7                 # PAPER.md:544, 7 s.f.
    orc = make(case)
    Q = case.Q0.copy()
    h, n = case.halo, case.n
    # spoil the wall planes: the fill must rebuild them from the interior
    Q[1:, :, h[1] + n[1] - 1, :] = 7.0
    Q[1:, :, h[1], :] = 7.0
    Q = orc.bc(Q)
    T = temperature(case, Q)
    assert np.abs(T[:, h[1] + n[1] - 1, h[0]:h[0] + n[0]] - 1.155520).max() < 5e-7      # adiabatic side, y = +1
    assert np.abs(T[:, h[1] + n[1] - 1, h[0]:h[0] + n[0]] - case.extra["T_aw"]).max() < 1e-12
    assert np.abs(T[:, h[1], h[0]:h[0] + n[0]] - 1.0).max() < 1e-13                     # isothermal side, y = -1
    assert np.all(Q[1:4, :, h[1] + n[1] - 1, :] == 0.0) and np.all(Q[1:4, :, h[1], :] == 0.0)   # no slip
    # halo temperatures: linear extrapolation through T_w with the first interior slope, eq. (42)
    top = h[1] + n[1] - 1
    for m in (1, 2, 3):
        np.testing.assert_allclose(T[:, top + m, h[0]:h[0] + n[0]],
                                   (m + 1) * T[:, top, h[0]:h[0] + n[0]] - m * T[:, top - 1, h[0]:h[0] + n[0]], rtol=1e-13)


@pytest.mark.parametrize("ny", [33, 64])
def test_analytic_solution_is_a_discrete_steady_state_of_the_viscous_and_force_terms(ny):
    case = W.channel(n=(16, ny, 1))
    orc = make(case)
    Q = orc.bc(case.Q0.copy())
    Rv = orc.interior(orc.rhs(Q, parts=O.PART_VISCOUS))
    # scale: the individual terms are O(1) in momentum (force = 1) and O(Re) in energy (u f = 45)
    assert np.abs(Rv[1]).max() < 1e-9 and np.abs(Rv[2]).max() < 1e-9 and np.abs(Rv[4]).max() < 1e-7, \
        [float(np.abs(Rv[c]).max()) for c in range(5)]
    # without the force the momentum residual is -1 everywhere: the force term is +f, not +rho f
    R0 = make(case, force=(0.0, 0.0, 0.0))
    R0 = R0.interior(R0.rhs(Q, parts=O.PART_VISCOUS))
    np.testing.assert_allclose(R0[1], -1.0, atol=1e-9)
    np.testing.assert_allclose(R0[4], -orc.interior(Q)[1] / orc.interior(Q)[0], atol=1e-7)   # -u f


@pytest.mark.parametrize("scheme", [W.TENO6, W.WENOZ5])
def test_full_residual_on_the_analytic_solution_is_at_truncation_level(scheme):
    errs = []
    for ny in (32, 64):
        case = W.channel(n=(8, ny, 1), scheme=scheme)
        orc = make(case)
        R = orc.interior(orc.rhs(orc.bc(case.Q0.copy())))
        errs.append([float(np.abs(R[c]).max()) for c in range(5)])
    # The y sweep sees p = const and v = 0, so what is left is the Lax-Friedrichs dissipation on the wall-normal
    # variation of rho, rho u, rho E (largest next to the walls, where the reflected halos have a kink).
    # Energy-sized fluxes are (|u|+a) rho E / dy ~ 145 * 1.9e4 * 32 ~ 1e8 here (M = 0.01): the residual is
    # 1e-6 of that and falls under refinement.
    assert max(errs[1]) < 1e-6 * 1e8, errs
    assert max(errs[1]) < 0.5 * max(errs[0]), errs
