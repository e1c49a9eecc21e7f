"""Pins of the seeded input generators (paper_2007_14933_b200/workloads.py): the BASELINE.json
config 4 slab is built from textbook pieces (compressible similarity boundary layer, Rankine-
Hugoniot jump, tanh stretching) whose values are fixed independently of this repository:
SURVEY.md section 8(d) lists them (computed there by a separate probe) and the closed forms below
re-derive them."""
import numpy as np
import pytest

from paper_2007_14933_b200 import workloads as W


@pytest.fixture(scope="module")
def bl():
    return W.similarity_boundary_layer()


def test_similarity_profile_values(bl):
    # f''(0) = 0.513435, T_aw = g(0) = 1.676194, I = 2.316717, x0 = 88.50
    assert abs(bl["fpp0"] - 0.513435) < 2e-6
    assert abs(bl["g0"] - 1.676194) < 2e-6
    assert abs(bl["I"] - 2.316717) < 5e-6
    assert abs(950.0 / (2 * bl["I"] ** 2) - 88.50) < 0.01
    # boundary conditions of the ODE system and monotone profiles
    assert bl["fp"][0] == 0.0 and abs(bl["fp"][-1] - 1.0) < 1e-12 and abs(bl["g"][-1] - 1.0) < 1e-12
    assert np.all(np.diff(bl["fp"]) > -1e-14) and np.all(np.diff(bl["g"]) < 1e-14)
    # adiabatic wall: g'(0) = 0 (one-sided second-order difference), recovery factor close to sqrt(Pr)
    h = bl["eta"][1]
    assert abs((-3 * bl["g"][0] + 4 * bl["g"][1] - bl["g"][2]) / (2 * h)) < 1e-4
    r = (bl["g0"] - 1.0) / (0.5 * 0.4 * 4.0)
    assert abs(r - np.sqrt(0.72)) < 0.01


def test_similarity_profile_satisfies_the_momentum_equation(bl):
    """Residual of (C f'')' + f f'' = 0 re-evaluated by central differences on the returned table."""
    h = bl["eta"][1]
    fp, g = bl["fp"], bl["g"]
    f = np.concatenate([[0.0], np.cumsum(0.5 * h * (fp[1:] + fp[:-1]))])
    C = W.sutherland(g) / g
    fpp = np.gradient(fp, h)
    res = np.gradient(C * fpp, h) + f * fpp
    assert np.abs(res[5:-5]).max() < 5e-4


def test_oblique_shock_values():
    sh = W.oblique_shock()
    # p2/p1 = 1.186467, rho2/rho1 = 1.129735, u2 = 0.966702, v2 = -0.052106, p2 = 0.211869
    assert abs(sh["p_ratio"] - 1.186467) < 1e-6 and abs(sh["rho_ratio"] - 1.129735) < 1e-6
    assert abs(sh["u"] - 0.966702) < 1e-6 and abs(sh["v"] + 0.052106) < 1e-6 and abs(sh["p"] - 0.211869) < 1e-6
    # conservation across the shock in the shock-normal frame: mass, normal momentum, tangential velocity
    b = np.deg2rad(32.58)
    nrm, tng = np.array([np.sin(b), np.cos(b)]), np.array([np.cos(b), -np.sin(b)])     # shock running down to the wall
    u1, u2 = np.array([1.0, 0.0]), np.array([sh["u"], sh["v"]])
    p1 = 1.0 / (1.4 * 4.0)
    assert abs(1.0 * u1 @ nrm - sh["rho"] * (u2 @ nrm)) < 1e-14
    assert abs(p1 + (u1 @ nrm) ** 2 - sh["p"] - sh["rho"] * (u2 @ nrm) ** 2) < 1e-14
    assert abs(u1 @ tng - u2 @ tng) < 1e-14
    assert abs(np.rad2deg(np.arctan2(-sh["v"], sh["u"])) - 3.085) < 2e-3          # flow deflection


def test_sbli_slab_structure():
    c = W.sbli_slab(n=(60, 40, 5))
    h = c.halo
    core = (slice(h[2], h[2] + 5), slice(h[1], h[1] + 40), slice(h[0], h[0] + 60))
    x, y, z = (c.coords[d][core] for d in range(3))
    assert x[0, 0, 0] == 0.0 and abs(x[0, 0, -1] - 300.0) < 1e-12 and y[0, 0, 0] == 0.0 and abs(y[0, -1, 0] - 115.0) < 1e-12
    assert np.all(np.diff(x, axis=2) > 0) and np.all(np.diff(y, axis=1) > 0)              # the grid does not fold
    assert np.abs(x[:, 0, :] - x[:, -1, :]).max() < 1e-10                                  # perturbation vanishes on the walls
    assert np.abs(np.diff(x, axis=1)).max() > 0.1                                          # ... and not inside: cross metrics
    assert abs(np.diff(z, axis=0).max() - 0.6) < 1e-15
    rho, mx, my, mz, E = (c.Q0[v][core] for v in range(5))
    assert np.all(my == 0) and np.all(mz == 0)
    u = mx / rho
    assert np.all(u[:, 0, :] == 0.0) and abs(u[:, -1, :].max() - 1.0) < 1e-12             # no slip, free stream
    p = 0.4 * (E - 0.5 * rho * u * u)
    assert np.abs(p - 1.0 / 5.6).max() < 1e-14
    # seeded noise: reproducible, bounded by 1e-4 relative, absent from the frozen boundary state
    c2 = W.sbli_slab(n=(60, 40, 5))
    assert np.array_equal(c.Q0, c2.Q0)
    d = c.dirichlet[0][core]
    inner = (slice(None), slice(0, 39), slice(None))
    rel = rho[inner] / d[inner] - 1.0
    assert 0.5e-4 < np.abs(rel).max() <= 1e-4 and abs(rel.mean()) < 1e-5
    # top boundary of the frozen state: free stream before x = 20, Rankine-Hugoniot state behind
    top = c.dirichlet[:, h[2], h[1] + 39, h[0]:h[0] + 60]
    xs = x[0, -1, :]
    sh = W.oblique_shock()
    assert np.all(top[0][xs < 20.0] == 1.0) and np.allclose(top[0][xs >= 20.0], sh["rho"], rtol=0, atol=1e-15)
    assert c.wall_T[1][0] == c.extra["bl"]["g0"] and c.bc[1][0] == W.BC_WALL_ISOTHERMAL


def test_sbli_slab_wall_spacing_full_size():
    c = W.sbli_slab()
    y = c.coords[1][3, 3:3 + 250, 3]
    assert abs((y[1] - y[0]) - 0.0314) < 1e-4 and abs((y[-1] - y[-2]) - 1.17) < 1e-2
    assert c.n == (500, 250, 8) and c.dt == 1e-3 and c.nsteps == 500 and c.scheme == W.WENOZ5
