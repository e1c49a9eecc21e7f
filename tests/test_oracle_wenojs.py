"""Pins of the oracle's WENO-JS5 weights (scheme 3; eq. (20)-(21): alpha_r =
d_r/(eps + beta_r)^2, eps = 1e-6).  Candidates, ideal weights and smoothness
indicators are the ones WENO-Z5 / TENO5 use (pinned in test_oracle_pins.py); what is new is eq. (21),
pinned by a worked example done by hand, the formal order, the ENO property and, as for the other
schemes, conservation / reflection of the residual and the brute-force NumPy residual (P12)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

JS = W.WENOJS5


def test_worked_example_step():
    """Data (0,0,0,1,1): beta_L = 0, beta_C = 13/12 + 1/4 = 4/3, beta_R = 13/12 + 9/4 = 10/3;
    q_L = 0, q_C = 1/3, q_R = 2/3; with eps = 1e-6 << beta the weight of the smooth stencil is
    1 - O(eps^2) and W = [d_C q_C/beta_C^2 + d_R q_R/beta_R^2] eps^2/d_L + O(eps^3)
      = (0.6/3 * 9/16 + 0.3 * 2/3 * 9/100) * 1e-12 / 0.1 = 1.305e-12."""
    w = O.reconstruct(JS, 0.0, 0.0, 0.0, 1.0, 1.0, eps=1e-6)
    assert abs(w - 1.305e-12) < 2e-17 * 1e3
    assert abs(O.reconstruct(JS, 1.0, 1.0, 1.0, 0.0, 0.0, eps=1e-6) - (1.0 - 1.305e-12)) < 1e-15


def test_equal_indicators_give_the_ideal_weights():
    """A ramp has beta_L = beta_C = beta_R, so eq. (20)-(21) return d_r and W is the linear 5th-order value;
    read off by differentiating about the ramp is not possible here (the weights move at first order), so
    compare with the linear scheme (2a - 13b + 47c + 27d - 3e)/60 on ramps of several slopes."""
    for s in (0.1, 1.0, -3.0):
        v = [s * k + 0.5 for k in range(5)]
        lin = (2 * v[0] - 13 * v[1] + 47 * v[2] + 27 * v[3] - 3 * v[4]) / 60
        assert abs(O.reconstruct(JS, *v, eps=1e-6) - lin) < 1e-14 * max(1.0, abs(lin))


def test_fifth_order_on_sine():
    errs = []
    for N in (32, 64, 128):
        h = 2 * np.pi / N
        x = h * np.arange(N) + 0.3                      # keep the critical points off the nodes
        f = np.sin(x)
        fh = np.array([O.reconstruct(JS, *[f[(i + m) % N] for m in range(-2, 3)], eps=1e-6) for i in range(N)])
        errs.append(np.abs((fh - np.roll(fh, 1)) / h - np.cos(x)).max())
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert (rates > 4.5).all(), (errs, rates)            # JS loses accuracy near critical points: >= 4.5 here


def _line(n=48):
    i, j, k = W.padded_index_grids((n, 1, 1))
    x = 2 * np.pi * i / n + 0 * j + 0 * k
    rho = 1.0 + 0.3 * np.sin(x) + 0.1 * np.cos(3 * x)
    u = 0.4 + 0.2 * np.sin(2 * x + 0.3)
    p = 1.0 + 0.2 * np.cos(x - 0.5)
    per = (W.BC_PERIODIC, W.BC_PERIODIC)
    return W.Case(name="line", n=(n, 1, 1), Q0=np.ascontiguousarray(W.conservative(rho, u, 0.0, 0.0, p, 1.4)), dt=1e-3,
                  nsteps=1, delta=(2 * np.pi / n, 1.0, 1.0), gamma=1.4, scheme=JS, eps=1e-6, bc=(per, (0, 0), (0, 0)))


def test_residual_conservation_reflection_and_sod():
    case = _line()
    orc = O.Oracle(**case.physics())
    R = orc.interior(orc.rhs(orc.bc(case.Q0.copy())))
    for c in (0, 1, 4):
        assert abs(R[c].sum()) <= 1e-12 * np.abs(R[c]).sum()
    Qm = orc.interior(case.Q0)[:, :, :, ::-1].copy()
    Qm[1] *= -1.0
    Qpad = case.Q0.copy()
    h = case.halo
    Qpad[:, :, :, h[0]:h[0] + case.n[0]] = Qm
    Rm = orc.interior(orc.rhs(orc.bc(Qpad)))
    np.testing.assert_allclose(Rm[0][..., ::-1], R[0], rtol=0, atol=1e-12)
    np.testing.assert_allclose(-Rm[1][..., ::-1], R[1], rtol=0, atol=1e-12)
    # Sod to t = 0.1: same first-order L1 band as WENO-Z5 (P1), a little more smeared
    sod = W.sod(nx=200, scheme=JS, dt=4e-4, nsteps=250)
    sod.eps = 1e-6
    rho = {}
    for sch in (JS, W.WENOZ5):
        o = O.Oracle(**{**sod.physics(), "scheme": sch, "eps": 1e-6 if sch == JS else 1e-16})
        rho[sch] = o.interior(o.run(sod.Q0.copy(), sod.dt, sod.nsteps))[0].ravel()
    assert np.isfinite(rho[JS]).all() and rho[JS].min() > 0.125 - 1e-4 and rho[JS].max() < 1.0 + 1e-4   # P1: no over/undershoot beyond 1e-4
    assert 0 < np.abs(rho[JS] - rho[W.WENOZ5]).mean() < 5e-3
