"""Pins of the oracle's third-order WENO-Z (scheme 5; "WENO-3Z"; the k = 2 member of
PAPER.md:147-167; Q37): candidates, ideal weights and indicators follow from the definitions the
paper gives for general k and are pinned by polynomial exactness, the 3rd-order linear limit, the formal order,
the ENO property and the residual's conservation / reflection; P12 covers the assembly."""
import numpy as np

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

Z3 = W.WENOZ3


def test_all_weights_ideal_gives_the_third_order_value():
    base = [0.5 * k for k in range(5)]                     # ramp: beta_0 = beta_1, tau = 0
    w0 = O.reconstruct(Z3, *base)
    coef = [(O.reconstruct(Z3, *[v + (1e-3 if j == m else 0.0) for m, v in enumerate(base)]) - w0) / 1e-3 for j in range(5)]
    np.testing.assert_allclose(coef, np.array([0, -1, 5, 2, 0]) / 6.0, atol=1e-5)    # (-b + 5c + 2d)/6; a, e unused


def test_exact_on_quadratic_cell_averages_when_smooth():
    import sympy as sp
    x = sp.symbols("x")
    poly = 2 + x / 3 + x ** 2 / 400          # nearly a ramp: the nonlinear weights stay at the ideal ones to O(tau^2)
    avg = [float(sp.integrate(poly, (x, k - sp.Rational(1, 2), k + sp.Rational(1, 2)))) for k in range(-2, 3)]
    assert abs(O.reconstruct(Z3, *avg) - float(poly.subs(x, sp.Rational(1, 2)))) < 1e-7


def test_third_order_on_sine_and_steps():
    errs = []
    for N in (32, 64, 128):
        h = 2 * np.pi / N
        x = h * np.arange(N) + 0.3
        f = np.sin(x)
        fh = np.array([O.reconstruct(Z3, *[f[(i + m) % N] for m in range(-2, 3)]) for i in range(N)])
        away = np.abs(np.cos(x)) > 0.5                      # WENO-Z3 with tau = |beta_0 - beta_1| drops to 2nd order around
        errs.append(np.abs((fh - np.roll(fh, 1)) / h - np.cos(x))[away].max())   # critical points (f' -> 0): a known property
    rates = np.log2(np.array(errs[:-1]) / np.array(errs[1:]))
    assert (rates > 2.7).all(), (errs, rates)              # 3rd order where f' is bounded away from 0
    assert O.reconstruct(Z3, 0.0, 0.0, 0.0, 1.0, 1.0) < 1e-15 and abs(O.reconstruct(Z3, 1.0, 1.0, 1.0, 0.0, 0.0) - 1.0) < 1e-15


def test_residual_conservation_and_reflection():
    n = 48
    i, j, k = W.padded_index_grids((n, 1, 1))
    x = 2 * np.pi * i / n + 0 * j + 0 * k
    per = (W.BC_PERIODIC, W.BC_PERIODIC)
    Q0 = np.ascontiguousarray(W.conservative(1.0 + 0.3 * np.sin(x) + 0.1 * np.cos(3 * x), 0.4 + 0.2 * np.sin(2 * x + 0.3), 0.0, 0.0,
                                             1.0 + 0.2 * np.cos(x - 0.5), 1.4))
    c = W.Case(name="line", n=(n, 1, 1), Q0=Q0, dt=1e-3, nsteps=1, delta=(2 * np.pi / n, 1.0, 1.0), gamma=1.4, scheme=Z3,
               bc=(per, (0, 0), (0, 0)))
    o = O.Oracle(**c.physics())
    R = o.interior(o.rhs(o.bc(c.Q0.copy())))
    for v in (0, 1, 4):
        assert abs(R[v].sum()) <= 1e-12 * np.abs(R[v]).sum()
    Qm = o.interior(c.Q0)[:, :, :, ::-1].copy()
    Qm[1] *= -1.0
    Qpad = c.Q0.copy()
    Qpad[:, :, :, 3:3 + n] = Qm
    Rm = o.interior(o.rhs(o.bc(Qpad)))
    np.testing.assert_allclose(Rm[0][..., ::-1], R[0], rtol=0, atol=1e-12)
    np.testing.assert_allclose(-Rm[1][..., ::-1], R[1], rtol=0, atol=1e-12)
