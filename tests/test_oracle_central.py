"""Pins of the oracle's 4th-order central convective scheme (scheme 4; eq. (28), 208-226
closures; the scheme of the paper's single-GPU timing case).  The stencils themselves are
pinned by P6; pinned here is their use on the flux vectors: the exact residual of the Taylor-Green field
(symbolic differentiation) at 4th order, conservation, exactness of the closures on a flux that is a polynomial,
and the brute-force NumPy residual (tests/test_oracle_bruteforce.py, P12)."""
import numpy as np

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W
from test_oracle_residual import tgv_exact_residual


def test_analytic_tgv_residual_fourth_order():
    errs = []
    for n in (16, 32):
        c = W.tgv(n, scheme=W.CENTRAL4)
        o = O.Oracle(**c.physics())
        R = o.interior(o.rhs(o.bc(c.Q0.copy())))
        ex = tgv_exact_residual(n)
        errs.append([np.max(np.abs(R[v] - ex[v])) for v in range(5)])
    for v in range(5):
        assert errs[1][v] < errs[0][v] / 11.0 or errs[1][v] < 1e-12, (v, errs)      # 2^4 = 16 asymptotically; 12.9 at 16 -> 32


def test_conservation_on_a_periodic_box():
    c = W.tgv(12, scheme=W.CENTRAL4, visc=W.VISC_NONE)
    rng = np.random.default_rng(4)
    c.Q0 = c.Q0 * (1.0 + 0.05 * rng.uniform(-1, 1, size=c.Q0.shape))
    o = O.Oracle(**c.physics())
    R = o.interior(o.rhs(o.bc(c.Q0.copy())))
    for v in range(5):
        assert abs(R[v].sum()) <= 1e-12 * np.abs(R[v]).sum()


def test_closures_are_exact_when_the_flux_is_a_cubic():
    """1-D, u = const > 0, p = const: the fluxes are rho u, rho u^2 + p, (rho E + p) u, all linear in rho, so a
    cubic rho(x) gives -dF/dx exactly at every node, the one-sided closure nodes included."""
    nx, u0, p0 = 24, 0.7, 1.3
    x = (np.arange(-3, nx + 3) / (nx - 1.0))[None, None, :]
    rho = 1.0 + 0.5 * x - 0.3 * x ** 2 + 0.2 * x ** 3
    drho = 0.5 - 0.6 * x + 0.6 * x ** 2
    ex = (W.BC_EXTRAP0, W.BC_EXTRAP0)
    c = W.Case(name="cubic", n=(nx, 1, 1), Q0=np.ascontiguousarray(W.conservative(rho, u0, 0.0, 0.0, p0, 1.4)), dt=1e-3,
               nsteps=1, delta=(1.0 / (nx - 1), 1.0, 1.0), gamma=1.4, scheme=W.CENTRAL4, bc=(ex, (0, 0), (0, 0)))
    o = O.Oracle(**c.physics())
    Q = c.Q0.copy()                      # halos hold the cubic too, but the closures must not need them
    R = o.interior(o.rhs(Q))
    d = drho[..., 3:3 + nx]
    np.testing.assert_allclose(R[0], -u0 * d, atol=1e-12)
    np.testing.assert_allclose(R[1], -u0 * u0 * d, atol=1e-12)
    np.testing.assert_allclose(R[4], -0.5 * u0 ** 3 * d, atol=1e-12)
