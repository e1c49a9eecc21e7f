"""Pins of the oracle's five-stage 4th-order low-storage Runge-Kutta scheme (eq. (36)-(38)
with "five sub-stages", coefficients "from [23]" = Carpenter & Kennedy's 2N-storage RK4; Q35).
The paper prints no coefficients; they are pinned by what a 4th-order five-stage scheme must satisfy."""
import numpy as np

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W


def test_stability_polynomial():
    """R(U) = lambda U: U1/U0 = 1 + z + z^2/2 + z^3/6 + z^4/24 + z^5/200 (the four order conditions of a linear
    problem; the z^5 coefficient 1/200 is the published one of this scheme)."""
    for lam, dt in ((-1.3, 0.4), (0.7, 0.25), (-20.0, 0.01), (2.0, 0.5)):
        U = np.array([1.7, -0.3])
        U0 = U.copy()
        dU = np.full(2, np.nan)                      # dU^(0) must never be read (A_1 = 0)
        for s in range(5):
            O.rk4_update(s, dt, U, dU, lam * U)
        z = lam * dt
        np.testing.assert_allclose(U / U0, 1 + z + z ** 2 / 2 + z ** 3 / 6 + z ** 4 / 24 + z ** 5 / 200, rtol=5e-12)


def test_fourth_order_on_a_nonlinear_ode():
    """y' = -y^2 (exact y = 1/(1 + t)): nonlinear order conditions, error falls by 16 per halving."""
    def run(nsteps):
        y, d = np.array([1.0]), np.zeros(1)
        dt = 1.0 / nsteps
        for _ in range(nsteps):
            for s in range(5):
                O.rk4_update(s, dt, y, d, -y * y)
        return abs(y[0] - 0.5)
    e = [run(k) for k in (8, 16, 32)]
    assert 13.0 < e[0] / e[1] < 19.0 and 13.0 < e[1] / e[2] < 19.0, e


def test_step_fourth_order_in_time_on_euler():
    nx = 32
    x = np.arange(-3, nx + 3) / nx
    rho = 1 + 0.2 * np.sin(2 * np.pi * x)
    Q0 = W.conservative(rho[None, None, :], 1.0, 0.0, 0.0, 1.0, 1.4)
    kw = dict(n=(nx, 1, 1), delta=(1.0 / nx, 1, 1), scheme=W.WENOZ5, bc=((0, 0),) * 3, nthreads=1)

    def run(nsteps):
        o = O.Oracle(**kw)
        Q = np.ascontiguousarray(Q0.copy())
        o.run(Q, 0.16 / nsteps, nsteps, rk4=True)
        return o.interior(Q)[0].ravel()

    ref = run(64)
    e = [np.max(np.abs(run(k) - ref)) for k in (2, 4, 8)]
    assert e[0] / e[1] > 11.0 and e[1] / e[2] > 10.0, e
