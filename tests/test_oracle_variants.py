"""P21 / P22: pins of the oracle's simple averaging (PAPER.md:104 step 2(a); Q38) and of the SSP
3rd-order low-storage Runge-Kutta scheme (Q39)."""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

G = 1.4


def flux_n(q, n):
    rho, m, E = q[0], q[1:4], q[4]
    u = m / rho
    p = (G - 1.0) * (E - 0.5 * rho * (u @ u))
    th = u @ n
    return np.array([rho * th, m[0] * th + p * n[0], m[1] * th + p * n[1], m[2] * th + p * n[2], (E + p) * th])


def jacobian_n(q, n):
    """dF_n/dQ by complex-step differentiation of the flux function itself (nothing of the oracle restated)."""
    J = np.zeros((5, 5))
    for c in range(5):
        qc = q.astype(complex)
        qc[c] += 1e-30j
        rho, m, E = qc[0], qc[1:4], qc[4]
        u = m / rho
        p = (G - 1.0) * (E - 0.5 * rho * (u @ u))
        th = u @ n
        f = np.array([rho * th, m[0] * th + p * n[0], m[1] * th + p * n[1], m[2] * th + p * n[2], (E + p) * th])
        J[:, c] = f.imag / 1e-30
    return J


def random_state(rng):
    rho = rng.uniform(0.3, 2.0)
    u = rng.uniform(-1.5, 1.5, 3)
    p = rng.uniform(0.2, 3.0)
    return np.array([rho, *(rho * u), p / (G - 1.0) + 0.5 * rho * (u @ u)])


# --------------------------------------------------------------------------- P21: simple averaging ----
def test_p21_simple_average_is_the_eigensystem_of_the_mean_state():
    """U_{i+1/2} = (U_i + U_{i+1})/2: L R = I and A_n(U_{i+1/2}) R = R Lambda with the flux Jacobian taken at that
    mean conservative state; Lambda = diag(theta, theta, theta, theta + a, theta - a) of the same state."""
    rng = np.random.default_rng(21)
    for _ in range(20):
        QL, QR = random_state(rng), random_state(rng)
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        L, R, roe = O.eigensystem(G, QL, QR, n, averaging=O.AVG_SIMPLE)
        qm = 0.5 * (QL + QR)
        um = qm[1:4] / qm[0]
        pm = (G - 1.0) * (qm[4] - 0.5 * qm[0] * (um @ um))
        am = np.sqrt(G * pm / qm[0])
        np.testing.assert_allclose(roe[:3], um, rtol=1e-14, atol=1e-15)
        np.testing.assert_allclose(roe[4], am, rtol=1e-13)
        np.testing.assert_allclose(roe[3], (qm[4] + pm) / qm[0], rtol=1e-14)
        np.testing.assert_allclose(L @ R, np.eye(5), atol=1e-13)
        th = um @ n
        lam = np.diag([th, th, th, th + am, th - am])
        A = jacobian_n(qm, n)
        np.testing.assert_allclose(A @ R, R @ lam, atol=2e-12 * np.abs(A).max())


def test_p21_simple_equals_roe_for_equal_states_and_differs_otherwise():
    rng = np.random.default_rng(22)
    q = random_state(rng)
    n = np.array([0.6, 0.0, 0.8])
    Ls, Rs, _ = O.eigensystem(G, q, q, n, averaging=O.AVG_SIMPLE)
    Lr, Rr, _ = O.eigensystem(G, q, q, n, averaging=O.AVG_ROE)
    np.testing.assert_allclose(Ls, Lr, rtol=1e-13, atol=1e-14)
    np.testing.assert_allclose(Rs, Rr, rtol=1e-13, atol=1e-14)
    q2 = random_state(rng)
    assert np.abs(O.eigensystem(G, q, q2, n, averaging=O.AVG_SIMPLE)[1] - O.eigensystem(G, q, q2, n)[1]).max() > 1e-3
    # symmetric in its two arguments (the Roe average is too)
    a = O.eigensystem(G, q, q2, n, averaging=O.AVG_SIMPLE)
    b = O.eigensystem(G, q2, q, n, averaging=O.AVG_SIMPLE)
    for x, y in zip(a, b):
        np.testing.assert_array_equal(x, y)


def test_p21_sod_with_simple_averaging_converges_to_the_exact_solution():
    """The averaging only picks the frame of the characteristic projection: Sod still converges at first order,
    with an L1 error within a few per cent of the Roe-averaged run (golden constants: tests/golden/sod_exact.txt
    through test_oracle_pins)."""
    from test_oracle_pins import exact_riemann_sod
    errs = {}
    for avg in (O.AVG_ROE, O.AVG_SIMPLE):
        for nx in (200, 400):
            c = W.sod(nx)
            c.averaging = avg
            o = O.Oracle(**c.physics(), nthreads=1)
            Q = o.run(c.Q0.copy(), c.dt, c.nsteps)
            rho = o.interior(Q)[0].ravel()
            errs[(avg, nx)] = np.abs(rho - exact_riemann_sod(c.extra["x"], c.extra["t_end"])[0]).mean()
    assert 1.0e-3 < errs[(O.AVG_SIMPLE, 400)] < 2.0e-3, errs
    assert errs[(O.AVG_SIMPLE, 400)] < 0.6 * errs[(O.AVG_SIMPLE, 200)], errs
    assert abs(errs[(O.AVG_SIMPLE, 400)] / errs[(O.AVG_ROE, 400)] - 1.0) < 0.1, errs
    assert errs[(O.AVG_SIMPLE, 400)] != errs[(O.AVG_ROE, 400)]


def test_p21_simple_averaging_conservation_and_consistency():
    """Flux-difference form is untouched (sum of R = 0 on a periodic box); a constant state still returns the
    exact flux."""
    c = W.tgv(8, visc=W.VISC_NONE)
    c.Q0 = W.perturb(c, seed=3, amp=0.05)
    c.averaging = O.AVG_SIMPLE
    o = O.Oracle(**c.physics())
    Q = o.bc(c.Q0.copy())
    R = o.interior(o.rhs(Q))
    for v in range(5):
        assert abs(R[v].sum()) <= 1e-11 * np.abs(R[v]).sum()
    q = random_state(np.random.default_rng(5))
    Qc = np.ascontiguousarray(np.broadcast_to(q[:, None, None, None], o.shape))
    for d in range(3):
        n = np.eye(3)[d]
        np.testing.assert_allclose(o.interface_flux(Qc, d, 3, 3, 3), flux_n(q, n), rtol=1e-13, atol=1e-14)


# ------------------------------------------------------------------------------- P22: SSP-RK3 ----
SSP_A = (0.0, -2.915493957701923, 0.0)
SSP_B = (0.924574, 0.287713063186749, 0.626538109512740)


def _step(update, lam, u0, dt, nstages=3):
    U = np.array([u0], dtype=np.float64)
    dU = np.zeros(1)
    for s in range(nstages):
        R = lam * U
        update(s, dt, U, dU, R)
    return U[0]


def test_p22_ssp_rk3_stability_polynomial():
    """Linear test equation: one step multiplies by 1 + z + z^2/2 + z^3/6 up to the precision the published
    coefficients carry (B_1 is printed to six digits: the order conditions hold to 5e-7, not to round-off)."""
    for z in (-0.5, -0.1, 0.3, 1.0):
        g = _step(O.rk3ssp_update, z, 1.0, 1.0)
        assert abs(g - (1 + z + z * z / 2 + z ** 3 / 6)) < 1.5e-6 * max(1.0, abs(z)), (z, g)


def test_p22_ssp_rk3_is_a_convex_combination_of_euler_steps():
    """Effective Butcher tableau of the 2N-storage form eq. (36)-(37): all a_ij, b_j >= 0 (the SSP/TVD property of
    ref. [44]); order conditions to the printed precision; and in Shu-Osher form every stage is a convex
    combination of forward-Euler steps with step ratio <= 1/0.32 (the published CFL coefficient 0.32)."""
    m = 3
    dU = np.zeros(m)
    U = np.zeros(m)
    a = np.zeros((m, m))
    for i in range(m):
        a[i] = U
        dU = SSP_A[i] * dU
        dU[i] += 1.0
        U = U + SSP_B[i] * dU
    b, c = U, a.sum(1)
    assert (a >= 0).all() and (b >= 0).all()
    assert abs(b.sum() - 1) < 1e-6 and abs(b @ c - 0.5) < 1e-6 and abs(b @ c ** 2 - 1 / 3) < 1e-6 and abs(b @ (a @ c) - 1 / 6) < 1e-6
    # the oracle's update reproduces this tableau on a problem with stage-dependent residuals
    rng = np.random.default_rng(2)
    Rs = rng.normal(size=3)
    Uo, dUo = np.array([0.7]), np.array([123.0])       # dU^(0) is never read (A_1 = 0)
    for s in range(3):
        O.rk3ssp_update(s, 0.1, Uo, dUo, np.array([Rs[s]]))
    assert abs(Uo[0] - (0.7 + 0.1 * (b @ Rs))) < 1e-15


def test_p22_ssp_rk3_tvd_on_upwind_advection_where_williamson_form_is_not_guaranteed():
    """First-order upwind advection of a step, CFL 0.3 (< 0.32): total variation never increases with the SSP
    coefficients."""
    n, cfl = 64, 0.3
    u = np.where(np.arange(n) < n // 2, 1.0, 0.0)
    dU = np.zeros(n)

    def tv(v):
        return np.abs(np.diff(np.concatenate([v, v[:1]]))).sum()

    tv0 = tv(u)
    for _ in range(40):
        for s in range(3):
            R = -(u - np.roll(u, 1))
            O.rk3ssp_update(s, cfl, u, dU, R)
        assert tv(u) <= tv0 + 1e-13
        assert u.min() >= -1e-13 and u.max() <= 1 + 1e-13


def test_p22_ssp_rk3_third_order_on_a_nonlinear_ode_and_through_the_step():
    """y' = -y^2, y(0) = 1 -> 1/(1+t): error falls ~8x per halving of dt (until the 5e-7 consistency floor of the
    printed coefficients); oracle_rk3_step with rk3_form = SSP uses exactly these updates."""
    def run(dt):
        y, dy = np.array([1.0]), np.zeros(1)
        for _ in range(int(round(1.0 / dt))):
            for s in range(3):
                O.rk3ssp_update(s, dt, y, dy, -y * y)
        return abs(y[0] - 0.5)
    e1, e2 = run(0.2), run(0.1)
    assert 5.0 < e1 / e2 < 12.0, (e1, e2)
    c = W.sod(nx=50, nsteps=2)
    c.rk3_form = O.RK3_SSP
    o = O.Oracle(**c.physics())
    Q = o.run(c.Q0.copy(), c.dt, 1)
    ow = O.Oracle(**{**c.physics(), "rk3_form": O.RK3_WILLIAMSON})
    Q2 = c.Q0.copy()
    dU, R = np.zeros_like(Q2), np.zeros_like(Q2)
    for s in range(3):
        ow.bc(Q2)
        R = ow.rhs(Q2)
        for v in range(5):
            Ui = np.ascontiguousarray(ow.interior(Q2)[v].ravel())
            dUi = np.ascontiguousarray(ow.interior(dU)[v].ravel())
            O.rk3ssp_update(s, c.dt, Ui, dUi, np.ascontiguousarray(ow.interior(R)[v].ravel()))
            ow.interior(Q2)[v][...] = Ui.reshape(ow.interior(Q2)[v].shape)
            ow.interior(dU)[v][...] = dUi.reshape(ow.interior(dU)[v].shape)
    ow.bc(Q2)
    np.testing.assert_array_equal(Q, Q2)
