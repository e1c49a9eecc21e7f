"""Pins of the CPU oracle against things other than itself (P1-P11).

Each test checks the oracle against what the paper and the mathematics fix: the exact Riemann
solution, closed forms, polynomial exactness, invariants, library routines (numpy.pad), the
Roe property, analytic derivatives (sympy).  None of them retypes an oracle formula.
All CPU-only.
"""
import math

import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

GOLDEN = __import__("pathlib").Path(__file__).parent / "golden"


# ------------------------------------------------------------------ P1: Sod vs exact -------
def exact_riemann_sod(x, t, gamma=1.4, left=(1.0, 0.0, 1.0), right=(0.125, 0.0, 0.1), x0=0.5):
    """Textbook exact solution of the Riemann problem (Toro, ch. 4): left rarefaction, contact,
    right shock.  Newton iteration on the pressure function."""
    rl, ul, pl = left
    rr, ur, pr = right
    al, ar = math.sqrt(gamma * pl / rl), math.sqrt(gamma * pr / rr)
    g1, g2 = (gamma - 1) / (2 * gamma), (gamma + 1) / (2 * gamma)

    def f(p, rk, pk, ak):
        if p > pk:  # shock
            A, B = 2 / ((gamma + 1) * rk), (gamma - 1) / (gamma + 1) * pk
            return (p - pk) * math.sqrt(A / (p + B)), math.sqrt(A / (p + B)) * (1 - (p - pk) / (2 * (B + p)))
        return 2 * ak / (gamma - 1) * ((p / pk) ** g1 - 1), 1 / (rk * ak) * (p / pk) ** (-g2)

    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = f(p, rl, pl, al)
        fr, dfr = f(p, rr, pr, ar)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p -= dp
        if abs(dp) < 1e-15:
            break
    us = 0.5 * (ul + ur) + 0.5 * (f(p, rr, pr, ar)[0] - f(p, rl, pl, al)[0])
    rsl = rl * (p / pl) ** (1 / gamma)                                             # behind the rarefaction
    rsr = rr * ((p / pr + (gamma - 1) / (gamma + 1)) / ((gamma - 1) / (gamma + 1) * p / pr + 1))
    asl = al * (p / pl) ** g1
    S = ur + ar * math.sqrt(g2 * p / pr + g1)                                      # shock speed
    xi = (np.asarray(x) - x0) / t
    rho = np.empty_like(xi)
    head, tail = ul - al, us - asl
    fan = (xi > head) & (xi <= tail)
    rho[xi <= head] = rl
    rho[fan] = rl * (2 / (gamma + 1) + (gamma - 1) / ((gamma + 1) * al) * (ul - xi[fan])) ** (2 / (gamma - 1))
    rho[(xi > tail) & (xi <= us)] = rsl
    rho[(xi > us) & (xi <= S)] = rsr
    rho[xi > S] = rr
    return rho, dict(p=p, u=us, rsl=rsl, rsr=rsr, S=S, head=head, tail=tail)


def _golden_table(name):
    out = {}
    for line in (GOLDEN / name).read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            k, v = line.split()
            out[k] = float(v)
    return out


def test_p1_exact_riemann_constants():
    """The evaluator itself against the tabulated Sod constants (tests/golden/sod_exact.txt)."""
    g = _golden_table("sod_exact.txt")
    _, s = exact_riemann_sod(np.array([0.0]), 0.2)
    assert abs(s["p"] - g["p_star"]) < 1e-6
    assert abs(s["u"] - g["u_star"]) < 1e-6
    assert abs(s["rsl"] - g["rho_star_L"]) < 1e-6
    assert abs(s["rsr"] - g["rho_star_R"]) < 1e-6
    assert abs(s["S"] - g["shock_speed"]) < 1e-6
    assert abs(0.5 + 0.2 * s["head"] - g["x_head"]) < 1e-6
    assert abs(0.5 + 0.2 * s["tail"] - g["x_tail"]) < 1e-6
    assert abs(0.5 + 0.2 * s["u"] - g["x_contact"]) < 1e-6
    assert abs(0.5 + 0.2 * s["S"] - g["x_shock"]) < 1e-6


@pytest.mark.parametrize("scheme", [W.WENOZ5, W.TENO5])
def test_p1_sod_vs_exact(scheme):
    """characteristic decomposition + LF splitting + WENO/TENO + RK3 + EXTRAP0
    against the exact solution at t = 0.2; first-order decay of the L1 error (shocked flow)."""
    errs = {}
    for nx in (200, 400):
        c = W.sod(nx, scheme=scheme)
        o = O.Oracle(**c.physics(), nthreads=1)
        Q = c.Q0.copy()
        o.run(Q, c.dt, c.nsteps)
        rho = o.interior(Q)[0, 0, 0]
        ex, _ = exact_riemann_sod(c.extra["x"], c.extra["t_end"])
        errs[nx] = np.mean(np.abs(rho - ex))
        assert rho.min() > 0.125 - 1e-4 and rho.max() < 1.0 + 1e-4          # essentially non-oscillatory
        assert np.all(Q[2] == 0.0) and np.all(Q[3] == 0.0)                 # unused momenta stay exactly 0
    assert 1.0e-3 < errs[400] < 2.0e-3, errs
    assert 1.6 < errs[200] / errs[400] < 2.3, errs


# ------------------------------------------------ P2: 5th-order convergence on sine data ----
@pytest.mark.parametrize("scheme", [W.WENOZ5, W.TENO5])
def test_p2_fifth_order_on_sine(scheme):
    """(f^_{i+1/2} - f^_{i-1/2})/h vs cos x for f = sin x: the linear 5th-order upwind scheme has
    leading error (h^5/60) f^(6), so L_inf -> h^5/60 (pins candidates, d_r, beta_r, weights)."""
    errs = []
    Ns = (32, 64, 128, 256)
    for N in Ns:
        h = 2 * np.pi / N
        x = np.arange(-3, N + 3) * h
        f = np.sin(x)
        fh = np.array([O.reconstruct(scheme, *f[i:i + 5]) for i in range(N + 1)])   # interface i+2+1/2
        d = (fh[1:] - fh[:-1]) / h                                                   # nodes i+3 -> x index 0..N-1
        errs.append(np.max(np.abs(d - np.cos(x[3:N + 3]))))
    for N, e in zip(Ns[1:], errs[1:]):
        h = 2 * np.pi / N
        assert abs(e / (h ** 5 / 60) - 1) < 0.05, (N, e, h ** 5 / 60)
    rates = [math.log2(errs[i] / errs[i + 1]) for i in range(len(errs) - 1)]
    assert all(4.8 < r < 5.3 for r in rates), rates


def test_p2_mirror_and_exactness():
    """Each candidate and the full stencil reproduce the cell-average-to-interface map of a
    polynomial: for point values of the primitive-difference h(x) = (F(x+1/2) - F(x-1/2)) with F a
    polynomial of degree <= 5, the smooth-limit reconstruction returns F'(1/2)... checked with
    F'(x) = x^4 (degree-4 exactness of the 5-point linear scheme) through tau = 0 data."""
    # constant and linear data: all betas equal -> tau = 0 -> ideal weights -> exact for any scheme
    for scheme in (W.WENOZ5, W.TENO5):
        assert O.reconstruct(scheme, 3.0, 3.0, 3.0, 3.0, 3.0) == pytest.approx(3.0, abs=1e-15)
        # f_i = point values of v(x) whose sliding average is linear: v = a + b x -> interface value a + b/2
        v = [1.0 + 0.5 * i for i in (-2, -1, 0, 1, 2)]
        assert O.reconstruct(scheme, *v) == pytest.approx(1.0 + 0.25, abs=1e-14)


def test_p2_discontinuity_selects_smooth_stencil():
    """ENO property: with a jump between d and e only the stencil {a,b,c} is smooth; TENO must cut
    the other two completely (weights exactly 0/0/1 -> q_L), WENO-Z to O(1e-?) accuracy."""
    a, b, c, d, e = 1.0, 1.1, 1.2, 1.3, 10.0          # jump inside {c,d,e}; {b,c,d}, {a,b,c} linear
    qL = (2 * a - 7 * b + 11 * c) / 6
    qC = (-b + 5 * c + 2 * d) / 6
    # beta_C = beta_L here (both linear data), beta_R huge: TENO keeps L and C with d_L:d_C = 1:6
    got = O.reconstruct(W.TENO5, a, b, c, d, e)
    assert got == pytest.approx((0.1 * qL + 0.6 * qC) / 0.7, rel=1e-14)
    a, b, c, d, e = 1.0, 1.1, 1.2, 10.0, 10.1         # jump between c and d: only {a,b,c} smooth
    got = O.reconstruct(W.TENO5, a, b, c, d, e)
    assert got == pytest.approx((2 * a - 7 * b + 11 * c) / 6, rel=1e-14)
    gz = O.reconstruct(W.WENOZ5, a, b, c, d, e)
    assert abs(gz - (2 * a - 7 * b + 11 * c) / 6) < 1e-3


# ------------------------------------------------------------- P5: eigen-identities --------
def euler_flux_n(Q, n, gamma):
    rho, mx, my, mz, E = Q
    u, v, w = mx / rho, my / rho, mz / rho
    p = (gamma - 1) * (E - 0.5 * rho * (u * u + v * v + w * w))
    th = n[0] * u + n[1] * v + n[2] * w
    return np.array([rho * th, mx * th + p * n[0], my * th + p * n[1], mz * th + p * n[2], (E + p) * th])


def random_state(rng):
    rho = rng.uniform(0.3, 2.0)
    vel = rng.uniform(-1.5, 1.5, 3)
    p = rng.uniform(0.3, 3.0)
    return np.array([rho, *(rho * vel), p / 0.4 + 0.5 * rho * vel @ vel])


def test_p5_eigen_identities_and_roe_property():
    rng = np.random.default_rng(5)
    gamma = 1.4
    for trial in range(50):
        n = rng.normal(size=3)
        n /= np.linalg.norm(n)
        if trial < 3:
            n = np.eye(3)[trial]
        QL, QR = random_state(rng), random_state(rng)
        L, R, roe = O.eigensystem(gamma, QL, QR, n)
        assert np.max(np.abs(L @ R - np.eye(5))) < 1e-13
        u, v, w, H, a = roe
        th = n @ roe[:3]
        lam = np.diag([th, th, th, th + a, th - a])
        # Roe property: F(QR) - F(QL) = R Lambda L (QR - QL) exactly (pins the averaging, Q11)
        lhs = euler_flux_n(QR, n, gamma) - euler_flux_n(QL, n, gamma)
        rhs = R @ lam @ L @ (QR - QL)
        assert np.max(np.abs(lhs - rhs)) < 1e-12 * max(1.0, np.max(np.abs(lhs)))
        # A_n R = R Lambda with the exact Jacobian at a single state (QL = QR): complex-step
        Lq, Rq, rq = O.eigensystem(gamma, QL, QL, n)
        A = np.zeros((5, 5))
        for c in range(5):
            dq = np.zeros(5, dtype=complex)
            dq[c] = 1e-30j
            A[:, c] = np.imag(euler_flux_n(QL.astype(complex) + dq, n, gamma)) / 1e-30
        thq = n @ rq[:3]
        lamq = np.diag([thq, thq, thq, thq + rq[4], thq - rq[4]])
        assert np.max(np.abs(A @ Rq - Rq @ lamq)) < 1e-12 * np.max(np.abs(A))


def test_p5_constant_state_flux_is_exact_flux():
    """Consistency: f^ of a constant state equals f(Q) (uniform and 3-D, every direction)."""
    rng = np.random.default_rng(7)
    q = random_state(rng)
    n = (8, 7, 6)
    o = O.Oracle(n=n, delta=(0.1, 0.2, 0.3), scheme=W.TENO5, bc=((0, 0),) * 3, nthreads=1)
    Q = np.empty(o.shape)
    Q[:] = q[:, None, None, None]
    for d in range(3):
        f = o.interface_flux(Q, d, 3, 3, 3)
        assert np.max(np.abs(f - euler_flux_n(q, np.eye(3)[d], 1.4))) < 1e-13 * np.max(np.abs(f))


# -------------------------------------------------------- P6: stencil exactness ------------
@pytest.mark.parametrize("periodic", [False, True])
def test_p6_central_stencils_exact_to_degree_4(periodic):
    """eq. (28 corrected)-(35): every first/second-difference formula, interior
    and closures (and the mirrored closures), is exact on polynomials up to degree 4."""
    n, h, pad = 9, 0.37, 2
    x = (np.arange(-pad, n + pad)) * h + 0.2
    for deg in range(5):
        f = x ** deg
        for i in range(n):
            xi = x[pad + i]
            e1 = deg * xi ** (deg - 1) if deg >= 1 else 0.0
            e2 = deg * (deg - 1) * xi ** (deg - 2) if deg >= 2 else 0.0
            scale = max(1.0, abs(xi) ** deg / h ** 2)
            assert abs(O.d1(f, i, periodic, h, pad=pad) - e1) < 1e-12 * scale, (deg, i)
            assert abs(O.d2(f, i, periodic, h, pad=pad) - e2) < 1e-11 * scale, (deg, i)
    # the printed eq. (28) is -f' (Q1): the corrected sign gives +1 on f = x
    assert O.d1(x, 4, periodic, h, pad=pad) == pytest.approx(1.0, abs=1e-13)


def test_p6_printed_coefficients_of_eq_28_to_35():
    """Unit impulses through the oracle's difference operators reproduce the coefficients the paper
    prints (tests/golden/central_closure_coefficients.txt); eq. (34)-(35) mirrored
    at the far end (same coefficients, reversed order: DESIGN.md / SURVEY.md O3)."""
    n, h = 11, 0.25
    rows = {}
    for line in (GOLDEN / "central_closure_coefficients.txt").read_text().splitlines():
        if line.strip() and not line.startswith("#"):
            name, _cite, _node, first, coef = [t.strip() for t in line.split("|")]
            rows[name] = (int(first), [float(c) for c in coef.split()])
    node_of = {"interior": 5, "node0": 0, "node1": 1, "nodeN-2": n - 2, "nodeN-1": n - 1}
    for name, (first, coef) in rows.items():
        kind, where = name.split("_", 1)
        i = node_of[where]
        op, scale = (O.d1, 12.0 * h) if kind == "d1" else (O.d2, 12.0 * h * h)
        got = []
        for m in range(n):
            e = np.zeros(n)
            e[m] = 1.0
            got.append(op(e, i, False, h) * scale)
        want = np.zeros(n)
        want[i + first:i + first + 5] = coef
        assert np.allclose(got, want, atol=1e-12), (name, got, want)
    # mirrored second-derivative closures at N-1, N-2
    for where, src in (("nodeN-1", "d2_node0"), ("nodeN-2", "d2_node1")):
        i = node_of[where]
        first, coef = rows[src]
        want = np.zeros(n)
        lo = (n - 1) - (node_of[src.split("_", 1)[1]] + first + 4)
        want[lo:lo + 5] = coef[::-1]
        got = []
        for m in range(n):
            e = np.zeros(n)
            e[m] = 1.0
            got.append(O.d2(e, i, False, h) * 12.0 * h * h)
        assert np.allclose(got, want, atol=1e-12), (where, got, want)


def test_p6_closures_do_not_read_halos():
    n, h, pad = 9, 0.5, 2
    x = np.arange(-pad, n + pad) * h
    f = x ** 3
    g = f.copy()
    g[:pad] = np.nan
    g[-pad:] = np.nan
    for i in range(n):
        assert math.isfinite(O.d1(g, i, False, h, pad=pad))
        assert math.isfinite(O.d2(g, i, False, h, pad=pad))


# ---------------------------------------------------------- P7: RK3 closed form -------------
def test_p7_rk3_stability_polynomial():
    """With R(U) = lambda U one step must give U1/U0 = 1 + z + z^2/2 + z^3/6, z = lambda dt
    (third-order conditions sum b = 1, b.c = 1/2, b.c^2 = 1/3, b.A.c = 1/6)."""
    for lam, dt in ((-1.3, 0.4), (0.7, 0.25), (-20.0, 0.01)):
        U = np.array([1.7, -0.3])
        U0 = U.copy()
        dU = np.full(2, np.nan)                      # dU^(0) must never be read (A_0 = 0)
        for s in range(3):
            R = lam * U
            O.rk3_update(s, dt, U, dU, R)
        z = lam * dt
        assert np.allclose(U / U0, 1 + z + z * z / 2 + z ** 3 / 6, rtol=2e-15, atol=0)


def test_p7_rk3_step_third_order_in_time():
    """oracle_rk3_step on a smooth periodic 1-D Euler problem: error against a dt/16 self-
    reference falls by ~8 per halving of dt (bc -> rhs -> update ordering, coefficients)."""
    nx = 32
    x = np.arange(-3, nx + 3) / nx
    rho = 1 + 0.2 * np.sin(2 * np.pi * x)
    Q0 = W.conservative(rho[None, None, :], 1.0, 0.0, 0.0, 1.0, 1.4)
    kw = dict(n=(nx, 1, 1), delta=(1.0 / nx, 1, 1), scheme=W.WENOZ5, bc=((0, 0),) * 3, nthreads=1)

    def run(nsteps):
        o = O.Oracle(**kw)
        Q = np.ascontiguousarray(Q0.copy())
        o.run(Q, 0.08 / nsteps, nsteps)
        return o.interior(Q)[0].ravel()

    ref = run(64)
    e = [np.max(np.abs(run(k) - ref)) for k in (4, 8, 16)]
    assert 6.5 < e[0] / e[1] < 9.5 and 6.0 < e[1] / e[2] < 10.0, e


# ---------------------------------------------------------- O5: boundary fills --------------
def test_bc_periodic_and_extrap_match_numpy_pad():
    rng = np.random.default_rng(11)
    n = (7, 6, 5)
    core = rng.uniform(1, 2, size=(5, n[2], n[1], n[0]))
    for bc, mode in ((W.BC_PERIODIC, "wrap"), (W.BC_EXTRAP0, "edge")):
        o = O.Oracle(n=n, bc=((bc, bc),) * 3, nthreads=1)
        Q = np.full(o.shape, np.nan)
        o.interior(Q)[:] = core
        o.bc(Q)
        want = np.pad(core, [(0, 0), (3, 3), (3, 3), (3, 3)], mode=mode)
        assert np.array_equal(Q, want)


def test_bc_dirichlet_copies_plane_and_halos():
    rng = np.random.default_rng(12)
    n = (8, 1, 1)
    o0 = O.Oracle(n=n, nthreads=1)
    frozen = rng.uniform(1, 2, size=o0.shape)
    o = O.Oracle(n=n, bc=((W.BC_DIRICHLET, W.BC_EXTRAP0), (0, 0), (0, 0)), dirichlet=frozen, nthreads=1)
    Q = rng.uniform(3, 4, size=o.shape)
    keep = Q.copy()
    o.bc(Q)
    assert np.array_equal(Q[..., :4], frozen[..., :4])               # 3 halos + boundary node
    assert np.array_equal(Q[..., 4:11], keep[..., 4:11])             # interior untouched
    assert np.all(Q[..., 11:] == keep[..., 10:11])                   # zero-order extrapolation


def test_p11_isothermal_wall_halo():
    """eq. (40)-(46): with uniform pressure the halo temperature is the linear
    extrapolation through T_w with the first interior slope, rho_-m = gamma M^2 p_w / T_-m, the
    velocity is mirrored with reversed sign, the wall plane has zero momentum."""
    gamma, M, Tw = 1.4, 2.0, 1.5
    ny = 8
    for side in (0, 1):
        bcy = (W.BC_WALL_ISOTHERMAL, W.BC_EXTRAP0) if side == 0 else (W.BC_EXTRAP0, W.BC_WALL_ISOTHERMAL)
        wt = ((0, 0), (Tw, 0) if side == 0 else (0, Tw), (0, 0))
        o = O.Oracle(n=(1, ny, 1), gamma=gamma, Minf=M, bc=((0, 0), bcy, (0, 0)), wall_T=wt, nthreads=1)
        jj = np.arange(-3, ny + 3)
        dist = jj if side == 0 else (ny - 1 - jj)                      # distance from the wall in cells
        T = Tw + 0.05 * dist                                           # linear profile, T(wall) = Tw
        rho_wall = 0.8
        p0 = rho_wall * Tw / (gamma * M * M)                           # so that p is uniform incl. the wall
        rho = gamma * M * M * p0 / T
        u, v, w = 0.3 * dist, -0.1 * dist, 0.2 * dist
        Q = W.conservative(rho[None, :, None], u[None, :, None], v[None, :, None], w[None, :, None], p0, gamma)
        Q = np.ascontiguousarray(Q)
        jw = 3 if side == 0 else 3 + ny - 1
        Q[1:4, 0, jw, 0] = 7.0                                          # garbage on the wall plane
        Q[4, 0, jw, 0] = 99.0
        rho_wall = Q[0, 0, jw, 0]
        o.bc(Q)
        assert Q[0, 0, jw, 0] == rho_wall                               # wall density floats
        assert np.all(Q[1:4, 0, jw, 0] == 0.0)                          # eq. (40)
        assert Q[4, 0, jw, 0] == pytest.approx(rho_wall * Tw / (M * M * gamma * (gamma - 1)), rel=1e-15)  # eq. (41)
        for m in (1, 2, 3):
            jh = jw - m if side == 0 else jw + m
            ji = jw + m if side == 0 else jw - m
            Tm = (m + 1) * Tw - m * (Tw + 0.05)                         # eq. (42)
            rm = Q[0, 0, jh, 0]
            assert rm == pytest.approx(gamma * M * M * p0 / Tm, rel=1e-13)               # eq. (43)
            ui = Q[1:4, 0, ji, 0] / Q[0, 0, ji, 0]
            assert np.allclose(Q[1:4, 0, jh, 0], -rm * ui, rtol=1e-14, atol=0)          # eq. (44)-(46)
            ph = (gamma - 1) * (Q[4, 0, jh, 0] - 0.5 * np.sum(Q[1:4, 0, jh, 0] ** 2) / rm)
            assert ph == pytest.approx(p0, rel=1e-12)                                    # halo pressure = p_w
