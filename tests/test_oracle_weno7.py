"""Pins of the oracle's 7th-order WENO-Z reconstruction (oracle_reconstruct7; "any arbitrary odd
order", eq. (15)-(16), (20), (22); used at 7th order in PAPER.md:485-495, 531-533; Q40).

The paper prints the 5th-order candidates and indicators only.  The 7th-order ones follow from definitions it does
give, and each derived piece is pinned here by something other than the oracle's own formula:
  * candidates q_r and indicators beta_r: symbolic integration of eq. (16) on the interpolating cubics (sympy);
  * tau_7 = |beta_0 - beta_3| (the reading Q40), read back from the oracle's indicator output;
  * ideal weights: on smooth data the value is the 7th-order one, whose coefficients are derived here from the
    degree-6 interpolant; the derivative built on it converges at 7th order (error ratio 2^7 per halving);
  * ENO property: next to a jump only the candidates that do not cross it contribute;
  * the residual built on it (halo depth 4): conservation, mirror symmetry, free stream, periodic halo fill.
(The assembly of the 8-point window into the residual is pinned by P12, tests/test_oracle_bruteforce.py.)
"""
import numpy as np
import pytest
import sympy as sp

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

HALF = sp.Rational(1, 2)


def _interp(cells, values):
    """The polynomial whose cell averages over the unit cells centred at `cells` are `values`."""
    x = sp.symbols("x")
    co = sp.symbols(f"a0:{len(cells)}")
    p = sum(co[k] * x ** k for k in range(len(cells)))
    eqs = [sp.integrate(p, (x, c - HALF, c + HALF)) - v for c, v in zip(cells, values)]
    return x, p.subs(sp.solve(eqs, co))


def _jiang_shu(cells, values):
    x, p = _interp(cells, values)
    beta = sum(sp.integrate(sp.diff(p, x, l) ** 2, (x, -HALF, HALF)) for l in range(1, len(cells)))
    return p.subs(x, HALF), beta


def test_candidates_and_indicators_match_eq16():
    """Would catch a wrong Taylor coefficient, a swapped stencil or a wrong 3129/80, 13/3, 1/2 in reconstruct7."""
    rng = np.random.default_rng(7)
    for _ in range(3):
        v = [sp.Rational(int(t), 16) for t in rng.integers(-40, 40, size=7)]
        exact = [_jiang_shu(list(range(-r, 4 - r)), v[3 - r:7 - r])[1] for r in range(4)]
        _, ind = O.reconstruct7([float(t) for t in v], with_indicators=True)
        np.testing.assert_allclose(ind[:4], [float(t) for t in exact], rtol=1e-13)
        np.testing.assert_allclose(ind[4], abs(float(exact[0] - exact[3])), rtol=1e-11, atol=1e-12)   # Q40


def test_smooth_limit_is_the_seventh_order_value():
    """Ideal weights d_r = (4, 18, 12, 1)/35 and the four candidates: with tau -> 0 against beta the value is the one
    of the degree-6 interpolant.  Probed by differentiating about a ramp (beta_r all equal, tau = 0)."""
    sym = sp.symbols("v0:7")
    x, p = _interp(list(range(-3, 4)), sym)
    lin = sp.Poly(p.subs(x, HALF), *sym)
    want = [float(lin.coeff_monomial(s)) for s in sym]
    base = np.array([0.5 * k for k in range(7)])
    w0 = O.reconstruct7(base)
    got = []
    for j in range(7):
        v = base.copy()
        v[j] += 1e-5                                          # the weights move by O(perturbation^2)
        got.append((O.reconstruct7(v) - w0) / 1e-5)
    np.testing.assert_allclose(got, want, atol=1e-9)
    np.testing.assert_allclose(want, np.array([-3, 25, -101, 319, 214, -38, 4]) / 420.0, atol=1e-15)


def _derivative_error(h):
    f = lambda t: np.sin(t) + 2.0 * t                       # f' = cos + 2 > 0: no critical point
    xs = 0.3 + h * np.arange(-4, 5)
    fh = [O.reconstruct7(f(xs[i - 3:i + 4])) for i in (3, 4)]        # f^_{i-1/2}, f^_{i+1/2} about xs[4]
    return abs((fh[1] - fh[0]) / h - (np.cos(xs[4]) + 2.0))


def test_seventh_order_convergence():
    e1, e2 = _derivative_error(0.2), _derivative_error(0.1)
    assert e2 > 1e-13                                         # above round-off
    assert abs(np.log2(e1 / e2) - 7.0) < 0.35, (e1, e2)


def test_eno_property_next_to_a_jump():
    """Data cubic on nodes i-3..i (a jump behind node i): only candidate r = 3 is smooth and the value is the cubic's."""
    x = sp.symbols("x")
    poly = 1 + x / 3 - x ** 2 / 7 + x ** 3 / 50
    avg = [float(sp.integrate(poly, (x, k - HALF, k + HALF))) for k in range(-3, 1)]
    val = O.reconstruct7(avg + [40.0, -25.0, 60.0])
    assert abs(val - float(poly.subs(x, HALF))) < 1e-5        # WENO weights of the crossing stencils: O((beta_smooth/tau)^2), not 0
    # mirrored: jump in front of node i, smooth on i..i+3
    avg = [float(sp.integrate(poly, (x, k - HALF, k + HALF))) for k in range(0, 4)]
    val = O.reconstruct7([40.0, -25.0, 60.0] + avg)
    assert abs(val - float(poly.subs(x, HALF))) < 1e-5


def _line(nx=24, seed=5):
    rng = np.random.default_rng(seed)
    n = (nx, 1, 1)
    i, _, _ = W.padded_index_grids(n, W.WENOZ7)
    x = 2 * np.pi * i / nx
    ph = rng.uniform(0, 2 * np.pi, 4)
    rho = 1.0 + 0.3 * np.sin(x + ph[0]) + 0.5 * (np.sin(x) > 0.3)
    u = 0.4 * np.cos(x + ph[1])
    p = 1.0 + 0.2 * np.sin(2 * x + ph[2])
    Q0 = np.ascontiguousarray(W.conservative(rho, u, 0.0, 0.0, p, 1.4))
    per = (W.BC_PERIODIC, W.BC_PERIODIC)
    return W.Case(name="line7", n=n, Q0=Q0, dt=1e-3, nsteps=1, delta=(2 * np.pi / nx, 1.0, 1.0), scheme=W.WENOZ7,
                  bc=(per, (0, 0), (0, 0)))


def test_halo_depth_and_periodic_fill():
    case = _line()
    assert case.halo == (4, 0, 0)
    orc = O.Oracle(**case.physics())
    assert orc.h == (4, 0, 0) and orc.shape == case.Q0.shape
    Q = case.Q0.copy()
    Q[..., :4] = -7.0
    Q[..., -4:] = -7.0
    Q = orc.bc(Q)
    np.testing.assert_array_equal(Q[..., :4], Q[..., -8:-4])
    np.testing.assert_array_equal(Q[..., -4:], Q[..., 4:8])


def test_residual_conservation_mirror_and_free_stream():
    case = _line()
    orc = O.Oracle(**case.physics())
    R = orc.interior(orc.rhs(orc.bc(case.Q0.copy())))
    scale = np.abs(R).max()
    assert np.abs(R.sum(axis=-1)).max() < 1e-12 * scale * R.shape[-1]          # telescoping flux differences
    # mirror image x -> -x, u -> -u: the residual mirrors (rho, E even; momentum odd)
    Qm = orc.interior(case.Q0)[..., ::-1].copy()
    Qm[1] *= -1.0
    Rm = orc.interior(orc.rhs(orc.bc(orc.pad(Qm))))
    sign = np.array([1.0, -1.0, 1.0, 1.0, 1.0])[:, None, None, None]
    np.testing.assert_allclose(Rm, sign * R[..., ::-1], atol=1e-11 * scale)
    # uniform flow: zero residual
    Qc = np.ascontiguousarray(np.broadcast_to(W.conservative(1.1, 0.3, 0.0, 0.0, 0.9, 1.4).reshape(5, 1, 1, 1), case.Q0.shape))
    assert np.abs(orc.interior(orc.rhs(orc.bc(Qc.copy())))).max() < 1e-13


# ------------------------- the whole Euler path against an exact solution, PAPER.md:497-533 --
def _wave_error(N, scheme, dt, t_end, curvilinear):
    c = W.euler_wave(N, scheme=scheme, dt=dt, t_end=t_end, curvilinear=curvilinear)
    metrics = O.metrics_from_coords(c.coords, c.n, c.periodic, delta=c.delta, scheme=scheme) if curvilinear else None
    o = O.Oracle(metrics=metrics, **c.physics())
    Q = c.Q0.copy()
    o.run(Q, c.dt, c.nsteps)
    e = np.abs(o.interior(Q)[0] - c.extra["rho_exact"])
    return e.mean(), e.max()


def test_euler_wave_converges_at_seventh_order_on_the_uniform_mesh():
    """Travelling density wave eq. (47) on the uniform periodic mesh: halo fill (depth 4), 8-point characteristic
    reconstruction in both directions, flux differences and RK3 together reach the exact solution at 7th order
    ("within 10 % of the formal order"); would catch a wrong window index, weight or mirror image in the
    assembly that the point-wise pins above cannot see."""
    import math
    a = _wave_error(16, W.WENOZ7, 5e-4, 0.25, False)
    b = _wave_error(32, W.WENOZ7, 2.5e-4, 0.25, False)
    r1, rinf = math.log2(a[0] / b[0]), math.log2(a[1] / b[1])
    assert r1 > 6.3 and rinf > 6.3, (a, b, r1, rinf)
    assert b[1] < 2e-8


def test_euler_wave_on_the_sinusoidal_mesh():
    """The same on the mesh of eq. (48)-(49): point-wise area-weighted normals over the 8-point window, interface
    normal from nodes i, i+1.  The metric terms are 4th-order central differences (eq. (28)), so the
    curvilinear scheme is formally 4th order whatever the reconstruction (Q42): 7Z must converge at that
    rate and beat 5Z's error on both grids."""
    import math
    z7 = [_wave_error(N, W.WENOZ7, dt, 0.5, True) for N, dt in ((32, 1e-3), (64, 5e-4))]
    z5 = [_wave_error(N, W.WENOZ5, dt, 0.5, True) for N, dt in ((32, 1e-3), (64, 5e-4))]
    r1, rinf = math.log2(z7[0][0] / z7[1][0]), math.log2(z7[0][1] / z7[1][1])
    assert r1 > 3.7 and rinf > 3.6, (z7, r1, rinf)
    assert z7[0][0] < 0.6 * z5[0][0] and z7[1][0] < 0.8 * z5[1][0], (z7, z5)
