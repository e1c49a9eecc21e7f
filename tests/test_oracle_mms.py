"""P19 / P20: manufactured-solution pins of the oracle's variable-viscosity and curvilinear viscous terms.

Every other external pin of `viscous_at` (oracle/osbli_oracle.cpp) runs with mu = 1 on a uniform grid (P10: the
Taylor-Green field, where moreover T = 1; P12; the channel pins), so a wrong sign or index in the terms that only
exist when mu varies or when the grid is curved would pass them all.  Here a smooth analytic field with
non-constant rho, u, v, w, T lives on a genuinely non-separable 3-D mapping (every cross metric and every
second-derivative metric is non-zero), with Re = 1 so nothing hides, and the oracle's PART_VISCOUS residual is
compared with the exact

    d_j tau_ij                       (momentum, eq. 2)
    d_j (u_i tau_ij) - d_j q_j       (energy,   PAPER.md:51 eq. 3)
    tau_ij = mu/Re (d_j u_i + d_i u_j - 2/3 delta_ij d_k u_k)        (eq. 5)
    q_j    = -mu / ((gamma-1) M^2 Pr Re) d_j T                       (eq. 4)
    mu     = T^(3/2) (1 + S)/(T + S), S = SuthT/RefT                 (eq. 6, listing at 317-318)

differentiated symbolically (sympy) in PHYSICAL coordinates -- nothing of the oracle's expanded product-rule
form, chain rule or stencils is restated.  The operators are 4th order (eq. 28-29, metrics by the same
operators), so the error must fall >= 12x per grid doubling; any O(1) mistake stops convergence.
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

GAMMA, MACH, PR, RE, S = 1.4, 0.5, 0.72, 1.0, 110.4 / 288.0
TW = 2.0 * np.pi


def _exact_viscous(visc):
    """sympy -> numpy callables f(x,y,z) for rho,u,v,w,T and the exact viscous residual of the 4 equations."""
    import sympy as sp

    x, y, z = sp.symbols("x y z", real=True)
    X = (x, y, z)
    tw = 2 * sp.pi
    rho = 1 + sp.Rational(1, 10) * sp.cos(tw * (x - y + z))
    u = [1 + sp.Rational(3, 10) * sp.sin(tw * (x - z)) * sp.cos(tw * y),
         sp.Rational(1, 5) * sp.cos(tw * (x + y + z)),
         sp.Rational(1, 4) * sp.sin(tw * y) * sp.sin(tw * (z + x))]
    T = 1 + sp.Rational(1, 5) * sp.sin(tw * (x + y)) * sp.cos(tw * z) + sp.Rational(1, 10) * sp.cos(tw * (y - 2 * z))
    Ssym = sp.Rational(1104, 2880)
    mu = T ** sp.Rational(3, 2) * (1 + Ssym) / (T + Ssym) if visc == W.VISC_SUTHERLAND else sp.Integer(1)
    div = sum(sp.diff(u[k], X[k]) for k in range(3))
    tau = [[mu / RE * (sp.diff(u[i], X[j]) + sp.diff(u[j], X[i]) - (sp.Rational(2, 3) * div if i == j else 0))
            for j in range(3)] for i in range(3)]
    q = [-mu / ((GAMMA - 1) * MACH ** 2 * PR * RE) * sp.diff(T, X[j]) for j in range(3)]
    res = [sum(sp.diff(tau[i][j], X[j]) for j in range(3)) for i in range(3)]
    res.append(sum(sp.diff(sum(u[i] * tau[i][j] for i in range(3)) - q[j], X[j]) for j in range(3)))
    fields = [sp.lambdify(X, e, "numpy") for e in (rho, u[0], u[1], u[2], T)]
    return fields, [sp.lambdify(X, e, "numpy") for e in res]


_CACHE = {}


def exact(visc):
    if visc not in _CACHE:
        _CACHE[visc] = _exact_viscous(visc)
    return _CACHE[visc]


def mms_case(n, curved, visc, periodic=True, amp=0.03):
    """Unit box, n^3 nodes.  curved: x = xi + a sin(2pi(xi+eta)) cos(2pi zeta), y = eta + a sin(2pi(eta-zeta))
    sin(2pi xi + 0.3), z = zeta + a cos(2pi(zeta+xi)) sin(2pi eta): no direction separates, all nine first and all
    eighteen second metric derivatives are non-zero."""
    nn = (n, n, n)
    i, j, k = W.padded_index_grids(nn)
    den = float(n if periodic else n - 1)
    xi, et, ze = i / den + 0.0 * j + 0.0 * k, j / den + 0.0 * i + 0.0 * k, k / den + 0.0 * i + 0.0 * j
    a = amp if curved else 0.0
    x = xi + a * np.sin(TW * (xi + et)) * np.cos(TW * ze)
    y = et + a * np.sin(TW * (et - ze)) * np.sin(TW * xi + 0.3)
    z = ze + a * np.cos(TW * (ze + xi)) * np.sin(TW * et)
    fields, _ = exact(visc)
    rho, u, v, w, T = (f(x, y, z) + 0.0 * x for f in fields)
    p = rho * T / (GAMMA * MACH ** 2)
    Q0 = np.ascontiguousarray(W.conservative(rho, u, v, w, p, GAMMA))
    b = (W.BC_PERIODIC,) * 2 if periodic else (W.BC_EXTRAP0,) * 2
    coords = np.ascontiguousarray(np.stack([x, y, z]))
    return W.Case(name="mms", n=nn, Q0=Q0, dt=0.0, nsteps=0, delta=(1.0 / den,) * 3,
                  coords=coords if curved else None, gamma=GAMMA, Re=RE, Pr=PR, Minf=MACH, scheme=W.WENOZ5,
                  visc=visc, suth_ratio=S, bc=(b, b, b)), (x, y, z)


def viscous_error(n, curved, visc, periodic=True, crop=0):
    case, (x, y, z) = mms_case(n, curved, visc, periodic)
    metrics = O.metrics_from_coords(case.coords, case.n, case.periodic) if curved else None
    orc = O.Oracle(metrics=metrics, **case.physics())
    Q = case.Q0.copy()
    if periodic:
        orc.bc(Q)          # non-periodic: halos stay as they are -- the closures eq. (30)-(35) never read them
    R = orc.interior(orc.rhs(Q, parts=O.PART_VISCOUS))
    assert np.all(R[0] == 0.0)                                # the continuity equation has no viscous term
    _, res = exact(visc)
    xi_, yi_, zi_ = (orc.interior(c) for c in (x, y, z))
    out = []
    sl = (slice(crop, n - crop),) * 3
    for c in range(4):
        ex = res[c](xi_, yi_, zi_)
        out.append(float(np.abs(R[1 + c] - ex)[sl].max() / np.abs(ex).max()))
    return np.array(out)


def _assert_fourth_order(curved, visc, periodic=True, sizes=(16, 32), factor=12.0, coarse_max=0.2, crop=0):
    e0 = viscous_error(sizes[0], curved, visc, periodic, crop)
    e1 = viscous_error(sizes[1], curved, visc, periodic, crop)
    assert (e0 < coarse_max).all(), e0
    assert (e1 < e0 / factor).all(), (e0, e1, e0 / e1)
    return e0, e1


def test_p19a_sutherland_uniform_grid():
    """(a) uniform grid, mu(T) of eq. (6).  Catches, in `viscous_at`: the `cross` term sum_j d_j mu (d_j u_i +
    d_i u_j), the `- 2/3 d_i mu div` term, `dmu . dT` in the heat flux, mu multiplying the Laplacians, and
    `prim_of`'s Sutherland law itself (a wrong law gives the wrong d mu everywhere)."""
    _assert_fourth_order(False, W.VISC_SUTHERLAND)


def test_p19b_curvilinear_constant_viscosity():
    """(b) curved grid, mu = 1.  Catches the chain rule of `viscous_at`: `D[k][j]` in the first derivatives, the
    off-diagonal products `D[k][i] * D[l][j]` with the mixed differences delta_kl, and the second-metric term
    `E[l][IJ[i][j]] * c1[f][l]` (E != 0 for all l, ij on this mapping), plus `metrics_from_coords`."""
    _assert_fourth_order(True, W.VISC_CONST)


def test_p19c_curvilinear_sutherland():
    """(c) both at once: d_j mu through the chain rule (`g1[4]` from `c1[4]`)."""
    _assert_fourth_order(True, W.VISC_SUTHERLAND)


def test_p19d_curvilinear_sutherland_closures():
    """Non-periodic in every direction: the one-sided closures eq. (30)-(35) inside the chain rule (mixed
    differences built from closure x closure next to edges) and in the metric generation.  The five-point
    one-sided second differences eq. (34)-(35) are 3rd-order accurate (the first differences eq. (30)-(33) are
    4th), so over all nodes incl. the boundary planes the error falls 8x per doubling (measured 7.4-8.1 between
    33^3 and 65^3); two nodes away from every boundary the interior operators apply and it is 4th order again."""
    _assert_fourth_order(True, W.VISC_SUTHERLAND, periodic=False, sizes=(33, 65), factor=7.0, coarse_max=0.05)
    _assert_fourth_order(True, W.VISC_SUTHERLAND, periodic=False, sizes=(17, 33), factor=12.0, coarse_max=0.05, crop=2)


def test_p19_sensitivity_each_term_matters():
    """The pin is only worth something if each targeted term is large enough to be seen: on the 32^3 curved
    Sutherland case the converged error is < 2e-3 of the residual, while switching off (i) the viscosity
    variation or (ii) the grid curvature in the ORACLE INPUT moves the residual by far more than that."""
    e = viscous_error(32, True, W.VISC_SUTHERLAND)
    assert e.max() < 2e-3, e
    case, _ = mms_case(32, True, W.VISC_SUTHERLAND)
    metrics = O.metrics_from_coords(case.coords, case.n, case.periodic)
    orc = O.Oracle(metrics=metrics, **case.physics())
    Q = orc.bc(case.Q0.copy())
    R = orc.interior(orc.rhs(Q, parts=O.PART_VISCOUS))
    kw = case.physics()
    kw["visc"] = W.VISC_CONST
    R_mu1 = O.Oracle(metrics=metrics, **kw).interior(O.Oracle(metrics=metrics, **kw).rhs(Q, parts=O.PART_VISCOUS))
    flat = {k: (v if k != "E" else [[np.zeros_like(a) for a in row] for row in v]) for k, v in metrics.items()}
    oe = O.Oracle(metrics=flat, **case.physics())
    R_noE = oe.interior(oe.rhs(Q, parts=O.PART_VISCOUS))
    for c in range(1, 5):
        s = np.abs(R[c]).max()
        assert np.abs(R[c] - R_mu1[c]).max() > 0.05 * s, c      # Sutherland terms are > 5 % of the residual
        assert np.abs(R[c] - R_noE[c]).max() > 0.02 * s, c      # second-metric terms are > 2 %


# ------------------------------------------------------------------------------------ P20 ----
def mu_sutherland(T):
    return T ** 1.5 * (1.0 + S) / (T + S)


def dmu_sutherland(T):
    return (1.0 + S) * (1.5 * np.sqrt(T) * (T + S) - T ** 1.5) / (T + S) ** 2


def test_p20_sutherland_law_value():
    """eq. (6) by hand: S = 110.4/288 = 0.383333...; mu(1) = 1 exactly;
    mu(1.5) = 1.5^1.5 * 1.383333/1.883333 = 1.837117 * 0.734513 = 1.349387."""
    assert abs(S - 0.3833333333333333) < 1e-15
    assert mu_sutherland(1.0) == 1.0
    assert abs(mu_sutherland(1.5) - 1.349387) < 2e-6


def test_p20_shear_layer_closed_form():
    """eq. (6) seen through the residual.  u = 1/2 + y, v = w = 0, T = 1 + y/2, p constant on a uniform 2-D grid,
    y non-periodic: every velocity / temperature difference is exact (linear data), so

        R_{rho u} = d_y(mu u_y)/Re                      = mu'(T) T_y u_y / Re
        R_{rho v} = d_y(mu (4/3) v_y) + ...             = 0
        R_{rho E} = d_y(u mu u_y)/Re + cq d_y(mu T_y)   = (u mu' T_y u_y + mu u_y^2)/Re + cq mu' T_y^2

    with only d_y mu approximated (4th order in h on the smooth mu(T(y)): < 1e-7 relative at n_y = 65).  A wrong
    Sutherland law, a wrong sign of `cross` or of `dmu . dT`, or mu missing from tau_ij d_j u_i fails this."""
    n = (8, 65, 1)
    i, j, k = W.padded_index_grids(n)
    y = j / (n[1] - 1.0) + 0.0 * i + 0.0 * k
    Re, Pr, M = 7.0, 0.72, 0.8
    T = 1.0 + 0.5 * y
    u = 0.5 + y
    p = 1.0 / (GAMMA * M * M) + 0.0 * y
    rho = GAMMA * M * M * p / T
    Q0 = np.ascontiguousarray(W.conservative(rho, u, 0.0 * y, 0.0 * y, p, GAMMA))
    per, ex = (W.BC_PERIODIC,) * 2, (W.BC_EXTRAP0,) * 2
    orc = O.Oracle(n=n, delta=(1.0 / n[0], 1.0 / (n[1] - 1.0), 1.0), gamma=GAMMA, Re=Re, Pr=Pr, Minf=M,
                   visc=O.VISC_SUTHERLAND, suth_ratio=S, bc=(per, ex, (0, 0)))
    Q = orc.bc(Q0.copy())
    R = orc.interior(orc.rhs(Q, parts=O.PART_VISCOUS))
    yi, Ti, ui = orc.interior(y), orc.interior(T), orc.interior(u)
    cq = 1.0 / ((GAMMA - 1.0) * M * M * Pr * Re)
    Ty, uy = 0.5, 1.0
    ex_u = dmu_sutherland(Ti) * Ty * uy / Re
    ex_E = (ui * dmu_sutherland(Ti) * Ty * uy + mu_sutherland(Ti) * uy * uy) / Re + cq * dmu_sutherland(Ti) * Ty * Ty
    inner = (yi > 0.04) & (yi < 0.96)          # closure rows have a larger (still 4th-order) error constant
    assert np.abs(R[1] - ex_u)[inner].max() < 1e-7 * np.abs(ex_u).max()
    assert np.abs(R[4] - ex_E)[inner].max() < 1e-7 * np.abs(ex_E).max()
    assert np.abs(R[1] - ex_u).max() < 1e-5 * np.abs(ex_u).max()
    assert np.abs(R[4] - ex_E).max() < 1e-5 * np.abs(ex_E).max()
    assert np.abs(R[2]).max() < 1e-12 and np.abs(R[3]).max() == 0.0 and np.abs(R[0]).max() == 0.0
