"""P12: an independently written, vectorised NumPy statement of the whole residual on tiny grids.

The other pins fix the oracle's parts (reconstruction, eigenvectors, stencils, boundary fills, RK3);
this one fixes their assembly -- indices, signs, which point feeds which stencil slot, the order of
the sweeps -- by writing the algorithm of PAPER.md:100-111 and eq. (2)-(5), (10), (13)-(19), (22)-(29)
a second time in a different shape: whole-array operations on periodically rolled copies, dense 5x5
eigenvector matrices applied with einsum, no loops over points.  It shares nothing with
oracle/osbli_oracle.cpp (triple loops, one interface at a time) beyond the paper.

Uniform grids, periodic boxes in 1-D, 2-D and 3-D, WENO-Z3/Z5/Z7 / TENO5 / TENO6 / WENO-JS5 / central, mu = 1 viscous terms.
(Closures, wall and Dirichlet fills, Sutherland and metric terms are pinned on their own: P6, P11,
P4/P8/P9, P10.)
"""
import numpy as np
import pytest

from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W

G = 1.4


def prim(Q):
    rho = Q[0]
    vel = Q[1:4] / rho
    p = (G - 1.0) * (Q[4] - 0.5 * rho * (vel ** 2).sum(0))
    return rho, vel, p


def weights_and_value(pts, scheme, eps=1e-16, ct=1e-6):
    """pts: the stencil values [a, b, c, d, e(, f)], upwind side a, b, c; interface between c and d."""
    if scheme == W.WENOZ7:
        # k = 4: cubic candidates and the expanded indicators of the 7th-order scheme [18] (pts = nodes i-3..i+3),
        # ideal weights (4, 18, 12, 1)/35 for candidates {i..i+3}, {i-1..i+2}, {i-2..i+1}, {i-3..i}; tau = |beta_0 - beta_3|
        m3, m2, m1, c0, p1, p2, p3 = pts
        q7 = [(3 * c0 + 13 * p1 - 5 * p2 + p3) / 12, (-m1 + 7 * c0 + 7 * p1 - p2) / 12,
              (m2 - 5 * m1 + 13 * c0 + 3 * p1) / 12, (-3 * m3 + 13 * m2 - 23 * m1 + 25 * c0) / 12]
        b7 = [(c0 * (2107 * c0 - 9402 * p1 + 7042 * p2 - 1854 * p3) + p1 * (11003 * p1 - 17246 * p2 + 4642 * p3)
               + p2 * (7043 * p2 - 3882 * p3) + 547 * p3 ** 2) / 240,
              (m1 * (547 * m1 - 2522 * c0 + 1922 * p1 - 494 * p2) + c0 * (3443 * c0 - 5966 * p1 + 1602 * p2)
               + p1 * (2843 * p1 - 1642 * p2) + 267 * p2 ** 2) / 240,
              (m2 * (267 * m2 - 1642 * m1 + 1602 * c0 - 494 * p1) + m1 * (2843 * m1 - 5966 * c0 + 1922 * p1)
               + c0 * (3443 * c0 - 2522 * p1) + 547 * p1 ** 2) / 240,
              (m3 * (547 * m3 - 3882 * m2 + 4642 * m1 - 1854 * c0) + m2 * (7043 * m2 - 17246 * m1 + 7042 * c0)
               + m1 * (11003 * m1 - 9402 * c0) + 2107 * c0 ** 2) / 240]
        t7 = np.abs(b7[0] - b7[3])
        d7 = [4 / 35, 18 / 35, 12 / 35, 1 / 35]
        al7 = [d7[r] * (1 + (t7 / (b7[r] + eps)) ** 2) for r in range(4)]
        return sum(al7[r] * q7[r] for r in range(4)) / sum(al7)
    a, b, c, d, e = pts[:5]
    if scheme == W.WENOZ3:                                  # k = 2: two linear candidates, weights eq. (22)
        q3 = [(c + d) / 2, (-b + 3 * c) / 2]
        be = [(d - c) ** 2, (c - b) ** 2]
        t3 = np.abs(be[0] - be[1])
        al3 = [2 / 3 * (1 + (t3 / (be[0] + eps)) ** 2), 1 / 3 * (1 + (t3 / (be[1] + eps)) ** 2)]
        return (al3[0] * q3[0] + al3[1] * q3[1]) / (al3[0] + al3[1])
    q = [(2 * c + 5 * d - e) / 6, (-b + 5 * c + 2 * d) / 6, (2 * a - 7 * b + 11 * c) / 6]
    beta = [13 / 12 * (c - 2 * d + e) ** 2 + (3 * c - 4 * d + e) ** 2 / 4,
            13 / 12 * (b - 2 * c + d) ** 2 + (b - d) ** 2 / 4,
            13 / 12 * (a - 2 * b + c) ** 2 + (a - 4 * b + 3 * c) ** 2 / 4]
    dw = [0.3, 0.6, 0.1]
    tau = np.abs(beta[0] - beta[2])
    if scheme == W.TENO6:
        f = pts[5]
        q.append((3 * c + 13 * d - 5 * e + f) / 12)
        a1, a2, a3 = (-43 * c + 69 * d - 33 * e + 7 * f) / 24, (2 * c - 5 * d + 4 * e - f) / 2, (-c + 3 * d - 3 * e + f) / 6
        beta.append(a1 ** 2 + 13 / 3 * a2 ** 2 + 3129 / 80 * a3 ** 2 + a1 * a3 / 2)
        dw = [0.3, 0.45, 0.05, 0.2]
        tau = np.abs(beta[3] - (beta[0] + beta[2] + 4 * beta[1]) / 6)
    if scheme == W.WENOJS5:
        al = [dw[r] / (1e-6 + beta[r]) ** 2 for r in range(3)]       # eq. (21), eps = 1e-6
    elif scheme == W.WENOZ5:
        al = [dw[r] * (1 + (tau / (beta[r] + eps)) ** 2) for r in range(3)]
    else:
        gam = [(1 + tau / (beta[r] + eps)) ** 6 for r in range(len(q))]
        gs = sum(gam)
        al = [dw[r] * np.where(gam[r] / gs < ct, 0.0, 1.0) for r in range(len(q))]
    s = sum(al)
    return sum(al[r] / s * q[r] for r in range(len(q)))


def eigenvectors(ut, H, a, n):
    """Dense L (rows) and R (columns) of SURVEY.md 8(c) O2.3 for unit normal n; arrays [..., 5, 5]."""
    u, v, w = ut
    nx, ny, nz = n
    q2 = u * u + v * v + w * w
    th = nx * u + ny * v + nz * w
    b1 = (G - 1) / a ** 2
    b2 = 0.5 * b1 * q2
    one, zero = np.ones_like(u), np.zeros_like(u)
    R = np.stack([
        np.stack([nx * one, u * nx, v * nx + nz, w * nx - ny, 0.5 * q2 * nx + v * nz - w * ny], -1),
        np.stack([ny * one, u * ny - nz, v * ny, w * ny + nx, 0.5 * q2 * ny + w * nx - u * nz], -1),
        np.stack([nz * one, u * nz + ny, v * nz - nx, w * nz, 0.5 * q2 * nz + u * ny - v * nx], -1),
        np.stack([one, u + a * nx, v + a * ny, w + a * nz, H + a * th], -1),
        np.stack([one, u - a * nx, v - a * ny, w - a * nz, H - a * th], -1)], -1)          # [..., component, field]
    L = np.stack([
        np.stack([nx * (1 - b2) - (v * nz - w * ny), nx * b1 * u, nx * b1 * v + nz, nx * b1 * w - ny, -nx * b1 * one], -1),
        np.stack([ny * (1 - b2) - (w * nx - u * nz), ny * b1 * u - nz, ny * b1 * v, ny * b1 * w + nx, -ny * b1 * one], -1),
        np.stack([nz * (1 - b2) - (u * ny - v * nx), nz * b1 * u + ny, nz * b1 * v - nx, nz * b1 * w, -nz * b1 * one], -1),
        0.5 * np.stack([b2 - th / a, -b1 * u + nx / a, -b1 * v + ny / a, -b1 * w + nz / a, b1 * one], -1),
        0.5 * np.stack([b2 + th / a, -b1 * u - nx / a, -b1 * v - ny / a, -b1 * w - nz / a, b1 * one], -1)], -2)   # [..., field, component]
    return L, R, zero


def inviscid_sweep(Q, d, delta, scheme):
    """-(f^_{i+1/2} - f^_{i-1/2})/delta along direction d (0 = x: last axis) on a periodic interior array."""
    ax = -1 - d
    n = np.zeros(3)
    n[d] = 1.0
    at = lambda A, m: np.roll(A, -m, axis=ax)                      # value at node i + m
    rho, vel, p = prim(Q)
    a = np.sqrt(G * p / rho)
    th = vel[d]
    F = np.stack([rho * th, Q[1] * th + p * n[0], Q[2] * th + p * n[1], Q[3] * th + p * n[2], (Q[4] + p) * th])
    lam = [th, th, th, th + a, th - a]
    # Roe average of nodes i, i+1
    wl, wr = np.sqrt(rho), np.sqrt(at(rho, 1))
    ut = (wl * vel + wr * at(vel, 1)) / (wl + wr)
    Hn = (Q[4] + p) / rho
    H = (wl * Hn + wr * at(Hn, 1)) / (wl + wr)
    ar = np.sqrt((G - 1) * (H - 0.5 * (ut ** 2).sum(0)))
    L, R, _ = eigenvectors(ut, H, ar, n)
    ms = list(range(-3, 5)) if scheme == W.WENOZ7 else list(range(-2, 4))
    nw = len(ms)
    V = [np.einsum("...kc,c...->...k", L, at(Q, m)) for m in ms]    # [..., field] at stencil point m
    Gc = [np.einsum("...kc,c...->...k", L, at(F, m)) for m in ms]
    alpha = np.stack([np.max(np.stack([np.abs(at(lam[k], m)) for m in ms]), 0) for k in range(5)], -1)
    gp = [0.5 * (Gc[j] + alpha * V[j]) for j in range(nw)]
    gm = [0.5 * (Gc[j] - alpha * V[j]) for j in range(nw)]
    npts = 7 if scheme == W.WENOZ7 else (6 if scheme == W.TENO6 else 5)
    ghat = weights_and_value(gp[:npts], scheme) + weights_and_value(gm[::-1][:npts], scheme)
    fhat = np.einsum("...ck,...k->c...", R, ghat)                   # f^_{i+1/2}, component first
    return -(fhat - np.roll(fhat, 1, axis=ax)) / delta


def viscous(Q, delta, Re, Pr, M, active):
    rho, vel, p = prim(Q)
    T = G * M * M * p / rho

    def d1(f, k):
        if not active[k]:
            return np.zeros_like(f)
        r = lambda m: np.roll(f, -m, axis=-1 - k)
        return (r(-2) - 8 * r(-1) + 8 * r(1) - r(2)) / (12 * delta[k])

    def d2(f, k):
        if not active[k]:
            return np.zeros_like(f)
        r = lambda m: np.roll(f, -m, axis=-1 - k)
        return (-r(-2) + 16 * r(-1) - 30 * f + 16 * r(1) - r(2)) / (12 * delta[k] ** 2)

    dd = lambda f, k, l: d2(f, k) if k == l else d1(d1(f, max(k, l)), min(k, l))     # delta_k(delta_l f), k < l
    grad = [[d1(vel[i], j) for j in range(3)] for i in range(3)]
    div = grad[0][0] + grad[1][1] + grad[2][2]
    Mi = [sum(d2(vel[i], j) for j in range(3)) + sum(dd(vel[k], i, k) for k in range(3)) / 3 for i in range(3)]
    out = np.zeros_like(Q)
    for i in range(3):
        out[1 + i] = Mi[i] / Re
    phi = sum((grad[i][j] + grad[j][i] - (2 / 3 * div if i == j else 0.0)) * grad[i][j] for i in range(3) for j in range(3)) / Re
    cq = 1.0 / ((G - 1) * M * M * Pr * Re)
    out[4] = sum(vel[i] * Mi[i] for i in range(3)) / Re + phi + cq * sum(d2(T, j) for j in range(3))
    return out


def central_sweep(Q, d, delta):
    """-(F_{i-2} - 8 F_{i-1} + 8 F_{i+1} - F_{i+2})/(12 delta): eq. (28) applied to the point-wise flux vectors."""
    ax = -1 - d
    rho, vel, p = prim(Q)
    n = np.zeros(3)
    n[d] = 1.0
    th = vel[d]
    F = np.stack([rho * th, Q[1] * th + p * n[0], Q[2] * th + p * n[1], Q[3] * th + p * n[2], (Q[4] + p) * th])
    r = lambda m: np.roll(F, -m, axis=ax)
    return -(r(-2) - 8 * r(-1) + 8 * r(1) - r(2)) / (12 * delta)


def brute_residual(case, scheme, visc):
    h, n = case.halo, case.n
    Q = case.Q0[:, h[2]:h[2] + n[2], h[1]:h[1] + n[1], h[0]:h[0] + n[0]].copy()
    active = [v > 1 for v in n]
    R = np.zeros_like(Q)
    for d in range(3):
        if active[d]:
            R += central_sweep(Q, d, case.delta[d]) if scheme == W.CENTRAL4 else inviscid_sweep(Q, d, case.delta[d], scheme)
    if visc:
        R += viscous(Q, case.delta, case.Re, case.Pr, case.Minf, active)
    return R


def box(n, seed, scheme=None):
    rng = np.random.default_rng(seed)
    i, j, k = W.padded_index_grids(n, scheme)
    x, y, z = 2 * np.pi * i / n[0], 2 * np.pi * j / n[1], 2 * np.pi * k / n[2]
    ph = rng.uniform(0, 2 * np.pi, 8)
    rho = 1.0 + 0.3 * np.sin(x + ph[0]) * np.cos(y + ph[1]) + 0.1 * np.cos(z + ph[2])
    u = 0.5 * np.sin(x + y + ph[3]) + 0.2 * np.cos(z + ph[4])
    v = (0.4 * np.cos(x - y + ph[5]) + 0.0 * z) if n[1] > 1 else 0.0 * x
    w = (0.3 * np.sin(z + x + ph[6]) + 0.0 * y) if n[2] > 1 else 0.0 * x
    p = 1.0 + 0.3 * np.cos(x + ph[7]) * np.sin(y + z)
    # one steep feature so that the nonlinear weights (and the TENO cut-off) actually do something
    rho = rho + 0.8 * (np.tanh(4 * np.sin(x)) > 0.5)
    per = (W.BC_PERIODIC, W.BC_PERIODIC)
    bc = tuple(per if n[d] > 1 else (0, 0) for d in range(3))
    return W.Case(name="brute", n=n, Q0=np.ascontiguousarray(W.conservative(rho, u, v, w, p, G)), dt=1e-3, nsteps=1,
                  delta=tuple(2 * np.pi / v_ for v_ in n), gamma=G, Re=50.0, Pr=0.71, Minf=0.7, bc=bc,
                  **({} if scheme is None else {"scheme": scheme}))


@pytest.mark.parametrize("scheme", [W.WENOZ5, W.TENO5, W.TENO6, W.WENOJS5, W.CENTRAL4, W.WENOZ3, W.WENOZ7])
@pytest.mark.parametrize("n", [(8, 6, 5), (12, 10, 1), (16, 1, 1)])
@pytest.mark.parametrize("visc", [W.VISC_NONE, W.VISC_CONST])
def test_p12_oracle_equals_vectorised_numpy(scheme, n, visc):
    case = box(n, seed=sum(n) + scheme, scheme=scheme if scheme == W.WENOZ7 else None)      # the 7th-order scheme: halo 4
    orc = O.Oracle(**{**case.physics(), "scheme": scheme, "visc": visc, "eps": 1e-6 if scheme == W.WENOJS5 else 1e-16})
    Ro = orc.interior(orc.rhs(orc.bc(case.Q0.copy())))
    Rb = brute_residual(case, scheme, visc != W.VISC_NONE)
    scale = np.abs(Ro).max(axis=(1, 2, 3), keepdims=True)
    scale = np.where(scale < 1e-12 * scale.max(), scale.max(), scale)
    assert (np.abs(Ro - Rb) / scale).max() < 1e-12, (np.abs(Ro - Rb) / scale).max(axis=(1, 2, 3))
