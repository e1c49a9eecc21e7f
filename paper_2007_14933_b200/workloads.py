"""Seeded, synthetic input generators for the five BASELINE.json configurations (+ pin cases).

This module holds NO arithmetic of the method (no reconstruction, no flux, no difference
stencil, no boundary formula): it only evaluates analytic initial fields and grid coordinates
and packs them.  It is the one module both the CPU oracle's tests and the CUDA path's
tests/bench import, so that both sides receive identical bytes.

Exchange format ("dense padded"): a scalar field is a float64 array [NZ, NY, NX] with
N_d = n_d + 2 h_d, h_d = 3 if n_d > 1 else 0; a state is [5, NZ, NY, NX] holding
(rho, rho u, rho v, rho w, rho E).  Halo entries of an initial state are an
edge copy (they are overwritten by the first boundary fill).

Recipes: DESIGN.md "Input recipe"; PAPER.md:469-479 (Sod), 497-511 (Euler wave on the
sinusoidal mesh), 623 (Taylor-Green vortex), 576-601 (SBLI set-up the slab case is modelled on).
"""
from __future__ import annotations

from dataclasses import dataclass, field
from typing import Optional

import numpy as np

WENOZ5, TENO5, TENO6, WENOJS5, CENTRAL4, WENOZ3, WENOZ7 = 0, 1, 2, 3, 4, 5, 6
VISC_NONE, VISC_CONST, VISC_SUTHERLAND = 0, 1, 2
BC_PERIODIC, BC_EXTRAP0, BC_DIRICHLET, BC_WALL_ISOTHERMAL, BC_WALL_ADIABATIC = 0, 1, 2, 3, 4
AVG_ROE, AVG_SIMPLE = 0, 1
RK3_WILLIAMSON, RK3_SSP = 0, 1


@dataclass
class Case:
    name: str
    n: tuple                                   # (nx, ny, nz)
    Q0: np.ndarray                             # [5, NZ, NY, NX] dense padded
    dt: float
    nsteps: int
    delta: tuple = (1.0, 1.0, 1.0)             # uniform spacing (uniform mode)
    coords: Optional[np.ndarray] = None        # [3, NZ, NY, NX] node coordinates => curvilinear mode
    gamma: float = 1.4
    Re: float = 1.0
    Pr: float = 1.0
    Minf: float = 1.0
    scheme: int = WENOZ5
    teno_ct: float = 1e-6
    eps: float = 1e-16
    visc: int = VISC_NONE
    suth_ratio: float = 110.4 / 288.0
    bc: tuple = ((0, 0), (0, 0), (0, 0))
    wall_T: tuple = ((0.0, 0.0), (0.0, 0.0), (0.0, 0.0))
    dirichlet: Optional[np.ndarray] = None     # [5, NZ, NY, NX] frozen boundary state
    force: tuple = (0.0, 0.0, 0.0)             # constant body force per unit volume
    averaging: int = AVG_ROE                   # interface state of step 2(a)
    rk3_form: int = RK3_WILLIAMSON             # coefficient set of the 3-stage scheme
    extra: dict = field(default_factory=dict)  # analytic solutions etc. for the pins

    @property
    def halo(self):
        return halo_of(self.n, self.scheme)

    @property
    def periodic(self):
        return tuple(self.bc[d][0] == BC_PERIODIC for d in range(3))

    @property
    def npoints(self):
        return int(self.n[0]) * int(self.n[1]) * int(self.n[2])

    def physics(self):
        """Keyword arguments shared by both back-ends' constructors (metrics excluded)."""
        return dict(n=self.n, delta=self.delta, gamma=self.gamma, Re=self.Re, Pr=self.Pr, Minf=self.Minf,
                    scheme=self.scheme, teno_ct=self.teno_ct, eps=self.eps, visc=self.visc,
                    suth_ratio=self.suth_ratio, bc=self.bc, wall_T=self.wall_T, dirichlet=self.dirichlet,
                    force=self.force, averaging=self.averaging, rk3_form=self.rk3_form)


# ------------------------------------------------------------------------------ helpers ----
def halo_of(n, scheme=None):
    """Ghost points per side: 3, 4 for the 7th-order scheme (stencil i-3..i+4); 0 in a collapsed direction."""
    depth = 4 if scheme == WENOZ7 else 3
    return tuple(depth if v > 1 else 0 for v in n)


def padded_index_grids(n, scheme=None):
    """Integer node indices (i, j, k) on the dense padded grid, as broadcastable arrays."""
    h = halo_of(n, scheme)
    i = np.arange(-h[0], n[0] + h[0])[None, None, :]
    j = np.arange(-h[1], n[1] + h[1])[None, :, None]
    k = np.arange(-h[2], n[2] + h[2])[:, None, None]
    return i, j, k


def conservative(rho, u, v, w, p, gamma):
    """Pack primitive fields into the 5-variable conservative state (eq. 7)."""
    shape = np.broadcast_shapes(*(np.shape(a) for a in (rho, u, v, w, p)))
    rho, u, v, w, p = (np.broadcast_to(np.asarray(a, dtype=np.float64), shape) for a in (rho, u, v, w, p))
    Q = np.empty((5,) + shape)
    Q[0] = rho
    Q[1] = rho * u
    Q[2] = rho * v
    Q[3] = rho * w
    Q[4] = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return Q


def edge_pad_interior(A, n, scheme=None):
    """Overwrite halo entries of dense padded array(s) [..., NZ, NY, NX] by an edge copy."""
    h = halo_of(n, scheme)
    core = A[..., h[2]:h[2] + n[2], h[1]:h[1] + n[1], h[0]:h[0] + n[0]]
    pw = [(0, 0)] * (A.ndim - 3) + [(h[2],) * 2, (h[1],) * 2, (h[0],) * 2]
    return np.ascontiguousarray(np.pad(core, pw, mode="edge"))


def splitmix64_unit(seed, index):
    """Counter-based uniform numbers in [-1, 1): splitmix64(seed + index) -> top 53 bits."""
    z = (np.asarray(index, dtype=np.uint64) + np.uint64(seed)) + np.uint64(0x9E3779B97F4A7C15)
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) / float(1 << 52) - 1.0


# --------------------------------------------------------------------------------- C1 ------
def sod(nx=400, scheme=WENOZ5, dt=2e-4, nsteps=1000):
    """1-D Sod shock tube (BASELINE.json config 1).  x_i = i/(nx-1)."""
    n = (nx, 1, 1)
    i, _, _ = padded_index_grids(n, scheme)
    x = i / (nx - 1.0)
    left = x < 0.5
    rho = np.where(left, 1.0, 0.125)
    p = np.where(left, 1.0, 0.1)
    Q0 = conservative(rho, 0.0, 0.0, 0.0, p, 1.4)
    Q0 = edge_pad_interior(Q0, n, scheme)
    return Case(name=f"sod{nx}", n=n, Q0=Q0, dt=dt, nsteps=nsteps, delta=(1.0 / (nx - 1.0), 1.0, 1.0),
                gamma=1.4, Minf=1.0, scheme=scheme, visc=VISC_NONE,
                bc=((BC_EXTRAP0, BC_EXTRAP0), (0, 0), (0, 0)),
                extra={"x": np.arange(nx) / (nx - 1.0), "t_end": dt * nsteps})


def shu_osher(nx=320, scheme=WENOZ5, dt=2e-4, nsteps=9000):
    """1-D shock / density-wave interaction: x in [-5, 5], Dirichlet ends, t_end = 1.8.

    Left of x = -4 the post-shock state (3.857143, 2.629369, 10.33333); right of it rho = 1 + 0.2 sin(5x) at rest
    with p = 1 (the printed "(.., 1.0, 0.0)" has u and p swapped: p = 0 is not a state; Q41)."""
    n = (nx, 1, 1)
    i, _, _ = padded_index_grids(n, scheme)
    x = -5.0 + 10.0 * i / (nx - 1.0)
    left = x < -4.0
    rho = np.where(left, 3.857143, 1.0 + 0.2 * np.sin(5.0 * x))
    u = np.where(left, 2.629369, 0.0)
    p = np.where(left, 10.33333, 1.0)
    Q0 = np.ascontiguousarray(conservative(rho, u, 0.0, 0.0, p, 1.4))
    return Case(name=f"shu_osher{nx}", n=n, Q0=Q0, dt=dt, nsteps=nsteps, delta=(10.0 / (nx - 1.0), 1.0, 1.0),
                gamma=1.4, Minf=1.0, scheme=scheme, visc=VISC_NONE,
                bc=((BC_DIRICHLET, BC_DIRICHLET), (0, 0), (0, 0)), dirichlet=Q0.copy(),
                extra={"x": -5.0 + 10.0 * np.arange(nx) / (nx - 1.0), "t_end": dt * nsteps})


# ----------------------------------------------------------------------------- C2/C3/C5 ----
_TGV_DT = {64: (3.385e-3, 100), 256: (8.5e-4, 200), 512: (4.2e-4, 50)}


def tgv(n=64, scheme=TENO5, visc=VISC_CONST, dt=None, nsteps=None, M=0.1, Re=1600.0, Pr=0.71):
    """3-D viscous Taylor-Green vortex on [0, 2 pi)^3 (BASELINE.json configs 2, 3, 5)."""
    nn = (n, n, n)
    i, j, k = padded_index_grids(nn, scheme)
    h = 2.0 * np.pi / n
    x, y, z = i * h, j * h, k * h
    gamma = 1.4
    u = np.sin(x) * np.cos(y) * np.cos(z)
    v = -np.cos(x) * np.sin(y) * np.cos(z)
    p = 1.0 / (gamma * M * M) + (np.cos(2 * x) + np.cos(2 * y)) * (np.cos(2 * z) + 2.0) / 16.0
    rho = gamma * M * M * p
    Q0 = np.ascontiguousarray(conservative(rho, u, v, 0.0, p, gamma))
    if dt is None or nsteps is None:
        d0, s0 = _TGV_DT.get(n, (3.385e-3 * 64.0 / n, 10))
        dt = d0 if dt is None else dt
        nsteps = s0 if nsteps is None else nsteps
    per = (BC_PERIODIC, BC_PERIODIC)
    return Case(name=f"tgv{n}", n=nn, Q0=Q0, dt=dt, nsteps=nsteps, delta=(h, h, h), gamma=gamma, Re=Re, Pr=Pr,
                Minf=M, scheme=scheme, visc=visc, bc=(per, per, per))


# ------------------------------------------------------------- Euler wave, sinusoidal mesh --
def euler_wave(N=32, scheme=WENOZ5, A=0.04, dt=5e-4, t_end=2.5, curvilinear=True):
    """2-D travelling density wave on the sinusoidal mesh (eq. 47-49).

    rho = 1 + 0.2 sin(pi (x + y - t (u + v))), u = 1, v = -0.5, p = 1; periodic, L_x = L_y = 2.
    """
    n = (N, N, 1)
    i, j, k = padded_index_grids(n, scheme)
    L = 2.0
    d = L / N
    x = i * d + A * np.sin(6.0 * np.pi * j * d / L) + 0.0 * k
    y = j * d + A * np.sin(6.0 * np.pi * i * d / L) + 0.0 * k
    if not curvilinear:
        x = i * d + 0.0 * j + 0.0 * k
        y = j * d + 0.0 * i + 0.0 * k
    u0, v0, p0, gamma = 1.0, -0.5, 1.0, 1.4

    def rho_exact(xx, yy, t):
        return 1.0 + 0.2 * np.sin(np.pi * (xx + yy - t * (u0 + v0)))

    Q0 = np.ascontiguousarray(conservative(rho_exact(x, y, 0.0), u0, v0, 0.0, p0, gamma))
    coords = np.ascontiguousarray(np.stack([x, y, np.zeros_like(x)])) if curvilinear else None
    per = (BC_PERIODIC, BC_PERIODIC)
    nsteps = int(round(t_end / dt))
    h = halo_of(n, scheme)
    xi = x[:, h[1]:h[1] + N, h[0]:h[0] + N]
    yi = y[:, h[1]:h[1] + N, h[0]:h[0] + N]
    return Case(name=f"wave{N}", n=n, Q0=Q0, dt=dt, nsteps=nsteps, delta=(d, d, 1.0), coords=coords, gamma=gamma,
                Minf=1.0, scheme=scheme, visc=VISC_NONE, bc=(per, per, (0, 0)),
                extra={"rho_exact": rho_exact(xi, yi, dt * nsteps), "t_end": dt * nsteps})


# --------------------------------------------------------------------------------- C4 ------
def sutherland(T, S=110.4 / 288.0):
    """mu(T) of the problem statement -- used here only to build the inflow profile."""
    return T ** 1.5 * (1.0 + S) / (T + S)


def similarity_boundary_layer(M=2.0, Pr=0.72, gamma=1.4, S=110.4 / 288.0, eta_max=12.0, n_eta=2400):
    """Compressible laminar similarity profile over an adiabatic wall (White, ref. [61] of the paper;
    the SBLI inflow of PAPER.md:576-601 is such a profile):

        (C f'')' + f f'' = 0,   (C g'/Pr)' + f g' + (gamma-1) M^2 C f''^2 = 0,   C = mu(g)/g,
        f(0) = f'(0) = 0, g'(0) = 0, f'(inf) = g(inf) = 1,

    f' = u/u_e, g = T/T_e, eta the Illingworth-Levy variable.  Classical RK4 on a fixed grid and Newton
    shooting on (f''(0), g(0)).  Returns eta, f', g, Y = int_0^eta g and I = int (g - f') d eta.
    """
    h = eta_max / n_eta
    gm = (gamma - 1.0) * M * M

    def rhs(y):
        f, fp, s, g, q = y
        C = sutherland(g, S) / g
        fpp = s / C
        gp = Pr * q / C
        return np.array([fp, fpp, -f * fpp, gp, -f * gp - gm * s * s / C])

    def shoot(fpp0, g0, full=False):
        C0 = sutherland(g0, S) / g0
        y = np.array([0.0, 0.0, C0 * fpp0, g0, 0.0])
        out = [y.copy()] if full else None
        for _ in range(n_eta):
            k1 = rhs(y); k2 = rhs(y + 0.5 * h * k1); k3 = rhs(y + 0.5 * h * k2); k4 = rhs(y + h * k3)
            y = y + (h / 6.0) * (k1 + 2 * k2 + 2 * k3 + k4)
            if full:
                out.append(y.copy())
        return (np.array(out) if full else None), np.array([y[1] - 1.0, y[3] - 1.0])

    x = np.array([0.5, 1.0 + 0.5 * np.sqrt(Pr) * gm])          # recovery-factor guess for g(0)
    for _ in range(30):
        _, r = shoot(x[0], x[1])
        if np.abs(r).max() < 1e-13:
            break
        J = np.empty((2, 2))
        for c in range(2):
            d = np.zeros(2); d[c] = 1e-7
            _, rp = shoot(*(x + d))
            J[:, c] = (rp - r) / 1e-7
        x = x - np.linalg.solve(J, r)
    sol, _ = shoot(x[0], x[1], full=True)
    eta = h * np.arange(n_eta + 1)
    fp, g = sol[:, 1], sol[:, 3]
    trap = lambda a: np.concatenate([[0.0], np.cumsum(0.5 * h * (a[1:] + a[:-1]))])
    Y = trap(g)
    I = trap(g - fp)[-1]
    return dict(eta=eta, fp=fp, g=g, Y=Y, I=float(I), fpp0=float(x[0]), g0=float(x[1]))


def oblique_shock(M=2.0, beta_deg=32.58, gamma=1.4):
    """Rankine-Hugoniot state behind an oblique shock of angle beta in a (rho, u, v, p) = (1, 1, 0, 1/(gamma M^2))
    stream, turning the flow towards the wall (v < 0)."""
    b = np.deg2rad(beta_deg)
    mn2 = (M * np.sin(b)) ** 2
    pr = 1.0 + 2.0 * gamma / (gamma + 1.0) * (mn2 - 1.0)
    rr = (gamma + 1.0) * mn2 / ((gamma - 1.0) * mn2 + 2.0)
    ut, un2 = np.cos(b), np.sin(b) / rr
    return dict(rho=rr, u=ut * np.cos(b) + un2 * np.sin(b), v=-(ut * np.sin(b) - un2 * np.cos(b)),
                p=pr / (gamma * M * M), p_ratio=pr, rho_ratio=rr)


def sbli_slab(n=(500, 250, 8), seed=2007014933, noise=1e-4, dt=1e-3, nsteps=500, scheme=WENOZ5, x_shock=20.0):
    """BASELINE.json config 4: quasi-2-D laminar shock / boundary-layer interaction slab on a curvilinear grid
    (recipe: DESIGN.md "Input recipe"; set-up modelled on PAPER.md:576-601).  `n` can be reduced for quick runs:
    the domain, the stretching and the flow stay the same."""
    n = tuple(int(v) for v in n)
    nx, ny, nz = n
    gamma, M, Re, Pr, S = 1.4, 2.0, 950.0, 0.72, 110.4 / 288.0
    Lx, Ly, dz = 300.0, 115.0, 0.6
    i, j, k = padded_index_grids(n)
    xi = i / (nx - 1.0) + 0.0 * j + 0.0 * k
    et = j / (ny - 1.0) + 0.0 * i + 0.0 * k
    x = Lx * (xi + 0.01 * np.sin(4.0 * np.pi * xi) * np.sin(4.0 * np.pi * et))
    y = Ly * (1.0 + np.tanh(2.5 * (et - 1.0)) / np.tanh(2.5))
    z = dz * k + 0.0 * i + 0.0 * j
    coords = np.ascontiguousarray(np.stack([x, y, z]))

    bl = similarity_boundary_layer(M, Pr, gamma, S)
    x0 = Re / (2.0 * bl["I"] ** 2)                              # delta* = 1 at the inflow
    ysim = np.sqrt(2.0 * x0 / Re) * bl["Y"]
    yy = np.clip(y, 0.0, None)
    u = np.interp(yy, ysim, bl["fp"], right=1.0)
    T = np.interp(yy, ysim, bl["g"], right=1.0)
    p0 = 1.0 / (gamma * M * M)
    rho = 1.0 / T
    clean = np.ascontiguousarray(conservative(rho, u, 0.0 * u, 0.0 * u, p0 + 0.0 * u, gamma))
    clean = edge_pad_interior(clean, n)

    # frozen boundary state: inflow profile; top boundary free stream up to x_shock, post-shock state behind
    dirichlet = clean.copy()
    sh = oblique_shock(M, 32.58, gamma)
    post = conservative(sh["rho"], sh["u"], sh["v"], 0.0, sh["p"], gamma)
    free = conservative(1.0, 1.0, 0.0, 0.0, p0, gamma)
    h = halo_of(n)
    top = slice(h[1] + ny - 1, None)
    behind = (x[:, top, :] >= x_shock)
    for c in range(5):
        dirichlet[c][:, top, :] = np.where(behind, post[c], free[c])

    # seeded density noise on interior nodes; u, v, w, p unchanged
    ii, jj, kk = np.meshgrid(np.arange(nx), np.arange(ny), np.arange(nz), indexing="ij")
    lin = (ii + nx * (jj + ny * kk)).astype(np.uint64)
    r = splitmix64_unit(seed, lin).transpose(2, 1, 0)           # [nz, ny, nx]
    core = (slice(h[2], h[2] + nz), slice(h[1], h[1] + ny), slice(h[0], h[0] + nx))
    rho_n = rho.copy() + 0.0 * k
    rho_n = np.broadcast_to(rho_n, clean[0].shape).copy()
    rho_n[core] *= (1.0 + noise * r)
    ub = np.broadcast_to(u, clean[0].shape)
    Q0 = conservative(rho_n, ub, 0.0 * ub, 0.0 * ub, p0 + 0.0 * ub, gamma)
    Q0 = edge_pad_interior(np.ascontiguousarray(Q0), n)

    per = (BC_PERIODIC, BC_PERIODIC)
    bc = ((BC_DIRICHLET, BC_EXTRAP0), (BC_WALL_ISOTHERMAL, BC_DIRICHLET), per if nz > 1 else (0, 0))
    wt = ((0.0, 0.0), (bl["g0"], 0.0), (0.0, 0.0))
    return Case(name="sbli_slab", n=n, Q0=Q0, dt=dt, nsteps=nsteps, delta=(1.0, 1.0, 1.0), coords=coords, gamma=gamma,
                Re=Re, Pr=Pr, Minf=M, scheme=scheme, visc=VISC_SUTHERLAND, suth_ratio=S, bc=bc, wall_T=wt,
                dirichlet=dirichlet, extra={"bl": bl, "x0": x0, "shock": sh})


# ------------------------------------------------- laminar channel ----
def channel(n=(32, 64, 1), Re=90.0, Pr=0.72, M=0.01, scheme=TENO6, dt=1e-4, nsteps=10, noise=0.0, seed=3):
    """Laminar compressible channel of PAPER.md:535-546: isothermal wall (T = 1) at y = -1, adiabatic wall at
    y = +1, constant viscosity, periodic in x, driven by a unit body force; initial state = the analytic
    steady solution eq. (52)-(53) (plus optional seeded noise so that parity inputs are not a fixed point)."""
    n = tuple(int(v) for v in n)
    gamma = 1.4
    i, j, k = padded_index_grids(n)
    y = -1.0 + 2.0 * j / (n[1] - 1.0) + 0.0 * i + 0.0 * k
    yc = np.clip(y, -1.0, 1.0)
    u = Re * (1.0 - yc ** 2) / 2.0                                                   # eq. (52)
    T = 1.0 - Re ** 2 * M ** 2 * Pr * (gamma - 1.0) * (yc ** 4 - 4.0 * yc - 5.0) / 12.0   # eq. (53)
    p = 1.0 / (gamma * M * M)
    rho = 1.0 / T
    if noise:
        ii, jj, kk = np.meshgrid(np.arange(-halo_of(n)[0], n[0] + halo_of(n)[0]), np.arange(-halo_of(n)[1], n[1] + halo_of(n)[1]),
                                 np.arange(-halo_of(n)[2], n[2] + halo_of(n)[2]), indexing="ij")
        lin = ((ii + 8) + 4096 * ((jj + 8) + 4096 * (kk + 8))).astype(np.uint64)
        rho = rho * (1.0 + noise * splitmix64_unit(seed, lin).transpose(2, 1, 0))
        u = u * (1.0 + noise * splitmix64_unit(seed + 1, lin).transpose(2, 1, 0))
    Q0 = edge_pad_interior(np.ascontiguousarray(conservative(rho, u, 0.0 * u, 0.0 * u, p + 0.0 * u, gamma)), n)
    per = (BC_PERIODIC, BC_PERIODIC)
    bc = (per, (BC_WALL_ISOTHERMAL, BC_WALL_ADIABATIC), per if n[2] > 1 else (0, 0))
    Taw = 1.0 + 8.0 * Re ** 2 * M ** 2 * Pr * (gamma - 1.0) / 12.0
    return Case(name="channel", n=n, Q0=Q0, dt=dt, nsteps=nsteps,
                delta=(2.0 * np.pi / n[0], 2.0 / (n[1] - 1.0), (2.0 * np.pi / n[2]) if n[2] > 1 else 1.0), gamma=gamma,
                Re=Re, Pr=Pr, Minf=M, scheme=scheme, visc=VISC_CONST, bc=bc, wall_T=((0.0, 0.0), (1.0, 0.0), (0.0, 0.0)),
                force=(1.0, 0.0, 0.0), extra={"T_aw": Taw, "u": u, "T": T})


# --------------------------------------------------- small curvilinear box (parity cases) ----
def wavy_box(n=(24, 20, 8), seed=1, bc=None, scheme=WENOZ5, visc=VISC_SUTHERLAND, M=2.0, Re=950.0, Pr=0.72,
             amp=0.05, grid_amp=0.03, wall_T=1.2, dt=1e-3, nsteps=2):
    """Smooth seeded flow on a smooth fully 3-D curvilinear mapping; any mix of boundary types.

    Not one of the paper's cases: a small stand-in with the structure of the SBLI slab (curvilinear
    metrics incl. cross terms, Sutherland viscosity, wall / Dirichlet / extrapolation / periodic
    boundaries) that the oracle finishes in seconds.  Coordinates are analytic in the node index, so
    halo coordinates are the periodic continuation where a direction is periodic.
    """
    n = tuple(int(v) for v in n)
    if bc is None:
        bc = ((BC_DIRICHLET, BC_EXTRAP0), (BC_WALL_ISOTHERMAL, BC_DIRICHLET), (BC_PERIODIC, BC_PERIODIC))
    per = tuple(bc[d][0] == BC_PERIODIC for d in range(3))
    rng = np.random.default_rng(seed)
    i, j, k = padded_index_grids(n, scheme)
    # computational coordinates in [0,1): periodic directions use n points per period, others n-1 intervals
    den = [float(n[d] if per[d] else max(n[d] - 1, 1)) for d in range(3)]
    xi, et, ze = i / den[0] + 0.0 * j + 0.0 * k, j / den[1] + 0.0 * i + 0.0 * k, k / den[2] + 0.0 * i + 0.0 * j
    Lx, Ly, Lz = 2.0, 1.5, 1.0
    tw = 2.0 * np.pi
    active = [v > 1 for v in n]
    bump = np.sin(tw * xi) * (np.sin(tw * et) if active[1] else 1.0) * (np.cos(tw * ze) if active[2] else 1.0)
    x = Lx * (xi + grid_amp * bump)
    y = Ly * (et + grid_amp * np.sin(tw * xi + 0.3) * np.sin(tw * et)) if active[1] else 0.0 * xi
    z = Lz * (ze + grid_amp * np.sin(tw * ze) * np.cos(tw * xi)) if active[2] else 0.0 * xi
    coords = np.ascontiguousarray(np.stack([x, y, z]))
    ph = rng.uniform(0, tw, size=12)
    gamma = 1.4
    p0 = 1.0 / (gamma * M * M)

    def wave(a, b, c, q):
        return np.sin(tw * (a * xi + b * et + c * ze) + q)

    rho = 1.0 + amp * wave(1, 1, 1, ph[0]) + 0.5 * amp * wave(2, 0, 1, ph[1])
    u = 1.0 + amp * wave(1, 2, 0, ph[2])
    v = amp * wave(2, 1, 1, ph[3]) if active[1] else 0.0 * xi
    w = amp * wave(1, 1, 2, ph[4]) if active[2] else 0.0 * xi
    p = p0 * (1.0 + amp * wave(1, 1, 1, ph[5]) + 0.5 * amp * wave(0, 2, 1, ph[6]))
    Q0 = np.ascontiguousarray(conservative(rho, u, v, w, p, gamma))
    dirichlet = Q0.copy()
    wt = tuple(tuple(wall_T if bc[d][s] == BC_WALL_ISOTHERMAL else 0.0 for s in range(2)) for d in range(3))
    return Case(name="wavy_box", n=n, Q0=Q0, dt=dt, nsteps=nsteps, delta=(1.0, 1.0, 1.0), coords=coords, gamma=gamma,
                Re=Re, Pr=Pr, Minf=M, scheme=scheme, visc=visc, bc=bc, wall_T=wt, dirichlet=dirichlet)


def perturb(case, seed=0, amp=0.02):
    """Seeded perturbation of a case's initial state (rho, p stay > 0); returns a new dense Q0.

    Moves parity inputs away from the symmetric analytic fields, where many terms vanish.
    Momentum along an inactive direction stays exactly zero (Q27)."""
    rng = np.random.default_rng(seed)
    Q = case.Q0.copy()
    h = case.halo
    core = (slice(h[2], h[2] + case.n[2]), slice(h[1], h[1] + case.n[1]), slice(h[0], h[0] + case.n[0]))
    for c in range(5):
        if c in (1, 2, 3) and case.n[c - 1] == 1:
            continue
        ref = np.abs(Q[c][core]).max()
        scale = amp * (0.1 * ref if c in (0, 4) else max(ref, 0.1))
        Q[c][core] += scale * rng.uniform(-1.0, 1.0, size=Q[c][core].shape)
    return edge_pad_interior(Q, case.n, case.scheme)


def approximate_metrics(case):
    """Metric fields D = (dx/dxi)^-1, detJ, E = d(D) of a curvilinear case from 2nd-order numpy gradients of its
    analytic coordinates.  INPUT GENERATION for throughput runs and memory checks only (bench.py, tests/
    sanitizer_cases.py), where the values merely have to be smooth, finite and consistent; the parity tests feed
    both sides the metric fields of PAPER.md:228 computed by the oracle's `metrics_from_coords`."""
    X = case.coords
    A = np.zeros((3, 3) + X.shape[1:])
    axes = {0: 2, 1: 1, 2: 0}
    for c in range(3):
        for d in range(3):
            if case.n[d] > 1:
                A[c, d] = np.gradient(X[c], axis=axes[d])
            else:
                A[c, d] = case.delta[d] if c == d else 0.0
    Am = np.moveaxis(A, (0, 1), (-2, -1))
    det = np.linalg.det(Am)
    D = np.moveaxis(np.linalg.inv(Am), (-2, -1), (0, 1))          # D[k][j] = d xi_k / d x_j
    IJ = ((0, 0), (0, 1), (0, 2), (1, 1), (1, 2), (2, 2))
    E = [[None] * 6 for _ in range(3)]
    for l in range(3):
        grads = [[np.gradient(D[l, j], axis=axes[k]) if case.n[k] > 1 else 0.0 * det for k in range(3)] for j in range(3)]
        for m, (i, j) in enumerate(IJ):
            E[l][m] = np.ascontiguousarray(sum(D[k, i] * grads[j][k] for k in range(3)))
    return {"D": [[np.ascontiguousarray(D[k, j]) for j in range(3)] for k in range(3)], "detJ": np.ascontiguousarray(det), "E": E}
