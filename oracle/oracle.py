"""ctypes front end of the CPU oracle (oracle/osbli_oracle.cpp).

TEST INFRASTRUCTURE, NOT PRODUCT CODE.  Only tests/, __graft_entry__.smoke() and bench.py's
cpu_baseline / --impl reference legs may import this module.  It imports nothing from the CUDA
package; it takes plain numpy arrays in the oracle's own dense layout
([5][NZ][NY][NX], halo 3 in every active direction, 4 for the 7th-order scheme, see osbli_oracle.h).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from pathlib import Path

import numpy as np

_HERE = Path(__file__).resolve().parent
_SRC = _HERE / "osbli_oracle.cpp"
_HDR = _HERE / "osbli_oracle.h"
_LIB = _HERE / "libosbli_oracle.so"

WENOZ5, TENO5, TENO6, WENOJS5, CENTRAL4, WENOZ3, WENOZ7 = 0, 1, 2, 3, 4, 5, 6
VISC_NONE, VISC_CONST, VISC_SUTHERLAND = 0, 1, 2
BC_PERIODIC, BC_EXTRAP0, BC_DIRICHLET, BC_WALL_ISOTHERMAL = 0, 1, 2, 3
PART_INVISCID, PART_VISCOUS = 1, 2
AVG_ROE, AVG_SIMPLE = 0, 1
RK3_WILLIAMSON, RK3_SSP = 0, 1

_dp = C.POINTER(C.c_double)


class _Params(C.Structure):
    _fields_ = [
        ("n", C.c_int32 * 3),
        ("delta", C.c_double * 3),
        ("curvilinear", C.c_int32),
        ("D", (_dp * 3) * 3),
        ("detJ", _dp),
        ("E", (_dp * 6) * 3),
        ("gamma", C.c_double), ("Re", C.c_double), ("Pr", C.c_double), ("Minf", C.c_double),
        ("scheme", C.c_int32),
        ("teno_ct", C.c_double), ("eps", C.c_double),
        ("visc", C.c_int32),
        ("suth_ratio", C.c_double),
        ("bc", (C.c_int32 * 2) * 3),
        ("wall_T", (C.c_double * 2) * 3),
        ("dirichlet", _dp),
        ("nthreads", C.c_int32),
        ("force", C.c_double * 3),
        ("averaging", C.c_int32),
        ("rk3_form", C.c_int32),
    ]


def build(force: bool = False) -> Path:
    """Compile the oracle: g++ -O2 -ffp-contract=off (no FMA contraction), OpenMP outer loops."""
    newest = max(_SRC.stat().st_mtime, _HDR.stat().st_mtime)
    if force or not _LIB.exists() or _LIB.stat().st_mtime < newest:
        tmp = _LIB.with_suffix(f".tmp{os.getpid()}.so")
        cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC",
               "-Wall", "-Wextra", "-o", str(tmp), str(_SRC)]
        subprocess.run(cmd, check=True)
        os.replace(tmp, _LIB)
    return _LIB


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(str(_LIB))
        L.oracle_reconstruct.restype = C.c_double
        L.oracle_reconstruct.argtypes = [C.c_int32] + [C.c_double] * 7 + [_dp]
        L.oracle_reconstruct6.restype = C.c_double
        L.oracle_reconstruct6.argtypes = [C.c_double] * 8 + [_dp]
        L.oracle_reconstruct7.restype = C.c_double
        L.oracle_reconstruct7.argtypes = [_dp, C.c_double, _dp]
        L.oracle_teno6_indicators.restype = None
        L.oracle_teno6_indicators.argtypes = [C.c_double] * 6 + [_dp]
        L.oracle_eigensystem.restype = None
        L.oracle_eigensystem.argtypes = [C.c_double, _dp, _dp, _dp, _dp, _dp, _dp]
        L.oracle_eigensystem_avg.restype = None
        L.oracle_eigensystem_avg.argtypes = [C.c_double, C.c_int32, _dp, _dp, _dp, _dp, _dp, _dp]
        L.oracle_rk3ssp_update.restype = None
        L.oracle_rk3ssp_update.argtypes = [C.c_int32, C.c_double, C.c_int64, _dp, _dp, _dp]
        L.oracle_d1.restype = C.c_double
        L.oracle_d1.argtypes = [_dp, C.c_int32, C.c_int32, C.c_int32, C.c_double]
        L.oracle_d2.restype = C.c_double
        L.oracle_d2.argtypes = [_dp, C.c_int32, C.c_int32, C.c_int32, C.c_double]
        L.oracle_field_size.restype = C.c_int64
        L.oracle_field_size.argtypes = [C.POINTER(_Params)]
        L.oracle_halo.restype = C.c_int32
        L.oracle_halo.argtypes = [C.POINTER(_Params), C.POINTER(C.c_int32)]
        L.oracle_interface_flux.restype = None
        L.oracle_interface_flux.argtypes = [C.POINTER(_Params), _dp, C.c_int32, C.c_int32, C.c_int32, C.c_int32, _dp, _dp]
        L.oracle_bc.restype = C.c_int32
        L.oracle_bc.argtypes = [C.POINTER(_Params), _dp]
        L.oracle_rhs.restype = C.c_int32
        L.oracle_rhs.argtypes = [C.POINTER(_Params), _dp, _dp, C.c_int32, _dp]
        L.oracle_rhs_points.restype = C.c_int32
        L.oracle_rhs_points.argtypes = [C.POINTER(_Params), _dp, C.c_int32, C.c_int64, C.POINTER(C.c_int32), _dp]
        L.oracle_metrics.restype = C.c_int32
        L.oracle_metrics.argtypes = [C.POINTER(_Params), _dp, C.POINTER(_dp), _dp, C.POINTER(_dp)]
        L.oracle_rk3_step.restype = C.c_int32
        L.oracle_rk3_step.argtypes = [C.POINTER(_Params), _dp, _dp, _dp, C.c_double]
        L.oracle_rk3_update.restype = None
        L.oracle_rk3_update.argtypes = [C.c_int32, C.c_double, C.c_int64, _dp, _dp, _dp]
        L.oracle_rk4_step.restype = C.c_int32
        L.oracle_rk4_step.argtypes = [C.POINTER(_Params), _dp, _dp, _dp, C.c_double]
        L.oracle_rk4_update.restype = None
        L.oracle_rk4_update.argtypes = [C.c_int32, C.c_double, C.c_int64, _dp, _dp, _dp]
        _lib = L
    return _lib


def _ptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(_dp)


def reconstruct(scheme, a, b, c, d, e, eps=1e-16, ct=1e-6, with_margin=False):
    m = C.c_double(0.0)
    v = lib().oracle_reconstruct(scheme, a, b, c, d, e, eps, ct, C.byref(m))
    return (v, m.value) if with_margin else v


def reconstruct6(a, b, c, d, e, f, eps=1e-16, ct=1e-6, with_margin=False):
    m = C.c_double(0.0)
    v = lib().oracle_reconstruct6(a, b, c, d, e, f, eps, ct, C.byref(m))
    return (v, m.value) if with_margin else v


def reconstruct7(v7, eps=1e-16, with_indicators=False):
    """WENO-7Z value at i+1/2 from the seven nodes i-3..i+3; optionally (beta_0..beta_3, tau_7)."""
    v = np.ascontiguousarray(v7, dtype=np.float64)
    assert v.shape == (7,)
    out = np.zeros(5)
    val = lib().oracle_reconstruct7(_ptr(v), eps, _ptr(out))
    return (val, out) if with_indicators else val


def teno6_indicators(a, b, c, d, e, f):
    out = np.zeros(5)
    lib().oracle_teno6_indicators(a, b, c, d, e, f, _ptr(out))
    return out


def eigensystem(gamma, QL, QR, nhat, averaging=AVG_ROE):
    QL = np.ascontiguousarray(QL, dtype=np.float64)
    QR = np.ascontiguousarray(QR, dtype=np.float64)
    nhat = np.ascontiguousarray(nhat, dtype=np.float64)
    L = np.zeros((5, 5)); R = np.zeros((5, 5)); roe = np.zeros(5)
    lib().oracle_eigensystem_avg(gamma, int(averaging), _ptr(QL), _ptr(QR), _ptr(nhat), _ptr(L), _ptr(R), _ptr(roe))
    return L, R, roe


def d1(f, i, periodic, delta, pad=0):
    """f: 1-D array; if periodic, `pad` leading/trailing halo entries surround the n nodes."""
    f = np.ascontiguousarray(f, dtype=np.float64)
    n = f.size - 2 * pad
    base = C.cast(C.addressof(_ptr(f).contents) + 8 * pad, _dp)
    return lib().oracle_d1(base, n, i, int(periodic), delta)


def d2(f, i, periodic, delta, pad=0):
    f = np.ascontiguousarray(f, dtype=np.float64)
    n = f.size - 2 * pad
    base = C.cast(C.addressof(_ptr(f).contents) + 8 * pad, _dp)
    return lib().oracle_d2(base, n, i, int(periodic), delta)


def rk4_update(s, dt, U, dU, R):
    """One sub-stage (s = 0..4) of the five-stage 4th-order scheme on flat arrays, in place."""
    lib().oracle_rk4_update(int(s), float(dt), U.size, _ptr(U), _ptr(dU), _ptr(R))


def rk3ssp_update(s, dt, U, dU, R):
    """One sub-stage (s = 0..2) of the SSP 3rd-order scheme on flat arrays, in place."""
    lib().oracle_rk3ssp_update(int(s), float(dt), U.size, _ptr(U), _ptr(dU), _ptr(R))


def rk3_update(s, dt, U, dU, R):
    """One RK3 stage update (eq. 36-37) on flat float64 arrays, in place."""
    lib().oracle_rk3_update(int(s), float(dt), U.size, _ptr(U), _ptr(dU), _ptr(R))


def metrics_from_coords(coords, n, periodic, delta=(1.0, 1.0, 1.0), nthreads=None, scheme=WENOZ5):
    """PAPER.md:228 metric terms from node coordinates.

    coords: [3, NZ, NY, NX] (x, y, z on the halo-extended grid, periodic continuation in the
    halos of periodic directions).  Returns {"D": 3x3 list, "detJ": field, "E": 3x6 list} of
    halo-filled fields in oracle layout.  `scheme` only selects the halo depth (4 for WENO-7Z).
    """
    coords = np.ascontiguousarray(coords, dtype=np.float64)
    hd = 4 if int(scheme) == WENOZ7 else 3
    want = tuple(int(v) + (2 * hd if int(v) > 1 else 0) for v in reversed(tuple(n)))
    assert coords.shape == (3,) + want, (coords.shape, want, "coords must carry the halo depth of `scheme`")
    p = _Params()
    p.scheme = int(scheme)
    p.n[:] = [int(v) for v in n]
    p.delta[:] = [float(v) for v in delta]
    for d in range(3):
        for s in range(2):
            p.bc[d][s] = BC_PERIODIC if periodic[d] else BC_EXTRAP0
    p.nthreads = int(nthreads or os.cpu_count() or 1)
    fshape = coords.shape[1:]
    D = [np.zeros(fshape) for _ in range(9)]
    E = [np.zeros(fshape) for _ in range(18)]
    detJ = np.zeros(fshape)
    Dp = (_dp * 9)(*[_ptr(a) for a in D])
    Ep = (_dp * 18)(*[_ptr(a) for a in E])
    rc = lib().oracle_metrics(C.byref(p), _ptr(coords), Dp, _ptr(detJ), Ep)
    assert rc == 0
    return {"D": [[D[k * 3 + j] for j in range(3)] for k in range(3)], "detJ": detJ,
            "E": [[E[l * 6 + m] for m in range(6)] for l in range(3)]}


class Oracle:
    """One configured problem.  All state arrays are numpy float64 [5, NZ, NY, NX]."""

    def __init__(self, *, n, delta=(1.0, 1.0, 1.0), metrics=None, gamma=1.4, Re=1.0, Pr=1.0, Minf=1.0,
                 scheme=WENOZ5, teno_ct=1e-6, eps=1e-16, visc=VISC_NONE, suth_ratio=110.4 / 288.0,
                 bc=((0, 0), (0, 0), (0, 0)), wall_T=((0, 0), (0, 0), (0, 0)), dirichlet=None,
                 nthreads=None, force=(0.0, 0.0, 0.0), averaging=AVG_ROE, rk3_form=RK3_WILLIAMSON):
        self.n = tuple(int(v) for v in n)
        self.h = tuple((4 if int(scheme) == WENOZ7 else 3) if v > 1 else 0 for v in self.n)      # = oracle_halo()
        self.N = tuple(v + 2 * h for v, h in zip(self.n, self.h))
        self.shape = (5, self.N[2], self.N[1], self.N[0])
        self.fshape = self.shape[1:]
        if nthreads is None:
            # OpenMP regions cost more than they save on small grids
            npts = self.n[0] * self.n[1] * self.n[2]
            nthreads = max(1, min(os.cpu_count() or 1, npts // 2048))
        self.nthreads = int(nthreads)
        p = _Params()
        p.n[:] = self.n
        p.delta[:] = [float(v) for v in delta]
        self._keep = []
        if metrics is not None:
            p.curvilinear = 1
            for k in range(3):
                for j in range(3):
                    p.D[k][j] = self._field(metrics["D"][k][j])
                for m in range(6):
                    p.E[k][m] = self._field(metrics["E"][k][m])
            p.detJ = self._field(metrics["detJ"])
        else:
            p.curvilinear = 0
        p.gamma, p.Re, p.Pr, p.Minf = float(gamma), float(Re), float(Pr), float(Minf)
        p.scheme = int(scheme)
        p.teno_ct, p.eps = float(teno_ct), float(eps)
        p.visc = int(visc)
        p.suth_ratio = float(suth_ratio)
        for d in range(3):
            for s in range(2):
                p.bc[d][s] = int(bc[d][s])
                p.wall_T[d][s] = float(wall_T[d][s])
        if dirichlet is not None:
            a = np.ascontiguousarray(dirichlet, dtype=np.float64)
            assert a.shape == self.shape
            self._keep.append(a)
            p.dirichlet = _ptr(a)
        p.nthreads = self.nthreads
        p.force[:] = [float(v) for v in force]
        p.averaging = int(averaging)
        p.rk3_form = int(rk3_form)
        self.p = p

    def _field(self, a):
        a = np.ascontiguousarray(a, dtype=np.float64)
        assert a.shape == self.fshape, (a.shape, self.fshape)
        self._keep.append(a)
        return _ptr(a)

    # -- layout helpers -------------------------------------------------------------------
    def interior(self, A):
        """View of the interior nodes of a padded field/state (last three axes)."""
        hz, hy, hx = self.h[2], self.h[1], self.h[0]
        return A[..., hz:hz + self.n[2], hy:hy + self.n[1], hx:hx + self.n[0]]

    def pad(self, Aint):
        """Embed interior values [.., nz, ny, nx] into a padded array (halos = edge copy)."""
        Aint = np.asarray(Aint, dtype=np.float64)
        pw = [(0, 0)] * (Aint.ndim - 3) + [(self.h[2],) * 2, (self.h[1],) * 2, (self.h[0],) * 2]
        return np.ascontiguousarray(np.pad(Aint, pw, mode="edge"))

    # -- the path -------------------------------------------------------------------------
    def bc(self, Q):
        assert Q.shape == self.shape
        rc = lib().oracle_bc(C.byref(self.p), _ptr(Q))
        assert rc == 0
        return Q

    def rhs(self, Q, parts=PART_INVISCID | PART_VISCOUS, margin=False):
        assert Q.shape == self.shape
        R = np.zeros(self.shape)
        mg = np.full(self.fshape, np.inf) if margin else None
        rc = lib().oracle_rhs(C.byref(self.p), _ptr(Q), _ptr(R), parts, _ptr(mg) if margin else None)
        assert rc == 0
        return (R, mg) if margin else R

    def rhs_points(self, Q, ijk, parts=PART_INVISCID | PART_VISCOUS):
        ijk = np.ascontiguousarray(ijk, dtype=np.int32)
        assert ijk.ndim == 2 and ijk.shape[1] == 3
        out = np.zeros((ijk.shape[0], 5))
        rc = lib().oracle_rhs_points(C.byref(self.p), _ptr(Q), parts, ijk.shape[0],
                                     ijk.ctypes.data_as(C.POINTER(C.c_int32)), _ptr(out))
        assert rc == 0
        return out

    def interface_flux(self, Q, direction, i, j, k, with_margin=False):
        f = np.zeros(5)
        m = C.c_double(0.0)
        lib().oracle_interface_flux(C.byref(self.p), _ptr(Q), direction, i, j, k, _ptr(f), C.byref(m))
        return (f, m.value) if with_margin else f

    def rk3_step(self, Q, dU, R, dt):
        rc = lib().oracle_rk3_step(C.byref(self.p), _ptr(Q), _ptr(dU), _ptr(R), float(dt))
        assert rc == 0
        return Q

    def rk4_step(self, Q, dU, R, dt):
        rc = lib().oracle_rk4_step(C.byref(self.p), _ptr(Q), _ptr(dU), _ptr(R), float(dt))
        assert rc == 0
        return Q

    def run(self, Q, dt, nsteps, rk4=False):
        """Advance Q in place by nsteps RK3 (or five-stage RK4) steps."""
        dU = np.zeros(self.shape)
        R = np.zeros(self.shape)
        for _ in range(nsteps):
            (self.rk4_step if rk4 else self.rk3_step)(Q, dU, R, dt)
        return Q
