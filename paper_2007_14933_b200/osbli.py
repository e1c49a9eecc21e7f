"""Thin ctypes binding of libosbli (include/osbli.h).  Argument marshalling only: every step of
the path (halo fill, residual, RK3 update) runs in the CUDA kernels behind the C ABI.  PyTorch is
used for device memory and streams.  There is NO fallback: if libosbli.so is missing or fails to
load, importing this module raises.

Functions carry the C names (`osbli_get_layout`, `osbli_workspace_bytes`, `osbli_init`,
`osbli_bc`, `osbli_rhs`, `osbli_rk3_step`, `osbli_advance_host`, `osbli_launch_count`,
`osbli_destroy`, `osbli_strerror`); `Solver` bundles a handle with its torch-owned buffers.

Dense <-> padded conversion (`to_padded`, `from_padded`) is pure data movement between the
exchange format of `workloads.py` ([.., NZ, NY, NX] with halo 3; 4 for the 7th-order scheme) and the library's padded,
128-byte-aligned rows.
"""
from __future__ import annotations

import ctypes as C
from pathlib import Path

import numpy as np

_LIBPATH = Path(__file__).resolve().parent / "libosbli.so"
if not _LIBPATH.exists():
    raise ImportError(f"{_LIBPATH} not built: run `python -m paper_2007_14933_b200.build` "
                      "(there is no CPU fallback for the osbli hot path)")
_lib = C.CDLL(str(_LIBPATH))

OK, EINVAL, EUNSUPPORTED, ECUDA, EWORKSPACE, ESTATIC = 0, 1, 2, 3, 4, 5
SCHEME_WENOZ5, SCHEME_TENO5, SCHEME_TENO6, SCHEME_WENOJS5, SCHEME_CENTRAL4, SCHEME_WENOZ3, SCHEME_WENOZ7 = 0, 1, 2, 3, 4, 5, 6
VISC_NONE, VISC_CONST, VISC_SUTHERLAND = 0, 1, 2
BC_PERIODIC, BC_EXTRAP0, BC_DIRICHLET, BC_WALL_ISOTHERMAL, BC_WALL_ADIABATIC = 0, 1, 2, 3, 4
AVG_ROE, AVG_SIMPLE = 0, 1
RK3_WILLIAMSON, RK3_SSP = 0, 1

_dp = C.c_void_p   # device / host addresses travel as plain integers


class Metrics(C.Structure):
    _fields_ = [("D", (_dp * 3) * 3), ("detJ", _dp), ("E", (_dp * 6) * 3)]


class Params(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32),
        ("dx", C.c_double), ("dy", C.c_double), ("dz", C.c_double),
        ("metrics", C.POINTER(Metrics)),
        ("gamma", C.c_double), ("Re", C.c_double), ("Pr", C.c_double), ("Minf", C.c_double),
        ("scheme", C.c_int32),
        ("teno_ct", C.c_double), ("eps", C.c_double),
        ("visc", C.c_int32),
        ("suth_ratio", C.c_double),
        ("bc", (C.c_int32 * 2) * 3),
        ("wall_T", (C.c_double * 2) * 3),
        ("dirichlet", _dp),
        ("force", C.c_double * 3),
        ("averaging", C.c_int32),
        ("rk3_form", C.c_int32),
    ]


class Layout(C.Structure):
    _fields_ = [("halo", C.c_int32 * 3), ("x_offset", C.c_int64), ("stride_y", C.c_int64),
                ("stride_z", C.c_int64), ("stride_var", C.c_int64), ("total_doubles", C.c_int64)]


_h = C.c_void_p
_lib.osbli_get_layout.restype = C.c_int
_lib.osbli_get_layout.argtypes = [C.POINTER(Params), C.POINTER(Layout)]
_lib.osbli_workspace_bytes.restype = C.c_int
_lib.osbli_workspace_bytes.argtypes = [C.POINTER(Params), C.POINTER(C.c_size_t)]
_lib.osbli_init.restype = C.c_int
_lib.osbli_init.argtypes = [C.POINTER(Params), _dp, C.c_size_t, C.POINTER(_h)]
_lib.osbli_bc.restype = C.c_int
_lib.osbli_bc.argtypes = [_h, _dp, _dp]
_lib.osbli_rhs.restype = C.c_int
_lib.osbli_rhs.argtypes = [_h, _dp, _dp, _dp]
_lib.osbli_rk3_step.restype = C.c_int
_lib.osbli_rk3_step.argtypes = [_h, _dp, _dp, C.c_double, _dp]
_lib.osbli_static_scratch_bytes.restype = C.c_size_t
_lib.osbli_static_scratch_bytes.argtypes = []
_lib.osbli_rk3_step_static.restype = C.c_int
_lib.osbli_rk3_step_static.argtypes = [C.POINTER(Params), _dp, _dp, C.c_double, _dp]
_lib.osbli_rk4_step.restype = C.c_int
_lib.osbli_rk4_step.argtypes = [_h, _dp, _dp, C.c_double, _dp]
_lib.osbli_advance_host.restype = C.c_int
_lib.osbli_advance_host.argtypes = [_h, _dp, _dp, _dp, C.c_double, C.c_int32, _dp]
_lib.osbli_advance_host_batch.restype = C.c_int
_lib.osbli_advance_host_batch.argtypes = [_h, C.POINTER(_dp), C.c_int32, C.POINTER(_dp), _dp, C.c_double, C.c_int32, _dp]
_lib.osbli_launch_count.restype = C.c_int
_lib.osbli_launch_count.argtypes = [_h, C.POINTER(C.c_int64)]
_lib.osbli_profile_begin.restype = C.c_int
_lib.osbli_profile_begin.argtypes = [_h]
_lib.osbli_profile_end.restype = C.c_int
_lib.osbli_profile_end.argtypes = [_h, _dp, C.POINTER(C.c_double), C.POINTER(C.c_int64)]
_lib.osbli_measure_fp64_peak.restype = C.c_int
_lib.osbli_measure_fp64_peak.argtypes = [_dp, _dp, C.POINTER(C.c_double)]
_lib.osbli_destroy.restype = C.c_int
_lib.osbli_destroy.argtypes = [_h]
_lib.osbli_strerror.restype = C.c_char_p
_lib.osbli_strerror.argtypes = [C.c_int]

EXPORTS = ("osbli_get_layout", "osbli_workspace_bytes", "osbli_init", "osbli_bc", "osbli_rhs",
           "osbli_rk3_step", "osbli_rk3_step_static", "osbli_static_scratch_bytes", "osbli_rk4_step", "osbli_advance_host", "osbli_advance_host_batch", "osbli_launch_count", "osbli_profile_begin", "osbli_profile_end",
           "osbli_measure_fp64_peak", "osbli_destroy", "osbli_strerror")
K_CLASSES = ("bc", "primitives", "sweep_x", "sweep_y", "sweep_z", "viscous", "rk_update")


class OsbliError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__(f"{where}: {osbli_strerror(status)} (status {status})")


def _check(status, where):
    if status != OK:
        raise OsbliError(status, where)


# ---- the C entry points, same names ------------------------------------------------------------
def osbli_strerror(status: int) -> str:
    return _lib.osbli_strerror(int(status)).decode()


def osbli_get_layout(params: Params) -> Layout:
    out = Layout()
    _check(_lib.osbli_get_layout(C.byref(params), C.byref(out)), "osbli_get_layout")
    return out


def osbli_workspace_bytes(params: Params) -> int:
    out = C.c_size_t(0)
    _check(_lib.osbli_workspace_bytes(C.byref(params), C.byref(out)), "osbli_workspace_bytes")
    return int(out.value)


def osbli_init(params: Params, workspace_ptr: int, workspace_bytes: int) -> int:
    h = _h()
    _check(_lib.osbli_init(C.byref(params), workspace_ptr, workspace_bytes, C.byref(h)), "osbli_init")
    return h.value


def osbli_bc(handle, q_ptr, stream=0):
    _check(_lib.osbli_bc(handle, q_ptr, stream), "osbli_bc")


def osbli_rhs(handle, q_ptr, r_ptr, stream=0):
    _check(_lib.osbli_rhs(handle, q_ptr, r_ptr, stream), "osbli_rhs")


def osbli_rk3_step(handle, q_ptr, qtmp_ptr, dt, stream=0):
    _check(_lib.osbli_rk3_step(handle, q_ptr, qtmp_ptr, float(dt), stream), "osbli_rk3_step")


def osbli_static_scratch_bytes() -> int:
    return int(_lib.osbli_static_scratch_bytes())


def osbli_rk3_step_static(params: Params, q_ptr, qtmp_ptr, dt, stream=0):
    """One RK3 step with the workspace in the library's static device array: no handle, no allocation (osbli.h)."""
    _check(_lib.osbli_rk3_step_static(C.byref(params), q_ptr, qtmp_ptr, float(dt), stream), "osbli_rk3_step_static")


def osbli_rk4_step(handle, q_ptr, qtmp_ptr, dt, stream=0):
    _check(_lib.osbli_rk4_step(handle, q_ptr, qtmp_ptr, float(dt), stream), "osbli_rk4_step")


def osbli_advance_host(handle, hq_ptr, q_ptr, qtmp_ptr, dt, nsteps, stream=0):
    _check(_lib.osbli_advance_host(handle, hq_ptr, q_ptr, qtmp_ptr, float(dt), int(nsteps), stream),
           "osbli_advance_host")


def osbli_advance_host_batch(handle, hq_ptrs, q_ptrs, qtmp_ptr, dt, nsteps, stream=0):
    assert len(q_ptrs) == 3
    hq = (_dp * len(hq_ptrs))(*hq_ptrs)
    dq = (_dp * 3)(*q_ptrs)
    _check(_lib.osbli_advance_host_batch(handle, hq, len(hq_ptrs), dq, qtmp_ptr, float(dt), int(nsteps), stream),
           "osbli_advance_host_batch")


def osbli_launch_count(handle) -> int:
    out = C.c_int64(0)
    _check(_lib.osbli_launch_count(handle, C.byref(out)), "osbli_launch_count")
    return int(out.value)


def osbli_profile_begin(handle):
    _check(_lib.osbli_profile_begin(handle), "osbli_profile_begin")


def osbli_profile_end(handle, stream=0):
    ms = (C.c_double * len(K_CLASSES))()
    cnt = (C.c_int64 * len(K_CLASSES))()
    _check(_lib.osbli_profile_end(handle, stream, ms, cnt), "osbli_profile_end")
    return {k: (float(ms[i]), int(cnt[i])) for i, k in enumerate(K_CLASSES)}


def osbli_measure_fp64_peak(scratch_ptr, stream=0) -> float:
    out = C.c_double(0.0)
    _check(_lib.osbli_measure_fp64_peak(scratch_ptr, stream, C.byref(out)), "osbli_measure_fp64_peak")
    return float(out.value)


def osbli_destroy(handle):
    _check(_lib.osbli_destroy(handle), "osbli_destroy")


# ---- marshalling helpers ------------------------------------------------------------------------
def make_params(*, n, delta=(1.0, 1.0, 1.0), gamma=1.4, Re=1.0, Pr=1.0, Minf=1.0, scheme=SCHEME_WENOZ5,
                teno_ct=1e-6, eps=1e-16, visc=VISC_NONE, suth_ratio=110.4 / 288.0,
                bc=((0, 0), (0, 0), (0, 0)), wall_T=((0.0, 0.0), (0.0, 0.0), (0.0, 0.0)), force=(0.0, 0.0, 0.0),
                averaging=AVG_ROE, rk3_form=RK3_WILLIAMSON) -> Params:
    p = Params()
    p.nx, p.ny, p.nz = (int(v) for v in n)
    p.dx, p.dy, p.dz = (float(v) for v in delta)
    p.gamma, p.Re, p.Pr, p.Minf = float(gamma), float(Re), float(Pr), float(Minf)
    p.scheme, p.visc = int(scheme), int(visc)
    p.teno_ct, p.eps, p.suth_ratio = float(teno_ct), float(eps), float(suth_ratio)
    for d in range(3):
        for s in range(2):
            p.bc[d][s] = int(bc[d][s])
            p.wall_T[d][s] = float(wall_T[d][s])
    p.force[:] = [float(v) for v in force]
    p.averaging, p.rk3_form = int(averaging), int(rk3_form)
    return p


def dense_view(padded, lay: Layout, n):
    """View of a padded array [.., NZ, NY, stride_y] restricted to the dense exchange columns."""
    hx = lay.halo[0]
    return padded[..., lay.x_offset - hx: lay.x_offset + n[0] + hx]


class Solver:
    """A handle plus the torch-owned device buffers it borrows (workspace, metrics, Dirichlet state)."""

    def __init__(self, *, metrics=None, dirichlet=None, device="cuda:0", **physics):
        import torch
        self.torch = torch
        self.device = torch.device(device)
        self.params = make_params(**physics)
        self.n = (self.params.nx, self.params.ny, self.params.nz)
        self.layout = osbli_get_layout(self.params)
        lay = self.layout
        self.N = tuple(self.n[d] + 2 * lay.halo[d] for d in range(3))
        self.field_shape = (self.N[2], self.N[1], int(lay.stride_y))
        self.state_shape = (5,) + self.field_shape
        assert int(np.prod(self.state_shape)) == lay.total_doubles
        self._keep = []
        if dirichlet is not None:
            d = self.to_padded(dirichlet)
            self._keep.append(d)
            self.params.dirichlet = d.data_ptr()
        if metrics is not None:
            m = Metrics()
            for k in range(3):
                for j in range(3):
                    t = self.to_padded(metrics["D"][k][j]); self._keep.append(t); m.D[k][j] = t.data_ptr()
                for e in range(6):
                    t = self.to_padded(metrics["E"][k][e]); self._keep.append(t); m.E[k][e] = t.data_ptr()
            t = self.to_padded(metrics["detJ"]); self._keep.append(t); m.detJ = t.data_ptr()
            self._metrics = m
            self.params.metrics = C.pointer(m)
        nbytes = osbli_workspace_bytes(self.params)
        self.workspace = torch.empty(nbytes // 8, dtype=torch.float64, device=self.device)
        with torch.cuda.device(self.device):
            self.handle = osbli_init(self.params, self.workspace.data_ptr(), nbytes)

    # -- buffers --------------------------------------------------------------------------------
    def empty_state(self, fill=None):
        t = self.torch
        if fill is None:
            return t.empty(self.state_shape, dtype=t.float64, device=self.device)
        return t.full(self.state_shape, float(fill), dtype=t.float64, device=self.device)

    def to_padded(self, dense, pinned_host=False):
        """dense numpy [.., NZ, NY, NX] -> padded tensor [.., NZ, NY, stride_y] (pad entries = 1)."""
        t = self.torch
        dense = np.ascontiguousarray(dense, dtype=np.float64)
        assert dense.shape[-3:] == (self.N[2], self.N[1], self.N[0]), (dense.shape, self.N)
        shape = dense.shape[:-3] + self.field_shape
        host = t.ones(shape, dtype=t.float64, pin_memory=pinned_host)
        dense_view(host, self.layout, self.n).copy_(t.from_numpy(dense))
        return host if pinned_host else host.to(self.device)

    def from_padded(self, padded):
        """padded tensor -> dense numpy [.., NZ, NY, NX]."""
        return dense_view(padded, self.layout, self.n).cpu().numpy().copy()

    # -- the path -------------------------------------------------------------------------------
    def _stream(self):
        return self.torch.cuda.current_stream(self.device).cuda_stream

    def _on_device(self):
        """The handle's device made current for the duration of a call (launches go to the current device)."""
        return self.torch.cuda.device(self.device)

    def bc(self, Q):
        with self._on_device():
            osbli_bc(self.handle, Q.data_ptr(), self._stream())
        return Q

    def rhs(self, Q, R=None):
        if R is None:
            R = self.empty_state(0.0)
        with self._on_device():
            osbli_rhs(self.handle, Q.data_ptr(), R.data_ptr(), self._stream())
        return R

    def rk3_step(self, Q, Qtmp, dt):
        with self._on_device():
            osbli_rk3_step(self.handle, Q.data_ptr(), Qtmp.data_ptr(), dt, self._stream())
        return Q

    def rk4_step(self, Q, Qtmp, dt):
        with self._on_device():
            osbli_rk4_step(self.handle, Q.data_ptr(), Qtmp.data_ptr(), dt, self._stream())
        return Q

    def advance_host(self, hQ, Q, Qtmp, dt, nsteps):
        with self._on_device():
            osbli_advance_host(self.handle, hQ.data_ptr(), Q.data_ptr(), Qtmp.data_ptr(), dt, nsteps, self._stream())
        return hQ

    def advance_host_batch(self, hQs, Qs, Qtmp, dt, nsteps):
        with self._on_device():
            osbli_advance_host_batch(self.handle, [t.data_ptr() for t in hQs], [t.data_ptr() for t in Qs], Qtmp.data_ptr(),
                                     dt, nsteps, self._stream())
        return hQs

    def profile_begin(self):
        osbli_profile_begin(self.handle)

    def profile_end(self):
        return osbli_profile_end(self.handle, self._stream())

    def measure_fp64_peak(self):
        return osbli_measure_fp64_peak(self.workspace.data_ptr(), self._stream())

    def launch_count(self):
        return osbli_launch_count(self.handle)

    def close(self):
        if getattr(self, "handle", None):
            osbli_destroy(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
