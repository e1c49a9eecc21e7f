"""Memory-safety checks of the CUDA path that need no external tool (compute-sanitizer is closed on this GPU
pool, see profiles/r2_sanitizer.md), for the kernels the review singled out: per-thread cp.async slots, mbarrier
/ TMA plane ring, warp-private transposed tiles, and the fused sweep + update that writes other blocks' halos.

* guard bands: every state the library writes (Q, Qtmp, R, workspace) is carved out of a larger buffer whose
  surrounding bands hold a sentinel bit pattern; after residuals and steps the bands must be bit-identical
  (an out-of-bounds store of any kernel lands there or in a neighbouring state);
* row padding: entries of a written state that are neither interior nor halo are never written;
* uninitialised reads: workspace, Qtmp and the halos of Q start as NaN; the results must be finite (dU^(0) is
  never read, halos are always filled before they are read, the TMA zero-fill region is never consumed);
* races: the same step sequence twice gives bit-identical states (a race between blocks or between the
  asynchronous copies and their consumers shows up as run-to-run differences).
"""
import numpy as np
import pytest

import parity
from paper_2007_14933_b200 import osbli
from paper_2007_14933_b200 import workloads as W

pytestmark = pytest.mark.gpu

SENTINEL = -1.2345678901234567e+300
GUARD = 1 << 16           # doubles on either side of every carved buffer (512 KB)


NAMES = ("tgv32_teno5", "pbox_5x7x6", "pbox_70x37x35_teno6", "pbox2d_40x33", "pbox_mixed_bc", "sod", "tgv16_central4",
         "wavy_box", "channel3d", "tgv16_ssp_simple", "pbox_37x21x13_wenoz7", "wavy_box_wenoz7", "sod_wenoz7")


def _case(name):
    from test_gpu_parity import _periodic_box
    per, ex = (W.BC_PERIODIC, W.BC_PERIODIC), (W.BC_EXTRAP0, W.BC_EXTRAP0)
    if name == "tgv16_ssp_simple":
        ssp = W.tgv(16)
        ssp.rk3_form, ssp.averaging = W.RK3_SSP, W.AVG_SIMPLE
        return ssp, 2
    return {"tgv32_teno5": lambda: (W.tgv(32), 2),
            "pbox_5x7x6": lambda: (_periodic_box((5, 7, 6), dt=5e-4), 2),
            "pbox_70x37x35_teno6": lambda: (_periodic_box((70, 37, 35), scheme=W.TENO6), 1),
            "pbox2d_40x33": lambda: (_periodic_box((40, 33, 1)), 2),
            "pbox_mixed_bc": lambda: (_periodic_box((36, 20, 10), bc=(per, ex, per), dt=1e-3), 2),
            "sod": lambda: (W.sod(), 20),
            "tgv16_central4": lambda: (W.tgv(16, scheme=W.CENTRAL4), 2),
            "wavy_box": lambda: (W.wavy_box(n=(40, 21, 9)), 2),
            "pbox_37x21x13_wenoz7": lambda: (_periodic_box((37, 21, 13), scheme=W.WENOZ7), 2),    # halo 4, tiled sweeps, ragged tiles
            "wavy_box_wenoz7": lambda: (W.wavy_box(n=(40, 21, 9), scheme=W.WENOZ7), 2),
            "sod_wenoz7": lambda: (W.sod(scheme=W.WENOZ7), 20),
            "channel3d": lambda: (W.channel(n=(24, 33, 6), noise=1e-3, scheme=W.TENO5), 2)}[name]()


class Carved:
    """States carved out of one big sentinel-filled buffer, with guard bands between them."""

    def __init__(self, torch, sol, nstates, device):
        self.torch, self.sol = torch, sol
        self.size = int(sol.layout.total_doubles)
        self.ws = (osbli.osbli_workspace_bytes(sol.params) + 7) // 8
        # 256-byte alignment of every carved piece
        rnd = lambda v: (v + 31) // 32 * 32
        self.offs, o = [], rnd(GUARD)
        for _ in range(nstates):
            self.offs.append(o)
            o = rnd(o + self.size + GUARD)
        self.ws_off = o
        o = rnd(o + self.ws + GUARD)
        self.buf = torch.full((o,), SENTINEL, dtype=torch.float64, device=device)
        self.mask = torch.ones(o, dtype=torch.bool, device=device)          # True = guard
        for off in self.offs:
            self.mask[off:off + self.size] = False
        self.mask[self.ws_off:self.ws_off + self.ws] = False

    def state(self, i):
        return self.buf[self.offs[i]:self.offs[i] + self.size].view(self.sol.state_shape)

    def workspace(self):
        return self.buf[self.ws_off:self.ws_off + self.ws]

    def guards_intact(self):
        g = self.buf[self.mask]
        return bool((g.view(self.torch.int64) == self.torch.tensor(SENTINEL, dtype=self.torch.float64).view(self.torch.int64).item()).all())


def _run(case, nsteps, seed_nan=True):
    import torch
    metrics = parity.metrics_for(case)
    sol = parity.make_solver(case, metrics)
    car = Carved(torch, sol, 3, sol.device)
    # re-initialise the handle on the carved workspace (NaN-filled: nothing may be read before it is written)
    osbli.osbli_destroy(sol.handle)
    ws = car.workspace()
    ws.fill_(float("nan"))
    assert ws.data_ptr() % 256 == 0
    sol.workspace = ws
    sol.handle = osbli.osbli_init(sol.params, ws.data_ptr(), ws.numel() * 8)
    Q, Qtmp, R = car.state(0), car.state(1), car.state(2)
    Q.copy_(sol.to_padded(case.Q0))
    lay, h, n = sol.layout, case.halo, case.n
    inner = torch.zeros(sol.state_shape, dtype=torch.bool, device=sol.device)      # interior nodes
    inner[:, h[2]:h[2] + n[2], h[1]:h[1] + n[1], lay.x_offset:lay.x_offset + n[0]] = True
    halo_or_inner = torch.zeros_like(inner)
    halo_or_inner[:, :, :, lay.x_offset - h[0]:lay.x_offset + n[0] + h[0]] = True
    if seed_nan:
        Q[~inner] = float("nan")                       # halos and padding: must be filled before they are read
    Qtmp.fill_(float("nan"))                           # dU^(0) is never read (A_1 = 0)
    R.fill_(SENTINEL)
    pad_before = Q[~halo_or_inner].clone()
    sol.bc(Q)
    sol.rhs(Q, R)
    for _ in range(nsteps):
        sol.rk3_step(Q, Qtmp, case.dt)
    torch.cuda.synchronize()
    assert car.guards_intact(), f"{case.name}: a kernel wrote outside its buffers"
    assert bool(torch.isfinite(Q[inner]).all()) and bool(torch.isfinite(R[inner]).all()), f"{case.name}: uninitialised data was read"
    assert bool(torch.isfinite(Q[halo_or_inner]).all())
    # padding of Q never written; R written on interior nodes only
    pad_after = Q[~halo_or_inner]
    assert bool((pad_after.view(torch.int64) == pad_before.view(torch.int64)).all()), f"{case.name}: row padding of Q was written"
    sent = torch.tensor(SENTINEL, dtype=torch.float64).view(torch.int64).item()
    assert bool((R[~inner].view(torch.int64) == sent).all()), f"{case.name}: R written outside the interior"
    out = Q.clone()
    sol.close()
    return out


@pytest.mark.parametrize("name", NAMES)
def test_guard_bands_padding_and_uninitialised_reads(name):
    case, nsteps = _case(name)
    _run(case, nsteps)


def test_bitwise_reproducible_steps():
    """Races show up as run-to-run differences: three runs of the fused path must agree bit for bit."""
    import torch
    for name in NAMES[:3]:
        case, nsteps = _case(name)
        a = _run(case, nsteps, seed_nan=False)
        for _ in range(2):
            b = _run(case, nsteps, seed_nan=False)
            assert bool((a.view(torch.int64) == b.view(torch.int64)).all()), name
