"""Small invocations of the CUDA path for `compute-sanitizer` (memcheck / racecheck / initcheck / synccheck).

    compute-sanitizer --tool memcheck python tests/sanitizer_cases.py

Every kernel family runs once on a case small enough for the sanitizer's 10-100x slow-down: the fused sweep +
stage update with periodic write-through into other blocks' halos (the smallest legal box, 5 x 7 x 6, and a ragged
one spanning several tiles), the TMA + mbarrier plane ring of the fast viscous kernel, the cp.async per-thread
slots, the warp-private transposed tiles of the x sweep, the curvilinear / walled general path, the 1-D path,
the central scheme and the halo fills.  No oracle here: parity is tests/test_gpu_parity.py's job; this script only
has to touch the memory the kernels touch.  Results are checked for finiteness so that nothing is optimised away.
"""
import sys
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent.parent
sys.path.insert(0, str(ROOT))

import torch                                                     # noqa: E402
from paper_2007_14933_b200 import osbli                          # noqa: E402
from paper_2007_14933_b200 import workloads as W                 # noqa: E402


def periodic_box(n, scheme=W.TENO5, visc=W.VISC_CONST):
    c = W.tgv(8, scheme=scheme, visc=visc)
    i, j, k = W.padded_index_grids(n, scheme)
    x, y, z = 2 * np.pi * i / n[0], 2 * np.pi * j / n[1], 2 * np.pi * k / n[2]
    g, M = 1.4, 0.4
    u = np.sin(x) * np.cos(y) * np.cos(z)
    v = -np.cos(x) * np.sin(y) * np.cos(z)
    w = 0.3 * np.sin(x + y) * np.sin(z)
    p = 1.0 / (g * M * M) + (np.cos(2 * x) + np.cos(2 * y)) * (np.cos(2 * z) + 2.0) / 16.0
    rho = 1.0 + 0.2 * np.sin(x + 2 * y - z)
    c.n = n
    c.Q0 = np.ascontiguousarray(W.conservative(rho, u, v, w, p, g))
    c.delta = tuple(2 * np.pi / v_ for v_ in n)
    c.Minf, c.Re, c.dt = M, 100.0, 5e-4
    return c


def run(name, case, nsteps, metrics=None, rk4=False):
    sol = osbli.Solver(metrics=metrics, **case.physics())
    Q = sol.to_padded(case.Q0)
    Qtmp = sol.empty_state()
    R = sol.empty_state(0.0)
    sol.bc(Q)
    sol.rhs(Q, R)
    for _ in range(nsteps):
        (sol.rk4_step if rk4 else sol.rk3_step)(Q, Qtmp, case.dt)
    torch.cuda.synchronize()
    h, n, lay = case.halo, case.n, sol.layout
    core = Q[:, h[2]:h[2] + n[2], h[1]:h[1] + n[1], lay.x_offset:lay.x_offset + n[0]]
    rc = R[:, h[2]:h[2] + n[2], h[1]:h[1] + n[1], lay.x_offset:lay.x_offset + n[0]]
    ok = bool(torch.isfinite(core).all()) and bool(torch.isfinite(rc).all())
    print(f"{name}: {'ok' if ok else 'NON-FINITE'} launches={sol.launch_count()}", flush=True)
    sol.close()
    assert ok, name


def main():
    torch.cuda.set_device(0)
    run("tgv16_teno5_visc (fused update, write-through, TMA viscous ring)", W.tgv(16), 2)
    run("pbox_5x7x6 (smallest legal box: images on both sides)", periodic_box((5, 7, 6)), 2)
    run("pbox_70x37x35_teno6 (ragged tiles)", periodic_box((70, 37, 35), scheme=W.TENO6), 1)
    run("pbox_40x33x1_wenoz (2-D, last sweep = y)", periodic_box((40, 33, 1), scheme=W.WENOZ5), 2)
    run("sod (1-D path, separate update)", W.sod(), 50)
    run("tgv16_central4", W.tgv(16, scheme=W.CENTRAL4), 2)
    run("tgv16_rk4", W.tgv(16), 1, rk4=True)
    wb = W.wavy_box(n=(40, 21, 9))
    run("wavy_box (curvilinear, wall / Dirichlet / extrapolation / periodic, Sutherland)", wb, 2, metrics=W.approximate_metrics(wb))
    ch = W.channel(n=(24, 33, 6), noise=1e-3, scheme=W.TENO5)
    run("channel3d (adiabatic wall, body force)", ch, 2)
    ssp = W.tgv(16)
    ssp.rk3_form, ssp.averaging = W.RK3_SSP, W.AVG_SIMPLE
    run("tgv16_ssp_simple_avg", ssp, 1)
    run("pbox_37x21x13_wenoz7 (halo 4, tiled sweeps)", periodic_box((37, 21, 13), scheme=W.WENOZ7), 1)
    wb7 = W.wavy_box(n=(40, 21, 9), scheme=W.WENOZ7)
    run("wavy_box_wenoz7", wb7, 1, metrics=W.approximate_metrics(wb7))
    print("sanitizer cases done")


if __name__ == "__main__":
    main()
