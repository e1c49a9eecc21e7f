"""osbli_rk3_step_static (include/osbli.h): the RK3 step with the workspace in the library's static device array, for
callers that cannot call cudaMalloc or keep a handle.  Collected last on purpose (the run uses pytest -x).

It launches the same kernels in the same order as osbli_init + osbli_rk3_step, so the states must agree bit for bit
(asserted; the 1e-13 of the other step tests is the stated tolerance).  Two calls in a row per case, cases of
different shapes one after another (the array keeps the previous call's contents), the size limit, and that the
calls leave the device's free memory alone.
"""
import numpy as np
import pytest

import parity
from paper_2007_14933_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _torch():
    import torch
    return torch


def _static_vs_handle(case, nsteps=2, metrics=None):
    """nsteps RK3 steps through the existing path and through the static entry point; returns both final states."""
    from paper_2007_14933_b200 import osbli
    torch = _torch()
    sol = osbli.Solver(metrics=metrics, **case.physics())
    try:
        Qa = sol.to_padded(case.Q0)
        Qb = Qa.clone()
        Ta = sol.empty_state()
        Tb = sol.empty_state(float("nan"))                 # dU need not be initialised (A_0 = 0)
        stream = torch.cuda.current_stream(sol.device).cuda_stream
        for _ in range(nsteps):
            sol.rk3_step(Qa, Ta, case.dt)
        with torch.cuda.device(sol.device):
            for _ in range(nsteps):                        # calls in a row, same stream: serialised
                osbli.osbli_rk3_step_static(sol.params, Qb.data_ptr(), Tb.data_ptr(), case.dt, stream)
        torch.cuda.synchronize()
        return sol.from_padded(Qa), sol.from_padded(Qb)
    finally:
        sol.close()


def _check(name, a, b):
    assert np.isfinite(b).all(), name
    scale = np.abs(a).max(axis=(1, 2, 3), keepdims=True)
    scale = np.where(scale == 0.0, 1.0, scale)
    err = float((np.abs(a - b) / scale).max())
    assert err <= 1e-13, (name, err)                       # the tolerance of the step tests
    assert np.array_equal(a, b), f"{name}: same kernels, same order, but the states differ (max rel {err:.3e})"


def test_static_scratch_matches_the_handle_path():
    # 3-D periodic: fused update, TMA fast viscous path, Q -> Q2 -> Q3 -> Q through the scratch states
    tgv = W.tgv(32)
    _check("tgv32", *_static_vs_handle(tgv))
    # 1-D shocked case: in-place update kernel, R in the scratch
    sod = W.sod()
    _check("sod", *_static_vs_handle(sod, nsteps=5))
    # curvilinear walled box, Sutherland: staged primitives and first differences in the scratch (35 fields)
    box = W.wavy_box(n=(40, 21, 9))
    _check("wavy_box", *_static_vs_handle(box, metrics=parity.metrics_for(box)))
    # back to the first shape: the array now holds another problem's leftovers
    _check("tgv32_again", *_static_vs_handle(tgv))
    # the central fused path and the 7th-order scheme (halo 4) go through the same entry
    _check("tgv32_central4", *_static_vs_handle(W.tgv(32, scheme=W.CENTRAL4)))
    _check("tgv32_wenoz7", *_static_vs_handle(W.tgv(32, scheme=W.WENOZ7)))


def test_static_scratch_limit_and_arguments():
    from paper_2007_14933_b200 import osbli
    torch = _torch()
    assert osbli.osbli_static_scratch_bytes() == 64 << 20
    big = osbli.make_params(**{k: v for k, v in W.tgv(128).physics().items() if k != "dirichlet"})
    assert osbli.osbli_workspace_bytes(big) > osbli.osbli_static_scratch_bytes()
    q = torch.zeros(16, dtype=torch.float64, device="cuda:0")          # never touched: the call must refuse first
    with pytest.raises(osbli.OsbliError) as e:
        osbli.osbli_rk3_step_static(big, q.data_ptr(), q.data_ptr() + 64, 1e-3)
    assert e.value.status == osbli.ESTATIC and "64 MiB" in str(e.value)
    ok = osbli.make_params(**{k: v for k, v in W.tgv(64).physics().items() if k != "dirichlet"})
    assert osbli.osbli_workspace_bytes(ok) <= osbli.osbli_static_scratch_bytes()       # config 2 fits
    with pytest.raises(osbli.OsbliError) as e:
        osbli.osbli_rk3_step_static(ok, q.data_ptr(), q.data_ptr(), 1e-3)               # Q and dU alias
    assert e.value.status == osbli.EINVAL
    torch.cuda.synchronize()
    assert float(q.abs().sum()) == 0.0


def test_static_entry_point_leaves_free_memory_alone():
    from paper_2007_14933_b200 import osbli
    torch = _torch()
    case = W.tgv(32)
    sol = osbli.Solver(**case.physics())
    try:
        Q = sol.to_padded(case.Q0)
        T = sol.empty_state()
        stream = torch.cuda.current_stream(sol.device).cuda_stream
        with torch.cuda.device(sol.device):
            osbli.osbli_rk3_step_static(sol.params, Q.data_ptr(), T.data_ptr(), case.dt, stream)   # set-up, module load
            torch.cuda.synchronize()
            free0, _ = torch.cuda.mem_get_info()
            for _ in range(3):
                osbli.osbli_rk3_step_static(sol.params, Q.data_ptr(), T.data_ptr(), case.dt, stream)
            torch.cuda.synchronize()
            free1, _ = torch.cuda.mem_get_info()
        assert free1 >= free0, (free0, free1)
    finally:
        sol.close()
