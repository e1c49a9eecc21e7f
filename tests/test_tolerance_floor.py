"""Pins the tolerance model of tests/parity.py on the CPU (no GPU involved).

The oracle source is compiled a second time with FMA contraction enabled ("FMA twin": identical
source and operation order, only the rounding of a*b+c differs).  Whatever the twin's distance
from the oracle is, no independent fp64 implementation can be expected to come closer.

* 64^3 Taylor-Green vortex at M = 0.1 (BASELINE.json config 2): the twin differs from the oracle
  by MORE than north_star's 1e-11 (Q28 norm) -- the stated tolerance is below the rounding floor
  of this low-Mach problem -- but by only a few units of the floor model u * Phi_c * sum 1/Delta,
  of which tests/parity.py allows K_ULP = 32.
* Sod (config 1): the twin agrees to ~1e-14, so there the stated 1e-11 is the binding tolerance.
"""
import ctypes as C
import subprocess

import numpy as np
import pytest

import parity
from oracle import oracle as O
from paper_2007_14933_b200 import workloads as W


@pytest.fixture(scope="module")
def twin(tmp_path_factory):
    if "fma" not in open("/proc/cpuinfo").read():
        pytest.skip("host CPU has no FMA")
    out = tmp_path_factory.mktemp("twin") / "liboracle_fma.so"
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=fast", "-mfma", "-fopenmp", "-shared", "-fPIC",
           "-o", str(out), str(O._SRC)]
    subprocess.run(cmd, check=True)
    L = C.CDLL(str(out))
    L.oracle_rhs.restype = C.c_int32
    L.oracle_rhs.argtypes = [C.POINTER(O._Params), O._dp, O._dp, C.c_int32, O._dp]
    return L


def _both(twin, case, Q):
    orc = O.Oracle(**case.physics())
    orc.bc(Q)
    R = orc.rhs(Q)
    R2 = np.zeros_like(R)
    assert twin.oracle_rhs(C.byref(orc.p), O._ptr(Q), O._ptr(R2), 3, None) == 0
    return orc.interior(Q), orc.interior(R), orc.interior(R2)


def test_stated_1e11_is_below_rounding_floor_on_low_mach_tgv(twin):
    case = W.tgv(64)
    Qi, R, R2 = _both(twin, case, case.Q0.copy())
    rel = parity.q28(R2, R)
    assert max(rel) > 1e-11, rel                       # the twin itself fails the stated tolerance
    tol, tol_rel, floor = parity.residual_tolerance(case, Qi, R)
    err = np.array([np.abs(R2[c] - R[c]).max() for c in range(5)])
    units = err / (floor / parity.K_ULP)
    assert units.max() < 8.0, units                    # ... by a few rounding units only
    assert units.max() > 0.5, units                    # and the unit is not a gross over-estimate
    assert (err <= tol).all()


def test_stated_1e11_binds_on_sod(twin):
    case = W.sod()
    orc = O.Oracle(**case.physics())
    Q = orc.run(case.Q0.copy(), case.dt, 100)
    Qi, R, R2 = _both(twin, case, Q)
    assert max(parity.q28(R2, R)) < 1e-13
    tol, tol_rel, floor = parity.residual_tolerance(case, Qi, R)
    assert (tol_rel[[0, 1, 4]] >= floor[[0, 1, 4]]).all()      # 1e-11 relative is the larger term
