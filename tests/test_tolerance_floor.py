"""Pins the tolerance model of tests/parity.py on the CPU (no GPU involved).

The oracle source is compiled a second time with FMA contraction enabled ("FMA twin": identical
source and operation order, only the rounding of a*b+c differs).  Whatever the twin's distance
from the oracle is, no independent fp64 implementation can be expected to come closer.

* 64^3 Taylor-Green vortex at M = 0.1 (BASELINE.json config 2): the twin differs from the oracle
  by MORE than north_star's 1e-11 (Q28 norm) -- the stated tolerance is below the rounding floor
  of this low-Mach problem -- but by only a few units of the floor model u * Phi_c * sum 1/Delta,
  of which tests/parity.py allows K_ULP = 32.
* Sod (config 1): the twin agrees to ~1e-14, so there the stated 1e-11 is the binding tolerance.
* Quasi-2-D slab (config 4 at reduced size, same grid / flow / noise recipe): the twin misses 1e-11 on the
  spanwise momentum, whose residual is driven by the seeded noise alone.

The twin shares the oracle's operation order, so it UNDER-states what an independently ordered fp64 evaluation
can reach.  The second yardstick needs no second implementation at all: flip the last bit of every entry of the
oracle's input (a relative change of 2^-53, below anything a caller can control) and see how far the oracle's
own residual moves.  In units of the floor model 2^-53 Phi_c sum|grad xi| that is 1-7 for every variable of every
case -- the unit is neither an over- nor an under-estimate, and K_ULP = 16 is about 3x the oracle's own
sensitivity to input rounding.  With the first version of the model (momentum floor without the (|u|+a) rho term)
the slab's spanwise momentum alone falls out of that band, which is what the term repairs.
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


def test_twin_misses_1e11_on_the_spanwise_momentum_of_the_slab(twin):
    """Config 4's structure at 100 x 50 x 8: rho w = 0 up to the seeded density noise, so ||R_{rho w}|| is ~1e-5 of
    the other momentum residuals while its fluxes are built from theta-field contributions of size (|u|+a) rho."""
    case = W.sbli_slab(n=(100, 50, 8))
    metrics = parity.metrics_for(case)
    orc = parity.make_oracle(case, metrics)
    Q = orc.bc(case.Q0.copy())
    R = orc.rhs(Q)
    R2 = np.zeros_like(R)
    assert twin.oracle_rhs(C.byref(orc.p), O._ptr(Q), O._ptr(R2), 3, None) == 0
    Qi, R, R2 = orc.interior(Q), orc.interior(R), orc.interior(R2)
    rel = parity.q28(R2, R)
    assert rel[3] > 1e-11 and max(rel[c] for c in (0, 1, 2, 4)) < 1e-12, rel
    tol, tol_rel, floor = parity.residual_tolerance(case, Qi, R, metrics)
    err = np.array([np.abs(R2[c] - R[c]).max() for c in range(5)])
    assert (err / (floor / parity.K_ULP)).max() < 4.0


def _last_bit_sensitivity(case, steps=0, trials=2, seed=0):
    """max over trials of |R(Q with random last-bit flips) - R(Q)| per variable, in units of the floor model
    (current and first version), oracle only."""
    metrics = parity.metrics_for(case)
    orc = parity.make_oracle(case, metrics)
    Q = case.Q0.copy()
    if steps:
        orc.run(Q, case.dt, steps)
    orc.bc(Q)
    R = orc.interior(orc.rhs(Q))
    rng = np.random.default_rng(seed)
    worst = np.zeros(5)
    for _ in range(trials):
        Qp = Q.copy()
        core = orc.interior(Qp)
        sgn = rng.integers(-1, 2, size=core.shape)
        core[...] = np.where(sgn > 0, np.nextafter(core, np.inf), np.where(sgn < 0, np.nextafter(core, -np.inf), core))
        orc.bc(Qp)
        Rp = orc.interior(orc.rhs(Qp))
        worst = np.maximum(worst, [np.abs(Rp[c] - R[c]).max() for c in range(5)])
    Qi = orc.interior(Q)
    unit = parity.U * parity.flux_scale(case, Qi, metrics)
    unit_v1 = parity.U * parity.flux_scale(case, Qi, metrics, momentum_rho_term=False)
    den = np.array([np.abs(R[c]).max() for c in range(5)])
    return worst / unit, worst / unit_v1, worst / np.where(den > 0, den, 1.0)


def test_last_bit_of_the_input_moves_the_oracle_by_a_few_floor_units_everywhere():
    for case, steps, active in ((W.tgv(32), 0, (0, 1, 2, 3, 4)), (W.wavy_box(n=(24, 20, 8)), 0, (0, 1, 2, 3, 4)),
                                (W.sod(), 100, (0, 1, 4))):
        units, _, rel = _last_bit_sensitivity(case, steps)
        assert 0.5 < units[list(active)].min() and units[list(active)].max() < 8.0, (case.name, units)
    # low-Mach TGV: one flipped input bit already moves the residual by more than the stated 1e-11
    assert _last_bit_sensitivity(W.tgv(32))[2].max() > 1e-11


def test_momentum_floor_needs_the_rho_term_on_the_slab():
    """Developed reduced-size slab: in the current units every variable sits in the same 0.5-8 band; in the first
    version's units the spanwise momentum is the outlier (> 8 and more than 1.5x any other variable) -- and the
    stated 1e-11 is missed on that variable by the oracle against its own last-bit-perturbed input."""
    units, units_v1, rel = _last_bit_sensitivity(W.sbli_slab(n=(100, 50, 8)), steps=20, trials=3)
    assert 0.5 < units.min() and units.max() < 8.0, units
    assert units_v1[3] > 8.0 and units_v1[3] > 1.5 * max(units_v1[c] for c in (0, 1, 4)), units_v1
    assert rel[3] > 1e-11 and max(rel[c] for c in (0, 1, 2, 4)) < 1e-12, rel
