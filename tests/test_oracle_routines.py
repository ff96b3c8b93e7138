"""Pins of the oracle's routines O2-O4 against what the mathematics fixes (CPU only).
Citations: SURVEY.md section 8(c)-iii; golden values are re-derived in 40-digit arithmetic by
tests/golden/derive_pins.py (which calls nothing under oracle/)."""
import math

import numpy as np
import pytest

from oracle import fxoracle as fxo
from tests.helpers import golden_rows


def plan(riemann=fxo.RIEMANN_HLLC, gamma=1.4, recon=fxo.RECON_PLM_MINMOD):
    return fxo.OraclePlan((8, 1, 1), 4, 1, gamma, recon, riemann, 2)


# ---------------------------------------------------------------- O2
def test_c2p_closed_form_and_round_trip():
    p = plan()
    rng = np.random.default_rng(1)
    for _ in range(200):
        rho = 10 ** rng.uniform(-3, 3)
        u = rng.normal(size=3) * 10 ** rng.uniform(-2, 2)
        pr = 10 ** rng.uniform(-3, 3)
        E = pr / 0.4 + 0.5 * rho * float(u @ u)
        W = p.cons2prim([rho, rho * u[0], rho * u[1], rho * u[2], E])
        assert W[0] == rho
        np.testing.assert_allclose(W[1:4], u, rtol=4e-16, atol=0)
        # cancellation E - KE amplifies rounding by E/(E-KE)
        amp = E / (pr / 0.4)
        assert abs(W[4] - pr) <= 8 * amp * np.finfo(float).eps * pr


def test_c2p_floors_touch_primitives_only():
    p = plan()
    W = p.cons2prim([1e-20, 0.0, 0.0, 0.0, 1.0])
    assert W[0] == 1e-12
    W = p.cons2prim([1.0, 2.0, 0.0, 0.0, 1.0])  # E - KE = -1 -> p floor
    assert W[4] == 1e-12 and W[0] == 1.0 and W[1] == 2.0


# ---------------------------------------------------------------- O3 PLM
def test_minmod_cases():
    assert fxo.minmod(1.0, 2.0) == 1.0 and fxo.minmod(3.0, 2.0) == 2.0
    assert fxo.minmod(-1.0, -2.0) == -1.0 and fxo.minmod(-3.0, -2.0) == -2.0
    assert fxo.minmod(1.0, -2.0) == 0.0 and fxo.minmod(-1.0, 2.0) == 0.0
    assert fxo.minmod(0.0, 2.0) == 0.0 and fxo.minmod(float("nan"), 1.0) == 0.0
    assert fxo.minmod(1e-300, 1e-300) == 1e-300  # comparison form: no product underflow


# ---------------------------------------------------------------- O3 WENO5
def test_weno5_golden():
    for a, b, c, d, e, eps, val in golden_rows("weno5_pins.txt"):
        got = fxo.weno5(float(a), float(b), float(c), float(d), float(e), float(eps))
        assert got == pytest.approx(float(val), rel=2e-14 if float(val) > 1e-6 else 1e-9)


def test_weno5_survey_printed_values():
    # values printed in SURVEY.md 8(c)-iii (15-16 significant digits)
    assert fxo.weno5(1.0, 1.5, 1.2, 0.9, 1.4) == pytest.approx(1.049359726373859, rel=1e-14)
    assert fxo.weno5(1.4, 0.9, 1.2, 1.5, 1.0) == pytest.approx(1.350640273626141, rel=1e-14)


def test_weno5_quadratic_exact_and_fifth_order():
    # cell averages of a quadratic: all three candidates coincide -> exact face value
    q = lambda x: 0.7 - 1.3 * x + 2.1 * x * x
    Q = lambda x: 0.7 * x - 1.3 * x ** 2 / 2 + 2.1 * x ** 3 / 3
    h = 0.1
    avg = [(Q((i + 1) * h) - Q(i * h)) / h for i in range(-2, 3)]
    assert fxo.weno5(*avg) == pytest.approx(q(1 * h), rel=1e-13)
    # smooth data: error falls ~32x per halving
    errs = []
    for h in (0.1, 0.05, 0.025):
        F = lambda x: -math.cos(x)
        avg = [(F(1.0 + (i + 1) * h) - F(1.0 + i * h)) / h for i in range(-2, 3)]
        errs.append(abs(fxo.weno5(*avg) - math.sin(1.0 + h)))
    assert errs[0] / errs[1] > 20 and errs[1] / errs[2] > 20


# ---------------------------------------------------------------- O4
@pytest.mark.parametrize("solver", [fxo.RIEMANN_HLLE, fxo.RIEMANN_HLLC])
def test_riemann_consistency_bitwise(solver):
    p = plan(solver)
    rng = np.random.default_rng(2)
    for _ in range(100):
        W = np.array([10 ** rng.uniform(-2, 2), *rng.normal(size=3), 10 ** rng.uniform(-2, 2)])
        F = p.riemann_flux(W, W)
        rho, un, t1, t2, pr = W
        E = pr * (1.0 / (1.4 - 1.0)) + 0.5 * rho * (un * un + t1 * t1 + t2 * t2)
        cs = math.sqrt(1.4 * pr / rho)
        if abs(un) > cs * (1 + 1e-12):  # supersonic: F(W,W) = F(W) bitwise
            exact = np.array([rho * un, rho * un * un + pr, rho * un * t1, rho * un * t2, un * (E + pr)])
            assert np.array_equal(F, exact)
        else:
            exact = np.array([rho * un, rho * un * un + pr, rho * un * t1, rho * un * t2, un * (E + pr)])
            np.testing.assert_allclose(F, exact, rtol=1e-13, atol=1e-13 * (abs(exact).max() + pr))


@pytest.mark.parametrize("solver", [fxo.RIEMANN_HLLE, fxo.RIEMANN_HLLC])
def test_riemann_supersonic_upwind_bitwise(solver):
    p = plan(solver)
    WL = np.array([1.0, 5.0, 0.3, -0.2, 1.0])
    WR = np.array([0.5, 4.0, -0.1, 0.4, 0.7])
    flux = lambda W: np.array([W[0] * W[1], W[0] * W[1] * W[1] + W[4], W[0] * W[1] * W[2], W[0] * W[1] * W[3],
                               W[1] * ((W[4] * (1.0 / (1.4 - 1.0)) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)) + W[4])])
    assert np.array_equal(p.riemann_flux(WL, WR), flux(WL))
    WLm, WRm = WR.copy(), WL.copy()
    WLm[1] *= -1
    WRm[1] *= -1
    assert np.array_equal(p.riemann_flux(WLm, WRm), flux(WRm))


@pytest.mark.parametrize("solver", [fxo.RIEMANN_HLLE, fxo.RIEMANN_HLLC])
@pytest.mark.parametrize("speeds", [0, 1])
def test_riemann_mirror_antisymmetry_bitwise(solver, speeds):
    p = plan(solver)
    p.set_option(fxo.OPT_WAVESPEED, speeds)
    rng = np.random.default_rng(3)
    for _ in range(300):
        WL = np.array([10 ** rng.uniform(-1, 1), *rng.normal(size=3), 10 ** rng.uniform(-1, 1)])
        WR = np.array([10 ** rng.uniform(-1, 1), *rng.normal(size=3), 10 ** rng.uniform(-1, 1)])
        F = p.riemann_flux(WL, WR)
        WLm, WRm = WR.copy(), WL.copy()
        WLm[1] *= -1
        WRm[1] *= -1
        Fm = p.riemann_flux(WLm, WRm)
        assert np.array_equal(Fm, np.array([-F[0], F[1], -F[2], -F[3], -F[4]]))


def test_hllc_keeps_isolated_contact():
    p = plan(fxo.RIEMANN_HLLC)
    for u in (0.3, -0.3, 0.0):
        WL = np.array([1.0, u, 0.2, -0.1, 1.0])
        WR = np.array([0.25, u, -0.5, 0.7, 1.0])
        F = p.riemann_flux(WL, WR)
        W = WL if u >= 0 else WR
        E = W[4] / 0.4 + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)
        exact = np.array([W[0] * u, W[0] * u * u + W[4], W[0] * u * W[2], W[0] * u * W[3], u * (E + W[4])])
        np.testing.assert_allclose(F, exact, rtol=0, atol=4e-15)
    # HLLE smears it: mass flux differs from upwind
    pe = plan(fxo.RIEMANN_HLLE)
    F = pe.riemann_flux(np.array([1.0, 0.0, 0, 0, 1.0]), np.array([0.25, 0.0, 0, 0, 1.0]))
    assert abs(F[0]) > 0.1


def test_sod_interface_flux_golden():
    names = {"hlle": fxo.RIEMANN_HLLE, "hllc": fxo.RIEMANN_HLLC}
    for solver, speeds, f0, f1, f2 in golden_rows("sod_interface_flux.txt"):
        p = plan(names[solver])
        p.set_option(fxo.OPT_WAVESPEED, 0 if speeds == "einfeldt" else 1)
        F = p.riemann_flux(np.array([1.0, 0, 0, 0, 1.0]), np.array([0.125, 0, 0, 0, 0.1]))
        np.testing.assert_allclose(F[[0, 1, 4]], [float(f0), float(f1), float(f2)], rtol=2e-15 * 10)
        assert F[2] == 0 and F[3] == 0
    # the numbers SURVEY.md prints for the default (Einfeldt) speeds
    F = plan(fxo.RIEMANN_HLLE).riemann_flux(np.array([1.0, 0, 0, 0, 1.0]), np.array([0.125, 0, 0, 0, 0.1]))
    np.testing.assert_allclose(F[[0, 1, 4]], [0.510713703157072, 0.543964198004823, 1.31326380811819], rtol=1e-14)
    F = plan(fxo.RIEMANN_HLLC).riemann_flux(np.array([1.0, 0, 0, 0, 1.0]), np.array([0.125, 0, 0, 0, 0.1]))
    np.testing.assert_allclose(F[[0, 1, 4]], [0.431067162607704, 0.489954454827689, 1.1628640656485], rtol=1e-14)


def test_transverse_momentum_is_advected():
    # flux of t1 momentum = mass flux * upwind t1 for HLLC in a pure shear
    p = plan(fxo.RIEMANN_HLLC)
    F = p.riemann_flux(np.array([1.0, 0.5, 2.0, -1.0, 1.0]), np.array([1.0, 0.5, -3.0, 4.0, 1.0]))
    assert F[2] == pytest.approx(F[0] * 2.0, rel=1e-14) and F[3] == pytest.approx(F[0] * -1.0, rel=1e-14)


def test_plan_argument_checks():
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 1, 1, 1.4, 0, 0, 2)  # nguard < 2
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 2, 1, 1.4, 1, 0, 2)  # WENO5 needs 3
    with pytest.raises(ValueError):
        fxo.OraclePlan((2, 1, 1), 3, 1, 1.4, 0, 0, 2)  # nguard > block dim
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 4, 1, 1.0, 0, 0, 2)  # gamma <= 1
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 4, 1, 1.4, 0, 0, 4)  # rk order
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 4, 1, 1.4, 0, 0, 2, nvars=4)
    with pytest.raises(ValueError):
        fxo.OraclePlan((8, 1, 1), 4, 1, 1.4, 0, 0, 2, nvars=33)  # more than 27 passive scalars [B11]
