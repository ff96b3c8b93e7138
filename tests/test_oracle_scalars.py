"""Pins of the oracle's passive mass scalars (reading B11; "a perfect-gas EOS with a
multispecies variant").  The scalar code is new; what it is pinned to is not:
the mass flux and the transverse-momentum flux (pinned by the 40-digit Sod values and the routine tests of
test_oracle_routines.py), the exact solution of linear advection, conservation, and the hydro variables of a
run without scalars."""
import dataclasses

import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import oracle_plan_for


def _states(rng, n, ns):
    """Random face-frame states (rho, un, ut1, ut2, p, X_1..X_ns), subsonic and supersonic both ways."""
    W = np.empty((n, 5 + ns))
    W[:, 0] = np.exp(rng.normal(0, 0.7, n))
    W[:, 1] = rng.normal(0, 1.5, n)
    W[:, 2:4] = rng.normal(0, 1.0, (n, 2))
    W[:, 4] = np.exp(rng.normal(0, 0.7, n))
    W[:, 5:] = rng.random((n, ns))
    return W


@pytest.mark.parametrize("riemann", [fxo.RIEMANN_HLLE, fxo.RIEMANN_HLLC])
@pytest.mark.parametrize("wavespeed", [0, 1])
def test_flux_routine(riemann, wavespeed):
    ns = 3
    plan = fxo.OraclePlan((8, 1, 1), 2, 1, 1.4, 0, riemann, 2, nvars=5 + ns)
    plan.set_option(fxo.OPT_WAVESPEED, wavespeed)
    plan5 = fxo.OraclePlan((8, 1, 1), 2, 1, 1.4, 0, riemann, 2)
    plan5.set_option(fxo.OPT_WAVESPEED, wavespeed)
    rng = np.random.default_rng(11630)
    WL, WR = _states(rng, 400, ns), _states(rng, 400, ns)
    seen = set()
    for a, b in zip(WL, WR):
        F = plan.riemann_flux_nv(a, b)
        # the hydro components do not see the scalars
        assert np.array_equal(F[:5], plan5.riemann_flux(a[:5], b[:5]))
        # rounding scale: density times the fastest signal speed (the HLL average cancels terms of that size)
        scale = (a[0] + b[0]) * (abs(a[1]) + abs(b[1]) + np.sqrt(1.4 * a[4] / a[0]) + np.sqrt(1.4 * b[4] / b[0]))
        # a scalar equal to the transverse velocity is the transverse momentum, bit for bit
        a2, b2 = a.copy(), b.copy()
        a2[5], b2[5], a2[6], b2[6] = a[2], b[2], a[3], b[3]
        F2 = plan.riemann_flux_nv(a2, b2)
        assert F2[5] == F2[2] and F2[6] == F2[3]
        # X = 1 is the density, X = 0 is nothing, X = c on both sides is c times the mass flux
        a2[5], b2[5], a2[6], b2[6], a2[7], b2[7] = 1.0, 1.0, 0.0, 0.0, 0.375, 0.375
        F2 = plan.riemann_flux_nv(a2, b2)
        assert F2[5] == F2[0] and F2[6] == 0.0
        assert abs(F2[7] - 0.375 * F2[0]) <= 1e-15 * scale
        # linear in (X_L, X_R), and the two unit responses add up to the mass flux
        a2[5], b2[5], a2[6], b2[6] = 1.0, 0.0, 0.0, 1.0
        G = plan.riemann_flux_nv(a2, b2)
        assert abs(G[5] + G[6] - F[0]) <= 1e-15 * scale
        assert abs(a[7] * G[5] + b[7] * G[6] - F[7]) <= 1e-15 * scale
        if riemann == fxo.RIEMANN_HLLC:
            # HLLC: the flux is the upwind abundance times the mass flux (contact-resolving: G is one-sided)
            up = a[5:] if F[0] >= 0 else b[5:]
            assert np.all(np.abs(F[5:] - up * F[0]) <= 1e-15 * scale)
            seen.add(F[0] >= 0)
        # mirror antisymmetry, bitwise
        am, bm = b.copy(), a.copy()
        am[1], bm[1] = -am[1], -bm[1]
        Fm = plan.riemann_flux_nv(am, bm)
        assert np.array_equal(Fm[5:], -F[5:])
    if riemann == fxo.RIEMANN_HLLC:
        assert seen == {True, False}


def test_cons2prim_scalars():
    plan = fxo.OraclePlan((8, 1, 1), 2, 1, 1.4, 0, 1, 2, nvars=7)
    U = np.array([0.8, 0.4, -0.2, 0.1, 2.5, 0.2, 0.8])
    W = plan.cons2prim_nv(U)
    assert np.array_equal(W[:5], plan.cons2prim(U[:5]))
    assert abs(W[5] - 0.25) <= 1e-16 and W[6] == 1.0
    # floored density: the scalar is divided by the same density as the momenta
    U[0] = 1e-30
    W = plan.cons2prim_nv(U)
    assert W[5] == U[5] * (1.0 / 1e-12) and W[1] == U[1] * (1.0 / 1e-12)


def _setup(number, nb, ns, bc=None, recon=None, riemann=None, rk=None, order=inputs.ORDER_LEX):
    cfg = inputs.config(number, nb=nb)
    plan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk, nvars=5 + ns, order=order)
    Ui = inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), ns)
    return cfg, plan, coords, Ui


CASES = [(5, (2, 2, 2), None, None, None, None), (4, (2, 2, 2), None, None, None, None),
         (2, (4, 4, 1), None, 1, 0, 3), (5, (2, 2, 1), "reflect", None, 0, None),
         (5, (2, 1, 2), "outflow", 1, None, None)]


@pytest.mark.parametrize("number,nb,bc,recon,riemann,rk", CASES)
def test_hydro_unaffected_and_special_abundances(number, nb, bc, recon, riemann, rk):
    """The five hydro variables are bit for bit those of a run without scalars; rho X with X = 1 stays the density
    and a uniform abundance stays uniform (to rounding), X = 0 stays 0 exactly."""
    cfg, plan, coords, Ui = _setup(number, nb, 4, bc, recon, riemann, rk)
    Ui[5] = Ui[0]
    Ui[6] = 0.0
    Ui[7] = 0.3125 * Ui[0]
    plan5, _, _ = oracle_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk)
    U = inputs.embed(cfg, Ui).numpy().copy()
    U5 = inputs.embed(cfg, Ui[:5]).numpy().copy()
    dx = inputs.dx_array(cfg)
    for _ in range(4):
        dt = plan.compute_dt(U, dx, cfg.cfl)
        assert dt == plan5.compute_dt(U5, dx, cfg.cfl)
        plan.advance(U, dx, dt)
        plan5.advance(U5, dx, dt)
    I, I5 = plan.interior(U), plan5.interior(U5)
    assert not np.array_equal(I5, Ui[:5].numpy())  # something happened
    assert np.array_equal(I[:5], I5)
    assert np.max(np.abs(I[5] / I[0] - 1.0)) <= 2e-15  # rho * (1/rho) is 1 to an ulp, not exactly
    assert np.all(I[6] == 0.0)
    assert np.max(np.abs(I[7] / I[0] - 0.3125)) <= 2e-15
    assert np.all(np.isfinite(I[8]))


@pytest.mark.parametrize("recon,riemann,rk", [(0, 1, 2), (1, 0, 3), (0, 0, 2), (1, 1, 3)])
def test_scalar_follows_transverse_momentum(recon, riemann, rk):
    """2-D flow with a velocity component w out of the plane: m_z is advected passively (it enters the energy, not
    the in-plane dynamics' form), and a scalar with X = w is m_z bit for bit, step after step."""
    cfg, plan, coords, Ui = _setup(2, (4, 4, 1), 2, None, recon, riemann, rk)
    rho = Ui[0]
    w = Ui[5] / rho - 0.3          # smooth field of either sign
    Ui[3] = rho * w
    Ui[4] = Ui[4] + 0.5 * rho * w * w
    Ui[5] = Ui[3]
    U = inputs.embed(cfg, Ui).numpy().copy()
    dx = inputs.dx_array(cfg)
    for _ in range(6):
        plan.advance(U, dx, plan.compute_dt(U, dx, cfg.cfl))
        I = plan.interior(U)
        assert np.array_equal(I[5], I[3])
    assert np.abs(I[3]).max() > 0.1


@pytest.mark.parametrize("number,nb", [(2, (4, 4, 1)), (5, (2, 2, 2)), (4, (2, 2, 2))])
def test_scalar_mass_is_conserved(number, nb):
    cfg, plan, coords, Ui = _setup(number, nb, 3)
    U = inputs.embed(cfg, Ui).numpy().copy()
    dx = inputs.dx_array(cfg)
    before = plan.interior(U)[5:].sum(axis=(1, 2, 3, 4))
    absum = np.abs(plan.interior(U)[5:]).sum(axis=(1, 2, 3, 4))
    for _ in range(5):
        plan.advance(U, dx, plan.compute_dt(U, dx, cfg.cfl))
    after = plan.interior(U)[5:].sum(axis=(1, 2, 3, 4))
    assert np.all(np.abs(after - before) <= 1e-13 * absum)
    assert not np.array_equal(plan.interior(U)[5:], Ui[5:].numpy())


def _advection_error(N, recon, rk, riemann):
    """Uniform gas moving at u = 1 through a periodic unit interval carrying X(x) = 0.5 + 0.4 sin(2 pi x):
    the exact solution at time t is X(x - t)."""
    base = inputs.config(1)
    cfg = dataclasses.replace(base, block_dims=(N // 2, 1, 1), nb=(2, 1, 1), bc="periodic", full_nb=None)
    plan, neigh, coords = oracle_plan_for(cfg, recon=recon, riemann=riemann, rk=rk, nvars=6)
    x = (np.arange(N) + 0.5) / N
    X0 = 0.5 + 0.4 * np.sin(2 * np.pi * x)
    g = cfg.nguard
    U = np.full(plan.shape, np.nan)
    prim = [1.0, 1.0, 0.0, 0.0, 1.0 / 0.4 + 0.5]
    for b in range(2):
        for v in range(5):
            U[v, b, 0, 0, g:g + N // 2] = prim[v]
        U[5, b, 0, 0, g:g + N // 2] = X0[b * (N // 2):(b + 1) * (N // 2)]
    dx = np.full((2, 3), 1.0 / N)
    t_end, t = 0.5, 0.0
    while t < t_end:
        dt = min(plan.compute_dt(U, dx, 0.4), t_end - t)
        plan.advance(U, dx, dt)
        t += dt
    I = plan.interior(U)
    assert np.all(I[0] == 1.0) and np.all(I[1] == 1.0)     # the carrier stays uniform, bitwise
    X = np.concatenate([I[5, 0, 0, 0], I[5, 1, 0, 0]])
    return float(np.mean(np.abs(X - (0.5 + 0.4 * np.sin(2 * np.pi * (x - t_end))))))


@pytest.mark.parametrize("recon,rk,riemann,order_min,err_max", [(0, 2, 1, 1.6, 2e-3), (0, 2, 0, 1.6, 2e-3),
                                                                 (1, 3, 1, 2.8, 2e-6), (1, 3, 0, 2.8, 2e-6)])
def test_advection_against_exact_solution(recon, rk, riemann, order_min, err_max):
    e = [_advection_error(N, recon, rk, riemann) for N in (32, 64, 128)]
    assert e[0] > e[1] > e[2]
    order = np.log2(e[0] / e[2]) / 2
    assert order >= order_min, (e, order)
    assert e[2] <= err_max, e


def test_generator_scalars_are_blockwise_reproducible():
    cfg = inputs.config(5, nb=(2, 2, 2))
    coords = inputs.block_coords(cfg.nb)
    full = inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), 4)
    one = inputs.with_scalars(cfg, coords[3:4], inputs.block_interiors(cfg, coords[3:4]), 4)
    assert torch.equal(full[:, 3:4], one)
    X = full[5:] / full[0]
    assert float(X.min()) >= 0.0 and float(X.max()) <= 1.0 and float(X[1].max()) == 1.0 and float(X[1].min()) == 0.0
