"""Pins of the oracle's communication-avoiding step (fxo_hydro_advance_ca, reading B17).

The variant fills guard zones once per step and lets stage s update the interior extended by (n - s) R zones.  On blocks
that share dx with their neighbours every extended zone is a neighbour's interior zone updated with the same formula from
the same numbers, so the step must reproduce fxo_hydro_advance -- which is pinned on its own (tests/test_oracle_scheme.py:
Sod against the exact solution, conservation, symmetry, ...) -- BIT FOR BIT: a wrong reach (a zone read that no stage
wrote: the oracle poisons those with NaN), a missing re-imaging of a physical boundary, a wrong extension per stage or a
wrong beta fails the equality.  Where the premise does not hold (a different dx per block) the two must differ."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import oracle_plan_for

PLM, WENO = fxo.RECON_PLM_MINMOD, fxo.RECON_WENO5

CASES = [
    # config, nb, recon, rk, nguard, bc
    (5, (2, 2, 2), PLM, 2, 4, "periodic"),   # configs 3 / 5 as they are run: RK2, PLM, 4 guard zones
    (5, (2, 2, 2), PLM, 3, 6, "periodic"),
    (4, (2, 2, 2), WENO, 2, 6, "periodic"),
    (4, (2, 1, 2), WENO, 3, 9, "periodic"),  # config 4's scheme needs 9 guard zones
    (5, (2, 2, 2), PLM, 2, 4, "outflow"),
    (5, (2, 2, 1), PLM, 3, 6, "reflect"),
    (4, (1, 2, 2), WENO, 2, 7, "outflow"),   # more guard zones than needed
    (2, (2, 2, 1), PLM, 2, 4, "periodic"),   # 2-D
    (2, (2, 2, 1), PLM, 3, 6, "outflow"),
    (1, (1, 1, 1), PLM, 2, 4, "outflow"),    # 1-D, one block
]


def _setup(number, nb, recon, rk, g, bc, riemann=None):
    cfg = inputs.config(number, nb=nb)
    cfg.nguard = g
    plan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, rk=rk, riemann=riemann)
    U = inputs.embed(cfg, inputs.block_interiors(cfg, coords)).numpy()
    return cfg, plan, U, inputs.dx_array(cfg)


@pytest.mark.parametrize("number,nb,recon,rk,g,bc", CASES)
def test_ca_step_is_the_standard_step_bit_for_bit(number, nb, recon, rk, g, bc):
    cfg, plan, U, dx = _setup(number, nb, recon, rk, g, bc)
    A, B = U.copy(), U.copy()
    for step in range(3):
        dt = plan.compute_dt(A, dx, cfg.cfl)
        plan.advance(A, dx, dt)
        plan.advance_ca(B, dx, dt)
        assert np.array_equal(plan.interior(A), plan.interior(B)), step
    assert np.isfinite(plan.interior(B)).all()
    assert not np.array_equal(plan.interior(B), plan.interior(U))  # the state did move


@pytest.mark.parametrize("riemann", [fxo.RIEMANN_HLLE, fxo.RIEMANN_HLLC])
def test_ca_step_with_gravity_and_walls(riemann):
    cfg, plan, U, dx = _setup(5, (2, 2, 2), PLM, 2, 4, "reflect", riemann=riemann)
    plan.set_option(fxo.OPT_GRAVITY_Z, -0.7)
    plan.set_option(fxo.OPT_GRAVITY_X, 0.2)
    A, B = U.copy(), U.copy()
    for step in range(3):
        dt = plan.compute_dt(A, dx, cfg.cfl)
        plan.advance(A, dx, dt)
        plan.advance_ca(B, dx, dt)
    assert np.array_equal(plan.interior(A), plan.interior(B))


def test_ca_step_does_not_depend_on_guard_zone_contents_on_entry():
    cfg, plan, U, dx = _setup(5, (2, 2, 2), PLM, 2, 4, "periodic")
    A = U.copy()
    B = np.full_like(U, np.nan)
    plan.interior(B)[...] = plan.interior(U)
    dt = plan.compute_dt(A, dx, cfg.cfl)
    plan.advance_ca(A, dx, dt)
    plan.advance_ca(B, dx, dt)
    assert np.array_equal(plan.interior(A), plan.interior(B))


def test_ca_step_needs_rk_order_times_reach_guard_zones():
    for recon, rk, g in [(PLM, 3, 4), (WENO, 2, 4), (WENO, 3, 8)]:
        cfg, plan, U, dx = _setup(4, (2, 2, 2), recon, rk, g, "periodic")
        with pytest.raises(ValueError, match="-3"):
            plan.advance_ca(U, dx, 1e-4)


def test_ca_step_differs_where_neighbours_do_not_share_dx():
    """The premise, from the other side: with a different dx per block an extended zone is NOT what the neighbour computes."""
    cfg, plan, U, dx = _setup(5, (2, 2, 2), PLM, 2, 4, "periodic")
    dx = np.random.default_rng(3).uniform(1.0 / 40, 1.0 / 24, size=dx.shape)
    A, B = U.copy(), U.copy()
    dt = plan.compute_dt(A, dx, cfg.cfl)
    plan.advance(A, dx, dt)
    plan.advance_ca(B, dx, dt)
    assert not np.array_equal(plan.interior(A), plan.interior(B))


def test_ca_step_conserves_on_a_periodic_tiling():
    cfg, plan, U, dx = _setup(5, (2, 2, 2), PLM, 2, 4, "periodic")
    I0 = plan.interior(U).copy()
    for _ in range(5):
        plan.advance_ca(U, dx, plan.compute_dt(U, dx, cfg.cfl))
    for v in (0, 4):
        s0, s1 = I0[v].sum(dtype=np.longdouble), plan.interior(U)[v].sum(dtype=np.longdouble)
        assert abs(s1 - s0) <= 1e-13 * abs(s0)
