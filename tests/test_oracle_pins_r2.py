"""Round-2 oracle pins (CPU): the pieces VERDICT r1 listed as unpinned.

* the WENO5 positivity fallback [A6] -- per side, all variables (passive scalars too [B11]), status bit;
* fxo_debug_compute_fluxes (face indexing [A17], array layout [B1]) against the 40-digit Sod interface flux and the
  upwind flux of a uniform state;
* fxo_status bits after an advance that hits the floors [A7];
* the frame rotation of face_flux: config 1 laid along y and along z is the x run, bit for bit.
"""
import numpy as np
import pytest

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import cliff_state, golden_rows, oracle_plan_for


# ------------------------------------------------------------------------------------------------ A6
def _line_plan(ns=0, recon=fxo.RECON_WENO5):
    plan = fxo.OraclePlan((16, 1, 1), 4, 1, 1.4, recon, fxo.RIEMANN_HLLC, 3, nvars=5 + ns)
    return plan


def _cliff_line(ns, which):
    """Primitive line of 12 cells whose WENO5 value at the face between cells 5 and 6 is <= 0 in rho on the left side
    (which = 'L'), in p on the right side ('R') or both ('LR'): a linear ramp steeper than 2 q / cell running into a
    plateau 1e6 times higher, so that the smooth stencil is the extrapolating one."""
    n = 12
    W = np.empty((5 + ns, n))
    rng = np.random.default_rng(7)
    W[0] = 1.0 + rng.random(n)
    W[1:4] = 0.3 * rng.standard_normal((3, n))
    W[4] = 1.0 + rng.random(n)
    for s in range(ns):
        W[5 + s] = rng.random(n)
    if "L" in which:  # cells 3,4,5 = 5.5, 3, 0.5 then 1e6: p0 = (2*5.5 - 7*3 + 11*0.5)/6 = -0.75
        W[0, 3:6] = (5.5, 3.0, 0.5)
        W[0, 6:9] = 1e6
    if "R" in which:  # mirrored for the right state of the same face: cells 8,7,6 = 5.5, 3, 0.5, cells 5,4,3 = 1e6
        W[4, 6:9] = (0.5, 3.0, 5.5)
        W[4, 3:6] = 1e6
    return W


@pytest.mark.parametrize("which", ["L", "R", "LR"])
@pytest.mark.parametrize("ns", [0, 2])
def test_weno_positivity_fallback_reverts_the_side_to_the_cell_values(which, ns):
    plan = _line_plan(ns)
    W = _cliff_line(ns, which)
    cL, cR = 5, 6
    raw_L = np.array([fxo.weno5(*W[v, cL - 2:cL + 3]) for v in range(5 + ns)])
    raw_R = np.array([fxo.weno5(*W[v, cR - 2:cR + 3][::-1]) for v in range(5 + ns)])
    # the data do what they were built for (fxo_weno5 itself is pinned to 40-digit values in test_oracle_routines)
    assert (raw_L[0] <= 0.0) == ("L" in which) and raw_L[4] > 0.0
    assert (raw_R[4] <= 0.0) == ("R" in which) and raw_R[0] > 0.0
    WL, WR, hit = plan.face_states(W, cL)
    assert hit == fxo.STATUS_WENO_FALLBACK
    # [A6]: the failing side's values ALL revert to the cell's own (scalars with them [B11]), bit for bit;
    # the other side keeps the WENO5 values, bit for bit
    assert np.array_equal(WL, W[:, cL] if "L" in which else raw_L)
    assert np.array_equal(WR, W[:, cR] if "R" in which else raw_R)
    # a face two cells away from the cliff is untouched and raises nothing
    WL2, WR2, hit2 = plan.face_states(_cliff_line(ns, ""), cL)
    assert hit2 == 0
    assert np.array_equal(WL2, [fxo.weno5(*_cliff_line(ns, "")[v, cL - 2:cL + 3]) for v in range(5 + ns)])


def test_plm_never_falls_back():
    plan = _line_plan(0, recon=fxo.RECON_PLM_MINMOD)
    WL, WR, hit = plan.face_states(_cliff_line(0, "LR"), 5)
    assert hit == 0 and WL[0] > 0 and WR[4] > 0  # minmod keeps face values between the neighbours


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_weno_fallback_is_reached_inside_advance_and_counted(axis):
    """The same cliffs inside a stage: the status bit and a non-zero count come out of fxo_hydro_advance, and the
    state stays finite (without the fallback the square root of a negative c^2 would poison it)."""
    cfg = inputs.config(4, nb=(2, 2, 2))
    plan, neigh, coords = oracle_plan_for(cfg)
    import torch
    U = inputs.embed(cfg, torch.from_numpy(cliff_state(cfg, coords, axis))).numpy()
    dx = inputs.dx_array(cfg)
    dt = plan.compute_dt(U, dx, 0.1)
    plan.advance(U, dx, dt)
    f, counts = plan.status()
    assert f & fxo.STATUS_WENO_FALLBACK and counts[3] > 0
    assert not (f & fxo.STATUS_NONFINITE)
    assert np.isfinite(plan.interior(U)).all()


# ------------------------------------------------------------------------------------------------ A17 / B1
@pytest.mark.parametrize("solver,speeds", [("hlle", "einfeldt"), ("hlle", "davis"), ("hllc", "einfeldt"), ("hllc", "davis")])
def test_debug_fluxes_sod_interface_and_upwind(solver, speeds):
    """Config 1 at t = 0: every slope is 0, so face f (between zones f-1 and f [A17]) carries F(W_L) for f < 128,
    F(W_R) for f > 128 and the Sod interface flux of tests/golden/sod_interface_flux.txt (40-digit arithmetic) at
    f = 128 -- and nowhere else."""
    gold = {(r[0], r[1]): [float(x) for x in r[2:]] for r in golden_rows("sod_interface_flux.txt")}[(solver, speeds)]
    cfg = inputs.config(1)
    plan, neigh, coords = oracle_plan_for(cfg, riemann=fxo.RIEMANN_HLLE if solver == "hlle" else fxo.RIEMANN_HLLC)
    plan.set_option(fxo.OPT_WAVESPEED, 0 if speeds == "einfeldt" else 1)
    U = inputs.embed(cfg, inputs.block_interiors(cfg, coords)).numpy()
    plan.fill_guardcells(U)
    F = plan.debug_compute_fluxes(U, 0)
    assert F.shape == (5, 1, 1, 1, 257)  # [B1]: n_d + 1 faces along d
    F = F[:, 0, 0, 0, :]
    assert np.array_equal(F[:, :128], np.repeat([[0.0], [1.0], [0.0], [0.0], [0.0]], 128, axis=1))
    assert np.array_equal(F[:, 129:], np.repeat([[0.0], [0.1], [0.0], [0.0], [0.0]], 128, axis=1))
    assert np.allclose(F[[0, 1, 4], 128], gold, rtol=2e-15, atol=0)
    assert F[2, 128] == 0.0 and F[3, 128] == 0.0


@pytest.mark.parametrize("axis", [1, 2])
def test_debug_fluxes_face_index_along_y_and_z(axis):
    """The same line laid along y or z: the flux array's extent grows along that axis only, the interface flux sits at
    index 128 of it, and the normal-momentum flux moves to the momentum component of the axis."""
    gold = {(r[0], r[1]): [float(x) for x in r[2:]] for r in golden_rows("sod_interface_flux.txt")}[("hlle", "einfeldt")]
    plan, U, dx = _sod_along(axis)
    plan.fill_guardcells(U)
    F = plan.debug_compute_fluxes(U, axis)
    want = [1, 1, 1]
    want[2 - axis] = 257
    assert F.shape == (5, 1) + tuple(want)
    F = F.reshape(5, 257)
    assert np.allclose(F[[0, 1 + axis, 4], 128], gold, rtol=2e-15, atol=0)
    others = [v for v in (1, 2, 3) if v != 1 + axis]
    assert not F[others].any()
    assert np.array_equal(F[1 + axis, :128], np.full(128, 1.0)) and np.array_equal(F[1 + axis, 129:], np.full(128, 0.1))


# ------------------------------------------------------------------------------------------------ axis permutation
def _sod_along(axis, riemann=fxo.RIEMANN_HLLE, recon=fxo.RECON_PLM_MINMOD, rk=2):
    dims = [1, 1, 1]
    dims[axis] = 256
    plan = fxo.OraclePlan(tuple(dims), 4, 1, 1.4, recon, riemann, rk)
    neigh = np.full((1, 6), fxo.BC_NONE, np.int32)
    neigh[0, 2 * axis] = neigh[0, 2 * axis + 1] = fxo.BC_OUTFLOW
    plan.set_topology(neigh)
    U = np.full(plan.shape, np.nan)
    x = (np.arange(256) + 0.5) / 256
    rho = np.where(x < 0.5, 1.0, 0.125)
    p = np.where(x < 0.5, 1.0, 0.1)
    shape = [1, 1, 1, 1]
    shape[3 - axis] = 256
    I = plan.interior(U)
    I[0] = rho.reshape(shape)
    I[1:4] = 0.0
    I[4] = (p / (1.4 - 1.0)).reshape(shape)  # as inputs.py forms it
    dx = np.full((1, 3), 1.0 / 256)
    return plan, U, dx


@pytest.mark.parametrize("recon,riemann,rk", [(0, 0, 2), (0, 1, 2), (1, 1, 3)])
def test_sod_along_y_and_z_is_the_x_run_bit_for_bit(recon, riemann, rk):
    """face_flux rotates (u_n, u_t1, u_t2) per direction: a mistake in the rotation or in the way back (a transposed
    component) changes the y or z run.  40 steps, dt from compute_dt each step (it must agree too)."""
    runs = []
    for axis in range(3):
        plan, U, dx = _sod_along(axis, riemann, recon, rk)
        dts = []
        for _ in range(40):
            dts.append(plan.compute_dt(U, dx, 0.8))
            plan.advance(U, dx, dts[-1])
        runs.append((plan.interior(U).reshape(5, 256).copy(), dts))
    X, dts = runs[0]
    assert np.abs(X[1]).max() > 0.1  # the flow did develop
    for axis in (1, 2):
        Y, dty = runs[axis]
        assert dty == dts
        assert np.array_equal(Y[0], X[0]) and np.array_equal(Y[4], X[4])
        assert np.array_equal(Y[1 + axis], X[1])
        for v in (1, 2, 3):
            if v != 1 + axis:
                assert not Y[v].any()


# ------------------------------------------------------------------------------------------------ A7 status bits
def test_status_bits_after_a_floored_advance():
    """A zone below the density floor and a zone whose kinetic energy exceeds E (negative pressure): advance raises
    exactly the two floor bits, counts at least the two zones, leaves the conserved values of untouched far zones
    alone, and the primitives the floors produce are the floor values [A7]."""
    cfg = inputs.config(3, nb=(2, 2, 2))
    plan, neigh, coords = oracle_plan_for(cfg)
    U = inputs.embed(cfg, inputs.block_interiors(cfg, coords)).numpy()
    I = plan.interior(U)
    I[4] = 2.5  # p = 1 everywhere: a quiet gas
    f0, _ = plan.status()
    assert f0 == 0
    dx = inputs.dx_array(cfg)
    plan.advance(U, dx, 1e-4)
    assert plan.status()[0] == 0  # nothing raised on clean data
    I[0, 3, 5, 6, 7] = 1e-14                      # below rho_floor = 1e-12
    I[1, 5, 8, 9, 10] = 10.0                      # m^2 / 2 rho = 50 > E: p < 0 -> p_floor
    W = plan.cons2prim(I[:, 3, 5, 6, 7])
    assert W[0] == 1e-12
    W = plan.cons2prim(I[:, 5, 8, 9, 10])
    assert W[4] == 1e-12
    plan.status_reset()
    plan.advance(U, dx, 1e-9)
    f, counts = plan.status()
    assert f & fxo.STATUS_RHO_FLOOR and f & fxo.STATUS_P_FLOOR
    assert not (f & fxo.STATUS_WENO_FALLBACK)
    assert counts[1] >= 1 and counts[2] >= 1
    plan.status_reset()
    assert plan.status() == (0, [0, 0, 0, 0])
