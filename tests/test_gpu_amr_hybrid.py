"""Refinement jumps with 16 x 16 x nz blocks on the fused path (fx_hydro_plan_path = 5): the fused TMA kernel advances every
block -- those whose faces all have same-level neighbours or physical boundaries in chains, those that have a jump face as
segments of their own, reading their interpolated guard zones behind the jump and storing the jump faces' fluxes --, then
the flux correction.  Checked against the oracle on static two-level grids
(<= 1e-12 after one step, <= 1e-9 after ten [NS]), for conservation through the jumps, against the all-generic path, and
for bitwise independence of the chain length."""
import numpy as np
import pytest
import torch

from tests.helpers import two_level_grid, rel_err
from tests.test_oracle_amr import GAMMA, amr_plan, cons, dx_of, smooth_field, state_from, totals

pytestmark = pytest.mark.gpu

DIMS = (16, 16, 16)
CENTRE2 = {(x, y, z) for x in (1, 2) for y in (1, 2) for z in (1, 2)}
GRIDS16 = [((5, 5, 5), {(2, 2, 2)}, True), ((4, 4, 4), CENTRE2, True), ((4, 4, 3), {(0, 0, 0), (1, 0, 0), (3, 3, 2)}, False)]


class Cfg:
    gamma = GAMMA


def gpu_plan(grid, recon=0, riemann=1, rk=2, path=None, zchain=None, dims=DIMS, guard_x=None):
    from paper_2208_11630_b200 import binding as fx
    plan = fx.HydroPlan(dims, 4, len(grid["level"]), GAMMA, recon, riemann, rk)
    if guard_x is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
    if path is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
    if zchain is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_ZCHAIN, zchain)
    plan.fx_hydro_plan_set_refinement(grid["jump"])
    plan.fx_hydro_plan_set_topology(grid["neigh"])
    plan.fx_hydro_plan_set_workspace()
    return plan


@pytest.mark.parametrize("nbc,refined,periodic", GRIDS16)
@pytest.mark.parametrize("recon,riemann,rk", [(0, 1, 2), (1, 1, 3), (0, 0, 3)])
def test_hybrid_parity_conservation_and_generic(nbc, refined, periodic, recon, riemann, rk):
    grid = two_level_grid(nbc, refined, DIMS, periodic=periodic)
    oplan = amr_plan(grid, DIMS, recon=recon, riemann=riemann, rk=rk)
    gplan = gpu_plan(grid, recon, riemann, rk)
    ggen = gpu_plan(grid, recon, riemann, rk, path=1)
    assert gplan.path == 5 and ggen.path == 0
    L = [nbc[d] * DIMS[d] for d in range(3)]
    Uo = state_from(oplan, smooth_field(grid, DIMS, L))
    Ud, Ug = torch.from_numpy(Uo).cuda(), torch.from_numpy(Uo).cuda()
    dx = dx_of(grid)
    dxd = torch.from_numpy(dx).cuda()
    T0 = totals(oplan, grid, Uo, 3)
    dts = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
    Us = Ud.clone()
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, 0.3)
        dtg = float(gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).item())
        assert abs(dtg - dt) <= 1e-13 * dt
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        ggen.fx_hydro_advance(Ug, dxd, dt)
        if step < 3:  # fx_hydro_step: same states with the time step kept on the device (the reduction fused but for the corrected blocks)
            assert abs(float(dts.item()) - dt) <= 1e-12 * dt
            gplan.fx_hydro_step(Us, dxd, 0.3, dts)
        if step in (0, 9):
            err = rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
            assert err <= (1e-12 if step == 0 else 1e-9), (step, err)
            assert rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), ggen.interior(Ug).cpu().numpy()) <= (1e-12 if step == 0 else 1e-9)
    if periodic:  # what leaves the fine blocks enters the coarse ones, whichever kernel advanced either
        T1 = totals(oplan, grid, Ud.cpu().numpy(), 3)
        scale = np.array([T0[0], 2.4 * T0[0], 2.4 * T0[0], 2.4 * T0[0], T0[4]])
        assert np.max(np.abs(T1 - T0) / scale) <= 1e-13
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg == 0


def test_hybrid_uniform_state_bitwise_and_chain_length():
    grid = two_level_grid((4, 4, 4), CENTRE2, DIMS)
    n = len(grid["level"])
    shape = (n,) + DIMS
    oplan = amr_plan(grid, DIMS)
    dxd = torch.from_numpy(dx_of(grid)).cuda()
    W = (1.3, 0.4, -0.7, 0.2, 0.9)
    Uu = state_from(oplan, cons(*[np.full(shape, x) for x in W]))
    L = [4 * 16] * 3
    Usm = state_from(oplan, smooth_field(grid, DIMS, L))
    results = []
    for zc in (None, 1, 3, 8):
        gplan = gpu_plan(grid, zchain=zc)
        assert gplan.path == 5
        U = torch.from_numpy(Uu).cuda()
        U0 = gplan.interior(U).clone()
        dt = gplan.fx_hydro_compute_dt(U, dxd, 0.3).clone()
        for _ in range(4):
            gplan.fx_hydro_step(U, dxd, 0.3, dt)
        assert torch.equal(gplan.interior(U), U0)
        V = torch.from_numpy(Usm).cuda()
        dt = gplan.fx_hydro_compute_dt(V, dxd, 0.3).clone()
        for _ in range(4):
            gplan.fx_hydro_step(V, dxd, 0.3, dt)
        results.append(gplan.interior(V).clone())
    for r in results[1:]:
        assert torch.equal(r, results[0])


def test_a_grid_whose_every_block_has_a_jump_face():
    """Every block touches a jump: every segment of the fused kernel is a single block that reads its own guard zones."""
    grid = two_level_grid((2, 1, 1), {(0, 0, 0)}, DIMS)  # the coarse block sees the refined one through both x faces
    gplan = gpu_plan(grid)
    assert gplan.path == 5
    oplan = amr_plan(grid, DIMS)
    Uo = state_from(oplan, smooth_field(grid, DIMS, [32, 16, 16]))
    Ud = torch.from_numpy(Uo).cuda()
    dx = dx_of(grid)
    dt = oplan.compute_dt(Uo, dx, 0.3)
    oplan.advance(Uo, dx, dt)
    gplan.fx_hydro_advance(Ud, torch.from_numpy(dx).cuda(), dt)
    assert rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-12


@pytest.mark.parametrize("nbc,refined,periodic", GRIDS16[1:])
@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_wide_layout_gives_the_same_bits(nbc, refined, periodic, recon, rk):
    """FX_OPT_GUARD_X = 8 (256-byte row pitch, the layout bench.py runs): a block's own guard zones behind a jump then start
    8 zones into a row; three steps equal the compact layout's bit for bit."""
    grid = two_level_grid(nbc, refined, DIMS, periodic=periodic)
    oplan = amr_plan(grid, DIMS, recon=recon, rk=rk)
    L = [nbc[d] * DIMS[d] for d in range(3)]
    Uo = state_from(oplan, smooth_field(grid, DIMS, L))
    ga, gb = gpu_plan(grid, recon, 1, rk), gpu_plan(grid, recon, 1, rk, guard_x=8)
    assert ga.path == 5 and gb.path == 5 and gb.gd == (8, 4, 4)
    A = torch.from_numpy(Uo).cuda()
    B = gb.embed(np.ascontiguousarray(oplan.interior(Uo)))
    dxd = torch.from_numpy(dx_of(grid)).cuda()
    dta, dtb = ga.fx_hydro_compute_dt(A, dxd, 0.3).clone(), gb.fx_hydro_compute_dt(B, dxd, 0.3).clone()
    for _ in range(3):
        ga.fx_hydro_step(A, dxd, 0.3, dta)
        gb.fx_hydro_step(B, dxd, 0.3, dtb)
    assert torch.equal(dta, dtb) and torch.equal(ga.interior(A), gb.interior(B))


@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_jumps_next_to_walls_with_gravity(recon, rk):
    """Everything the kernel's EXTRAS variant carries at once: refinement jumps on blocks in the corners of a box with
    reflecting walls, and a constant gravity [B9, B10, B12-B14], against the oracle and the all-generic path."""
    from oracle import fxoracle as fxo
    from paper_2208_11630_b200 import binding as fx
    nbc = (4, 4, 3)
    grid = two_level_grid(nbc, {(0, 0, 0), (1, 0, 0), (3, 3, 2)}, DIMS, periodic=False)
    grid["neigh"] = np.where(grid["neigh"] == fxo.BC_OUTFLOW, fxo.BC_REFLECT, grid["neigh"]).astype(np.int32)
    assert fxo.BC_REFLECT == fx.BC_REFLECT and (grid["neigh"] == fx.BC_REFLECT).any()
    grav = (0.3, -0.2, 0.5)

    def gplan_with_gravity(path=None):
        plan = fx.HydroPlan(DIMS, 4, len(grid["level"]), GAMMA, recon, 1, rk)
        if path is not None:
            plan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
        for d in range(3):
            plan.fx_hydro_plan_set_option(fx.OPT_GRAVITY_X + d, grav[d])
        plan.fx_hydro_plan_set_refinement(grid["jump"])
        plan.fx_hydro_plan_set_topology(grid["neigh"])
        plan.fx_hydro_plan_set_workspace()
        return plan

    oplan = amr_plan(grid, DIMS, recon=recon, rk=rk)
    for d in range(3):
        oplan.set_option(fxo.OPT_GRAVITY_X + d, grav[d])
    gplan, ggen = gplan_with_gravity(), gplan_with_gravity(path=1)
    assert gplan.path == 5 and ggen.path == 0
    Uo = state_from(oplan, smooth_field(grid, DIMS, [nbc[d] * DIMS[d] for d in range(3)]))
    Ud, Ug = torch.from_numpy(Uo).cuda(), torch.from_numpy(Uo).cuda()
    dx = dx_of(grid)
    dxd = torch.from_numpy(dx).cuda()
    for step in range(4):
        dt = oplan.compute_dt(Uo, dx, 0.3)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        ggen.fx_hydro_advance(Ug, dxd, dt)
        tol = 1e-12 * (1 + 3 * step)
        assert rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= tol
        assert rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), ggen.interior(Ug).cpu().numpy()) <= tol
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg == 0


@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_step_time_step_wherever_the_fastest_zone_sits(recon, rk):
    """fx_hydro_step on the fused path forms the next time step in two pieces: the last stage kernel's own reduction over the
    blocks the flux correction leaves alone, then a pass over the corrected blocks (those with a finer neighbour).  With the
    fastest zone (a hot block) put in a corrected block, in a fine block behind a jump, or far from any jump, the step's dt
    equals fx_hydro_compute_dt of the state it produced and the oracle's [B7, B14]."""
    from paper_2208_11630_b200.binding import NEIGH_FINER, NEIGH_COARSER
    grid = two_level_grid((4, 4, 4), CENTRE2, DIMS)
    neigh = np.asarray(grid["neigh"]).reshape(-1, 6)
    corrected = [b for b in range(len(neigh)) if (neigh[b] == NEIGH_FINER).any()]
    fine = [b for b in range(len(neigh)) if (neigh[b] == NEIGH_COARSER).any()]
    plain = [b for b in range(len(neigh)) if b not in corrected and b not in fine]
    assert corrected and fine and plain
    oplan = amr_plan(grid, DIMS, recon=recon, rk=rk)
    gplan = gpu_plan(grid, recon, 1, rk)
    assert gplan.path == 5
    dx = dx_of(grid)
    dxd = torch.from_numpy(dx).cuda()
    prim = smooth_field(grid, DIMS, [64, 64, 64])
    seen = []
    for hot in (corrected[0], corrected[-1], fine[0], plain[0], plain[-1]):
        Uo = state_from(oplan, prim)
        Io = oplan.interior(Uo)
        Io[4, hot] *= 6.0  # total energy: a hot block, the largest sound speed by far
        Ud = torch.from_numpy(Uo).cuda()
        dts = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
        dt = oplan.compute_dt(Uo, dx, 0.3)
        assert abs(float(dts.item()) - dt) <= 1e-13 * dt
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_step(Ud, dxd, 0.3, dts)
        after = float(gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).item())
        assert abs(float(dts.item()) - after) <= 1e-14 * after, (hot, float(dts.item()), after)
        dto = oplan.compute_dt(Uo, dx, 0.3)
        assert abs(float(dts.item()) - dto) <= 1e-12 * dto
        seen.append(after)
    assert len({round(s / seen[0], 6) for s in seen}) > 1  # (the fastest zone really moved with the hot block)
