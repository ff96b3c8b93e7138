"""GPU <-> oracle parity of the fine-coarse boundary services [B12-B14] on static two-level grids: the face guard zones
behind refinement jumps bit for bit (restriction, prolongation), advance to the [NS] tolerances, conservation through the
jumps, uniform state bit for bit."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from tests.helpers import two_level_grid, rel_err
from tests.test_oracle_amr import GAMMA, GRIDS, amr_plan, cons, dx_of, smooth_field, state_from, totals

pytestmark = pytest.mark.gpu


def gpu_amr_plan(grid, dims, g=4, recon=0, riemann=1, rk=2):
    from paper_2208_11630_b200 import binding as fx
    plan = fx.HydroPlan(dims, g, len(grid["level"]), GAMMA, recon, riemann, rk)
    plan.fx_hydro_plan_set_refinement(grid["jump"])
    plan.fx_hydro_plan_set_topology(grid["neigh"])
    plan.fx_hydro_plan_set_workspace()
    assert plan.path == 0
    return plan


class Cfg:
    gamma = GAMMA


@pytest.mark.parametrize("nbc,refined,dims", GRIDS)
@pytest.mark.parametrize("recon,riemann,rk", [(0, 1, 2), (1, 0, 3), (1, 1, 3)])
def test_amr_fill_bitwise_and_advance_parity(nbc, refined, dims, recon, riemann, rk):
    grid = two_level_grid(nbc, refined, dims)
    oplan = amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk)
    gplan = gpu_amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk)
    ndim = sum(1 for d in dims if d > 1)
    L = [nbc[d] * dims[d] for d in range(3)]
    Uo = state_from(oplan, smooth_field(grid, dims, L))
    Ud = torch.from_numpy(Uo).cuda()
    # guard fill: every zone, jump faces included, bit for bit
    F = Uo.copy()
    oplan.fill_guardcells(F)
    Fg = Ud.clone()
    gplan.fx_fill_guardcells(Fg)
    assert np.array_equal(Fg.cpu().numpy(), F)
    assert np.array_equal(gplan.fx_guardcell_index_map().cpu().numpy(), oplan.index_map())
    dx = dx_of(grid)
    dxd = torch.from_numpy(dx).cuda()
    T0 = totals(oplan, grid, Uo, ndim)
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, 0.3)
        dtg = float(gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).item())
        assert abs(dtg - dt) <= 1e-14 * dt
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        if step in (0, 9):
            err = rel_err(Cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
            assert err <= (1e-12 if step == 0 else 1e-9), (step, err)
    got = Ud.cpu().numpy()
    T1 = totals(oplan, grid, got, ndim)
    scale = np.array([T0[0], 2.4 * T0[0], 2.4 * T0[0], 2.4 * T0[0], T0[4]])
    assert np.max(np.abs(T1 - T0) / scale) <= 1e-13
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg == 0


@pytest.mark.parametrize("nbc,refined,dims", GRIDS[1:3])
def test_amr_uniform_state_bitwise_and_step_api(nbc, refined, dims):
    grid = two_level_grid(nbc, refined, dims)
    gplan = gpu_amr_plan(grid, dims)
    n = len(grid["level"])
    shape = (n, dims[2], dims[1], dims[0])
    W = (1.3, 0.4, -0.7, 0.2 if dims[2] > 1 else 0.0, 0.9)
    oplan = amr_plan(grid, dims)
    U = torch.from_numpy(state_from(oplan, cons(*[np.full(shape, x) for x in W]))).cuda()
    U0 = gplan.interior(U).clone()
    dxd = torch.from_numpy(dx_of(grid)).cuda()
    dt = gplan.fx_hydro_compute_dt(U, dxd, 0.3).clone()
    for _ in range(5):
        gplan.fx_hydro_step(U, dxd, 0.3, dt)
    assert torch.equal(gplan.interior(U), U0)


def test_jumps_need_the_refinement_table():
    from paper_2208_11630_b200 import binding as fx
    dims = (8, 8, 8)
    grid = two_level_grid((3, 3, 3), {(1, 1, 1)}, dims)
    plan = fx.HydroPlan(dims, 4, len(grid["level"]), GAMMA, 0, 1, 2)
    with pytest.raises(fx.FxError) as e:
        plan.fx_hydro_plan_set_topology(grid["neigh"])
    assert e.value.code == -3  # FX_ERR_UNSUPPORTED


@pytest.mark.parametrize("nbc,refined,dims", [GRIDS[1], GRIDS[2], ((3, 3, 2), {(0, 0, 0), (2, 2, 1)}, (16, 16, 16))])
@pytest.mark.parametrize("recon,riemann,rk,ns", [(0, 1, 2, 2), (1, 0, 3, 1), (0, 0, 3, 6)])
def test_passive_scalars_through_jumps(nbc, refined, dims, recon, riemann, rk, ns):
    """Passive mass scalars on a two-level grid [B11 with B12-B14] (generic path; fused kernel + scalar pass for 16^3 PLM): guard fill of all variables bit for bit,
    advance to the [NS] tolerances, the scalars' fluxes corrected at the jumps (scalar mass conserved), hydro variables those
    of the plan without scalars (bit for bit with PLM + HLLC)."""
    from paper_2208_11630_b200 import binding as fx
    from tests.test_oracle_amr import amr_zone_centres, with_scalars
    grid = two_level_grid(nbc, refined, dims)
    n = len(grid["level"])
    oplan = amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk, nvars=5 + ns)

    def gplan_for(nvars, path=None):
        plan = fx.HydroPlan(dims, 4, n, GAMMA, recon, riemann, rk, nvars=nvars)
        if path is not None:
            plan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
        plan.fx_hydro_plan_set_refinement(grid["jump"])
        plan.fx_hydro_plan_set_topology(grid["neigh"])
        plan.fx_hydro_plan_set_workspace()
        return plan

    gplan, g5 = gplan_for(5 + ns), gplan_for(5, path=1)
    # 16 x 16 x nz blocks with PLM: the fused kernel with the scalar pass behind it (path 5); else the generic path
    fused = dims == (16, 16, 16) and recon == 0
    assert gplan.path == (5 if fused else 0) and g5.path == 0
    ndim = sum(1 for d in dims if d > 1)
    L = [nbc[d] * dims[d] for d in range(3)]
    f5 = smooth_field(grid, dims, L)
    X = amr_zone_centres(grid, dims)
    ab = [0.5 + 0.4 * np.sin(2 * np.pi * (s + 1) * X[:, s % ndim] / L[s % ndim] + 0.3 * s) for s in range(ns)]
    ab[0] = (np.abs(X[:, 1] - 0.5 * L[1]) < 0.2 * L[1]).astype(float)  # a slab that crosses the refined region
    Uo = state_from(oplan, with_scalars(f5, ab))
    Ud = torch.from_numpy(Uo).cuda()
    U5 = torch.from_numpy(np.ascontiguousarray(Uo[:5])).cuda()
    F = Uo.copy()
    oplan.fill_guardcells(F)
    Fg = Ud.clone()
    gplan.fx_fill_guardcells(Fg)
    assert np.array_equal(Fg.cpu().numpy(), F)
    dx = dx_of(grid)
    dxd = torch.from_numpy(dx).cuda()
    T0 = totals(oplan, grid, Uo, ndim)
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, 0.3)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        g5.fx_hydro_advance(U5, dxd, dt)
        if step in (0, 9):
            got, ref = gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)
            tol = 1e-12 if step == 0 else 1e-9
            assert rel_err(Cfg, got[:5], ref[:5]) <= tol
            assert float((np.abs(got[5:] - ref[5:]) / ref[0]).max()) <= tol
    if recon == 0 and riemann == 1 and not fused:
        assert torch.equal(gplan.interior(Ud)[:5], g5.interior(U5))
    else:  # (WENO5, HLLE: the kernel variant with scalars contracts some products differently -- rounding, not bits)
        assert rel_err(Cfg, gplan.interior(Ud)[:5].cpu().numpy(), g5.interior(U5).cpu().numpy()) <= 1e-12
    T1 = totals(oplan, grid, Ud.cpu().numpy(), ndim)
    for v in [0, 4] + list(range(5, 5 + ns)):
        assert abs(T1[v] - T0[v]) <= 1e-13 * T0[0], (v, T1[v] - T0[v])
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg == 0
