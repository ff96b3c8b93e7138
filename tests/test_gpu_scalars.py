"""GPU <-> oracle parity of the passive mass scalars (reading B11; run on the B200 box: pytest -m gpu).
Tolerances as for the hydro variables [NS]: <= 1e-12 after one RK step, <= 1e-9 after 10 steps; the error of a
scalar zone is |d(rho X_s)| / rho with the oracle's density (X_s is of order one), the hydro variables keep the
metric A21.  Guard-cell fill of all nvars variables bit-exact."""
import numpy as np
import pytest
import torch

from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for, oracle_plan_for, rel_err

pytestmark = pytest.mark.gpu

TOL_1, TOL_10 = 1e-12, 1e-9


def setup(number, nb, ns, **kw):
    cfg = inputs.config(number, nb=nb)
    oplan, neigh, coords = oracle_plan_for(cfg, nvars=5 + ns, **kw)
    gplan, gneigh, gcoords = gpu_plan_for(cfg, nvars=5 + ns, **kw)
    assert np.array_equal(neigh, gneigh) and np.array_equal(coords, gcoords)
    Ui = inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), ns)
    return cfg, oplan, gplan, inputs.embed(cfg, Ui), inputs.dx_array(cfg)


def scalar_err(got, ref):
    """got / ref: interiors [5 + ns, ...]."""
    if not np.all(np.isfinite(got)):
        return float("inf")
    return float((np.abs(got[5:] - ref[5:]) / ref[0]).max())


CASES = [  # number, nb, ns, kwargs
    (1, None, 2, {}), (2, None, 3, {}), (3, (2, 2, 2), 1, {}), (4, (2, 2, 2), 2, {}), (5, (3, 3, 3), 4, {}),
    (5, (2, 2, 2), 2, dict(riemann=0, rk=3)), (5, (2, 2, 2), 3, dict(recon=1, riemann=0)),
    (2, (3, 2, 1), 2, dict(recon=1, rk=3)), (5, (2, 2, 2), 2, dict(bc="outflow")),
    (5, (2, 2, 2), 2, dict(bc="reflect")), (2, (2, 2, 1), 27, dict(bc="reflect", riemann=0)),
    (1, None, 1, dict(bc="reflect", riemann=1)),
]


@pytest.mark.parametrize("number,nb,ns,kw", CASES)
def test_advance_1_and_10_steps(number, nb, ns, kw):
    cfg, oplan, gplan, Uh, dx = setup(number, nb, ns, **kw)
    # scalars follow the fused kernel in the scalar pass where it applies (3-D 16 x 16 blocks, PLM, same-level neighbours on
    # every face), else they ride on the generic path
    fused = cfg.block_dims == (16, 16, 16) and kw.get("recon", cfg.recon) == 0  # (physical boundaries included)
    assert gplan.path == (1 if fused else 0)
    Uo = Uh.numpy().copy()
    Ud = Uh.cuda()
    dxd = torch.from_numpy(dx).cuda()
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, cfg.cfl)
        if step == 0:
            dt_g = float(gplan.fx_hydro_compute_dt(Ud, dxd, cfg.cfl).item())
            assert abs(dt_g - dt) <= 1e-14 * dt
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        if step in (0, 9):
            got, ref = gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)
            tol = TOL_1 if step == 0 else TOL_10
            assert rel_err(cfg, got[:5], ref[:5]) <= tol
            assert scalar_err(got, ref) <= tol, (step, scalar_err(got, ref))
    assert not np.array_equal(oplan.interior(Uo)[5:], gplan.interior(Uh).numpy()[5:])  # the scalars moved
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg, (fo, fg)


def test_hydro_variables_do_not_see_the_scalars_and_paths_agree():
    """The hydro variables of a run with scalars are bit for bit those of the same path without them (generic path; fused
    kernel + scalar pass), the two paths agree within rounding, and so do their scalars."""
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 2), 3)
    gs, _, _ = gpu_plan_for(cfg, nvars=8, path=1)
    g5, _, _ = gpu_plan_for(cfg, path=1)
    gf, _, _ = gpu_plan_for(cfg)
    assert gplan.path == 1 and gs.path == 0 and g5.path == 0 and gf.path == 1
    dxd = torch.from_numpy(dx).cuda()
    A, S, B, C = Uh.cuda(), Uh.cuda(), Uh[:5].contiguous().cuda(), Uh[:5].contiguous().cuda()
    for _ in range(3):
        dt = float(g5.fx_hydro_compute_dt(B, dxd, cfg.cfl).item())
        gplan.fx_hydro_advance(A, dxd, dt)
        gs.fx_hydro_advance(S, dxd, dt)
        g5.fx_hydro_advance(B, dxd, dt)
        gf.fx_hydro_advance(C, dxd, dt)
    assert torch.equal(gs.interior(S)[:5], g5.interior(B))
    assert torch.equal(gplan.interior(A)[:5], gf.interior(C))
    assert rel_err(cfg, gf.interior(C).cpu().numpy(), g5.interior(B).cpu().numpy()) <= 1e-12
    assert scalar_err(gplan.interior(A).cpu().numpy(), gs.interior(S).cpu().numpy()) <= 1e-12


@pytest.mark.parametrize("dims,g,nb,bc", [((6, 4, 5), 3, (2, 1, 2), "reflect"), ((16, 16, 16), 4, (2, 2, 1), "periodic"),
                                          ((12, 1, 1), 4, (2, 1, 1), "outflow"), ((7, 6, 1), 3, (2, 2, 1), "reflect")])
def test_guard_fill_of_all_variables_bit_exact(dims, g, nb, bc):
    cfg = inputs.config(3)
    cfg.block_dims, cfg.nguard, cfg.nb, cfg.bc = dims, g, nb, bc
    oplan, neigh, coords = oracle_plan_for(cfg, nvars=8)
    gplan, _, _ = gpu_plan_for(cfg, nvars=8)
    rng = np.random.default_rng(7)
    Uh = np.full(oplan.shape, np.nan)
    oplan.interior(Uh)[...] = rng.normal(size=oplan.interior(Uh).shape)
    Ud = torch.from_numpy(Uh).cuda()
    oplan.fill_guardcells(Uh)
    gplan.fx_fill_guardcells(Ud)
    assert np.array_equal(Ud.cpu().numpy(), Uh)
    assert not np.isnan(Uh).any()


@pytest.mark.parametrize("number,nb,recon,riemann", [(2, (2, 2, 1), 0, 1), (5, (2, 2, 2), 1, 1), (4, (2, 2, 2), 1, 0),
                                                     (5, (2, 2, 2), 0, 0)])
def test_debug_fluxes(number, nb, recon, riemann):
    cfg, oplan, gplan, Uh, dx = setup(number, nb, 3, recon=recon, riemann=riemann)
    Un = Uh.numpy().copy()
    oplan.fill_guardcells(Un)
    Ud = torch.from_numpy(Un).cuda()
    for d in range(3):
        if cfg.block_dims[d] == 1:
            continue
        Fo = oplan.debug_compute_fluxes(Un, d)
        Fg = gplan.fx_debug_compute_fluxes(Ud, d).cpu().numpy()
        assert Fg.shape == Fo.shape and Fo.shape[0] == 8
        # rounding scale of an advected flux: density times the fastest signal speed
        W = oplan.interior(Un)
        scale = float((np.abs(W[1:4]).sum(axis=0) + np.sqrt(cfg.gamma * W[0] * W[4])).max())
        assert np.all(np.abs(Fg[5:] - Fo[5:]) <= 1e-13 * scale)
        assert np.abs(Fo[5:]).max() > 0


def test_host_interior_call_carries_the_scalars():
    """fx_hydro_advance_host_interior with nvars = 7: the packed host buffer holds all seven variables."""
    cfg, oplan, gplan, Uh, dx = setup(2, (2, 2, 1), 2)
    Uo = Uh.numpy().copy()
    nsteps = 3
    for _ in range(nsteps):
        oplan.advance(Uo, dx, oplan.compute_dt(Uo, dx, cfg.cfl))
    Uint = gplan.interior(Uh).contiguous().pin_memory()
    U_stage = gplan.alloc_state()
    packed = torch.empty(gplan.interior_shape, dtype=torch.float64, device="cuda")
    dx_stage = torch.empty((gplan.nblocks, 3), dtype=torch.float64, device="cuda")
    gplan.fx_hydro_advance_host_interior(Uint, torch.from_numpy(dx), cfg.cfl, nsteps, U_stage, packed, dx_stage)
    got, ref = Uint.numpy(), oplan.interior(Uo)
    assert rel_err(cfg, got[:5], ref[:5]) <= 1e-11 and scalar_err(got, ref) <= 1e-11


@pytest.mark.parametrize("nz,g,ns,riemann,rk", [(2, 2, 3, 1, 2), (3, 2, 6, 1, 3), (4, 4, 5, 0, 2), (8, 4, 7, 1, 2), (16, 4, 9, 0, 3)])
def test_scalar_march_block_heights_and_scalar_counts(nz, g, ns, riemann, rk):
    """The marching scalar pass on blocks of 16 x 16 x nz zones, down to the two planes its prefetch distance allows (the
    window's new cell is then always the block above's), with every launch shape: 1 to 4 scalars per launch, several
    launches per stage, HLLC (F_rho alone handed over) and HLLE (F_rho and Aq)."""
    cfg = inputs.config(5, nb=(2, 2, 3))
    cfg.block_dims, cfg.nguard = (16, 16, nz), g
    kw = dict(riemann=riemann, rk=rk)
    oplan, neigh, coords = oracle_plan_for(cfg, nvars=5 + ns, **kw)
    gplan, _, _ = gpu_plan_for(cfg, nvars=5 + ns, **kw)
    assert gplan.path == 1
    Uh = inputs.embed(cfg, inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), ns))
    rng = np.random.default_rng(7 + nz)
    dx = inputs.dx_array(cfg) * (1.0 + 0.2 * rng.random((12, 1)))  # a different zone width per block
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    for step in range(3):
        dt = oplan.compute_dt(Uo, dx, cfg.cfl)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        got, ref = gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)
        tol = TOL_1 * (1 + 2 * step)
        assert rel_err(cfg, got[:5], ref[:5]) <= tol and scalar_err(got, ref) <= tol, (step, rel_err(cfg, got[:5], ref[:5]), scalar_err(got, ref))
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg


@pytest.mark.parametrize("riemann,rk", [(1, 2), (0, 3)])
def test_scalars_in_a_closed_box_with_gravity_on_the_fused_path(riemann, rk):
    """Reflecting walls on every face and a constant gravity, with three scalars: the fused kernel's EXTRAS + SCAL variant and
    the marching pass with its mirrored halo cells and the walls' high faces taken from the 17th-face solves [B9, B10, B11]."""
    from oracle import fxoracle as fxo
    from paper_2208_11630_b200 import binding as fx
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 2), 3, bc="reflect", riemann=riemann, rk=rk)
    grav = (0.4, -0.3, 0.6)
    for d in range(3):
        oplan.set_option(fxo.OPT_GRAVITY_X + d, grav[d])
    # (options go in before the topology: a fresh plan)
    gplan = fx.HydroPlan(cfg.block_dims, cfg.nguard, 8, cfg.gamma, cfg.recon, riemann, rk, nvars=8)
    for d in range(3):
        gplan.fx_hydro_plan_set_option(fx.OPT_GRAVITY_X + d, grav[d])
    bcs = [fx.TOPO_REFLECT] * 3
    neigh, _ = fx.fx_topology_cartesian((2, 2, 2), bcs, bcs, fx.ORDER_LEX)
    gplan.fx_hydro_plan_set_topology(neigh)
    gplan.fx_hydro_plan_set_workspace()
    assert gplan.path == 1
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    T0 = [float(gplan.interior(Ud)[v].sum(dtype=torch.float64)) for v in (0, 5, 6, 7)]
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, cfg.cfl)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        if step in (0, 9):
            got, ref = gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)
            tol = TOL_1 if step == 0 else TOL_10
            assert rel_err(cfg, got[:5], ref[:5]) <= tol and scalar_err(got, ref) <= tol, (step, rel_err(cfg, got[:5], ref[:5]), scalar_err(got, ref))
    T1 = [float(gplan.interior(Ud)[v].sum(dtype=torch.float64)) for v in (0, 5, 6, 7)]
    for a, b in zip(T0, T1):  # nothing leaves a closed box
        assert abs(a - b) <= 1e-13 * T0[0]
