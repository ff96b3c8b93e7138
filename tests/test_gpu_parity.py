"""GPU <-> oracle parity through the C ABI (run on the B200 box: pytest -m gpu).
Tolerances [NS]: interior zones <= 1e-12 after one RK step, <= 1e-9 after 10 steps (metric A21);
dt <= 1e-14 relative; guard-cell index maps and filled guard data bit-exact."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for, oracle_plan_for, rel_err

pytestmark = pytest.mark.gpu

TOL_1, TOL_10, TOL_DT = 1e-12, 1e-9, 1e-14


def setup(number, nb=None, path=None, **kw):
    cfg = inputs.config(number, nb=nb)
    oplan, neigh, coords = oracle_plan_for(cfg, **kw)
    gplan, gneigh, gcoords = gpu_plan_for(cfg, path=path, **kw)
    assert np.array_equal(neigh, gneigh) and np.array_equal(coords, gcoords)
    Uh = inputs.embed(cfg, inputs.block_interiors(cfg, coords))
    return cfg, oplan, gplan, Uh, inputs.dx_array(cfg)


GUARD_CASES = [
    ((4, 4, 4), 2, (2, 2, 2), "periodic", 0), ((4, 4, 4), 4, (2, 2, 2), "periodic", 1),
    ((6, 4, 5), 3, (3, 1, 2), "outflow", 0), ((8, 6, 1), 3, (2, 3, 1), "periodic", 0),
    ((12, 1, 1), 4, (3, 1, 1), "outflow", 0), ((12, 1, 1), 4, (1, 1, 1), "periodic", 0),
    ((16, 16, 16), 4, (3, 2, 2), "periodic", 1), ((16, 16, 1), 4, (8, 8, 1), "periodic", 0),
    ((256, 1, 1), 4, (1, 1, 1), "outflow", 0),
    ((6, 4, 5), 3, (2, 1, 2), "reflect", 0), ((16, 16, 16), 4, (2, 2, 1), "reflect", 1), ((12, 1, 1), 4, (2, 1, 1), "reflect", 0),
]


@pytest.mark.parametrize("dims,g,nb,bc,order", GUARD_CASES)
def test_guard_index_map_and_fill_bit_exact(dims, g, nb, bc, order):
    cfg = inputs.config(3)
    cfg.block_dims, cfg.nguard, cfg.nb, cfg.bc = dims, g, nb, bc
    oplan, neigh, coords = oracle_plan_for(cfg, order=order)
    gplan, _, _ = gpu_plan_for(cfg, order=order)
    assert np.array_equal(gplan.fx_guardcell_index_map().cpu().numpy(), oplan.index_map())
    if gplan.nblocks > 2:
        assert np.array_equal(gplan.fx_guardcell_index_map(1, 2).cpu().numpy(), oplan.index_map(1, 2))
    rng = np.random.default_rng(42)
    Uh = np.full(oplan.shape, np.nan)
    oplan.interior(Uh)[...] = rng.normal(size=oplan.interior(Uh).shape)
    Ud = torch.from_numpy(Uh).cuda()
    oplan.fill_guardcells(Uh)
    gplan.fx_fill_guardcells(Ud)
    assert np.array_equal(Ud.cpu().numpy(), Uh)  # every zone, bit for bit (no NaN left)
    assert not np.isnan(Uh).any()


@pytest.mark.parametrize("number,nb", [(1, None), (2, None), (3, (4, 4, 4)), (4, (3, 3, 3)), (5, (3, 3, 3))])
def test_compute_dt(number, nb):
    cfg, oplan, gplan, Uh, dx = setup(number, nb)
    dt_o = oplan.compute_dt(Uh.numpy(), dx, cfg.cfl)
    dt_g = float(gplan.fx_hydro_compute_dt(Uh.cuda(), torch.from_numpy(dx).cuda(), cfg.cfl).item())
    assert abs(dt_g - dt_o) <= TOL_DT * dt_o
    # twice in a row: the scratch word re-arms itself
    dt_g2 = float(gplan.fx_hydro_compute_dt(Uh.cuda(), torch.from_numpy(dx).cuda(), cfg.cfl).item())
    assert dt_g2 == dt_g


def test_compute_dt_uniform_state_closed_form_and_per_block_dx():
    cfg = inputs.config(3, nb=(2, 2, 2))
    oplan, neigh, coords = oracle_plan_for(cfg)
    gplan, _, _ = gpu_plan_for(cfg)
    W = (0.5, 0.3, -1.1, 0.4, 0.8)
    E = W[4] / 0.4 + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)
    U = np.full(oplan.shape, np.nan)
    for v, val in enumerate((W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3], E)):
        oplan.interior(U)[v] = val
    dx = np.random.default_rng(0).uniform(0.01, 0.1, size=(8, 3))
    dt_o = oplan.compute_dt(U, dx, 0.3)
    dt_g = float(gplan.fx_hydro_compute_dt(torch.from_numpy(U).cuda(), torch.from_numpy(dx).cuda(), 0.3).item())
    assert abs(dt_g - dt_o) <= TOL_DT * dt_o


@pytest.mark.parametrize("number,nb,recon,riemann", [(2, (2, 2, 1), 0, 1), (3, (2, 2, 2), 0, 1), (3, (2, 2, 2), 0, 0),
                                                     (5, (2, 2, 2), 1, 1), (4, (2, 2, 2), 1, 0), (1, None, 0, 0)])
def test_debug_fluxes(number, nb, recon, riemann):
    cfg, oplan, gplan, Uh, dx = setup(number, nb, recon=recon, riemann=riemann)
    Un = Uh.numpy().copy()
    oplan.fill_guardcells(Un)
    Ud = torch.from_numpy(Un).cuda()
    for d in range(3):
        if cfg.block_dims[d] == 1:
            continue
        Fo = oplan.debug_compute_fluxes(Un, d)
        Fg = gplan.fx_debug_compute_fluxes(Ud, d).cpu().numpy()
        scale = np.abs(Fo).max(axis=(1, 2, 3, 4), keepdims=True)
        scale[1:4] = scale[1:4].max()
        assert np.all(np.abs(Fg - Fo) <= 1e-13 * scale)  # scale may be 0 (e.g. Sedov mass flux at t = 0): then exact


ADV_CASES = [  # number, nb, kwargs
    (1, None, {}), (2, None, {}), (3, None, {}), (4, (3, 3, 3), {}), (5, (3, 3, 3), {}),
    (3, (2, 2, 2), dict(riemann=0, rk=3)), (5, (2, 2, 2), dict(recon=1, riemann=0, rk=2)),
    (2, (3, 2, 1), dict(recon=1, rk=3)), (5, (2, 2, 2), dict(bc="outflow")),
    (5, (2, 2, 2), dict(bc="reflect")), (5, (1, 1, 3), dict(bc="reflect", recon=1, rk=3)), (2, (2, 2, 1), dict(bc="reflect")),
    (1, None, dict(bc="reflect")),
    # Davis wave speeds [A8] (FX_OPT_WAVESPEED = 1: its own template instantiation) on every path's shape
    (5, (2, 2, 2), dict(wavespeed=1)), (3, (2, 2, 2), dict(wavespeed=1, riemann=0)), (4, (2, 2, 2), dict(wavespeed=1)),
    (2, (3, 2, 1), dict(wavespeed=1)), (1, None, dict(wavespeed=1)),
]


@pytest.mark.parametrize("path", [None, 1])
@pytest.mark.parametrize("number,nb,kw", ADV_CASES)
def test_advance_1_and_10_steps(number, nb, kw, path):
    cfg, oplan, gplan, Uh, dx = setup(number, nb, path=path, **kw)
    if path == 1 and gplan.path == 0 and False:
        pytest.skip()
    Uo = Uh.numpy().copy()
    Ud = Uh.cuda()
    dxd = torch.from_numpy(dx).cuda()
    for step in range(10):
        dt = oplan.compute_dt(Uo, dx, cfg.cfl)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)  # same dt on both sides: the step itself is what is compared
        if step in (0, 9):
            err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
            assert err <= (TOL_1 if step == 0 else TOL_10), (step, err)
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg, (fo, fg)


@pytest.mark.parametrize("dims,path", [((16, 16, 16), None), ((16, 16, 16), 1), ((8, 8, 8), 2), ((8, 8, 8), 1), ((16, 16, 1), None)])
@pytest.mark.parametrize("rk", [2, 3])
def test_weno_positivity_fallback_taken_on_every_path(dims, path, rk):
    """[A6] A field with density and pressure cliffs (tests.helpers.cliff_state; the oracle's branch is pinned on the
    same profile in tests/test_oracle_pins_r2.py) along each axis: the fallback IS taken (non-zero count on both
    sides), the status bits agree, and the states agree to the one-step tolerance on the fused, generic and tile
    kernels.  The reverted side's WENO value is -0.75 against cell values of order 1, so rounding cannot flip the
    decision."""
    from tests.helpers import cliff_state
    ndim = sum(1 for d in dims if d > 1)
    for axis in range(ndim):
        cfg = inputs.config(4, nb=(2, 2, 2) if ndim == 3 else (2, 2, 1))
        cfg.block_dims = dims
        oplan, neigh, coords = oracle_plan_for(cfg, rk=rk)
        gplan, _, _ = gpu_plan_for(cfg, rk=rk, path=path)
        assert gplan.path == {None: (1 if dims == (16, 16, 16) else 2), 1: 0, 2: 2}[path]
        Uh = inputs.embed(cfg, torch.from_numpy(cliff_state(cfg, coords, axis, high=1e3)))
        dx = inputs.dx_array(cfg)
        Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
        dt = oplan.compute_dt(Uo, dx, 0.1)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        fo, co = oplan.status()
        fg, cg = gplan.fx_hydro_status()
        assert fo & fxo.STATUS_WENO_FALLBACK and co[3] > 0 and cg[3] > 0
        assert fo == fg, (fo, fg)
        err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
        assert err <= TOL_1, (axis, err)


@pytest.mark.parametrize("path", [None, 1])
@pytest.mark.parametrize("recon,riemann,rk", [(0, 0, 2), (1, 1, 3)])
def test_sod_along_y_and_z(recon, riemann, rk, path):
    """Config 1 laid along x, y and z (the oracle's three runs are bit for bit the same: tests/test_oracle_pins_r2.py):
    each GPU run matches the oracle's, so the kernels' frame rotation is the oracle's."""
    from paper_2208_11630_b200 import binding as fx
    from tests.test_oracle_pins_r2 import _sod_along
    for axis in range(3):
        oplan, Uo, dx = _sod_along(axis, riemann, recon, rk)
        dims = [1, 1, 1]
        dims[axis] = 256
        neigh = np.full((1, 6), fx.BC_NONE, np.int32)
        neigh[0, 2 * axis] = neigh[0, 2 * axis + 1] = fx.BC_OUTFLOW
        gplan = fx.HydroPlan(tuple(dims), 4, 1, 1.4, recon, riemann, rk)
        if path is not None:
            gplan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
        gplan.fx_hydro_plan_set_topology(neigh)
        gplan.fx_hydro_plan_set_workspace()
        Ud, dxd = torch.from_numpy(Uo).cuda(), torch.from_numpy(dx).cuda()
        cfg = inputs.config(1)
        for step in range(10):
            dt = oplan.compute_dt(Uo, dx, 0.8)
            dtg = float(gplan.fx_hydro_compute_dt(Ud, dxd, 0.8).item())
            assert abs(dtg - dt) <= TOL_DT * dt
            oplan.advance(Uo, dx, dt)
            gplan.fx_hydro_advance(Ud, dxd, dt)
            if step in (0, 9):
                err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
                assert err <= (TOL_1 if step == 0 else TOL_10), (axis, step, err)


@pytest.mark.parametrize("kw", [dict(), dict(riemann=0, rk=3), dict(wavespeed=1), dict(bc="outflow", rk=3)])
def test_pair_variant_of_the_fused_kernel(kw):
    """FX_OPT_PATH = 3: the fused kernel with two zones per thread (csrc/fx_stage_pair.cu; slower, kept for comparison).
    Same parity bar as every path, the fused dt included; uniform state bit for bit; results independent of the chain
    length; with a wall in the table the plan falls back to the default fused kernel."""
    from paper_2208_11630_b200 import binding as fx
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 3), path=3, **kw)
    assert gplan.path == 3
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    dt = gplan.fx_hydro_compute_dt(Ud, dxd, cfg.cfl).clone()
    for step in range(10):
        dto = oplan.compute_dt(Uo, dx, cfg.cfl)
        assert abs(float(dt.item()) - dto) <= 1e-13 * dto
        oplan.advance(Uo, dx, dto)
        gplan.fx_hydro_step(Ud, dxd, cfg.cfl, dt)
        if step in (0, 9):
            err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
            assert err <= (TOL_1 if step == 0 else TOL_10), (step, err)
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg
    # chain length 1 gives the same bits
    g1, _, _ = gpu_plan_for(cfg, path=3, zchain=1, **kw)
    A, B = Uh.cuda(), Uh.cuda()
    for _ in range(2):
        gplan.fx_hydro_advance(A, dxd, 1e-3)
        g1.fx_hydro_advance(B, dxd, 1e-3)
    assert torch.equal(gplan.interior(A), g1.interior(B))
    # uniform state
    U = torch.full(Uh.shape, float("nan"), dtype=torch.float64)
    I = inputs.interior_view(cfg, U)
    for v, val in enumerate((1.3, 0.4, -0.7, 0.2, 5.9485)):
        I[v] = val
    U = U.cuda()
    U0 = gplan.interior(U).clone()
    for _ in range(5):
        gplan.fx_hydro_advance(U, dxd, 0.01)
    assert torch.equal(gplan.interior(U), U0)
    wall, _, _ = gpu_plan_for(cfg, path=3, bc="reflect")
    assert wall.path == 1


@pytest.mark.parametrize("path", [None, 1])
def test_weno5_parity_in_cgs_like_units(path):
    """Large magnitudes: density x 1e7, pressure x 1e25 (velocities then ~ 1e9) -- inside the documented range of the
    kernels' single-division WENO5 weights (include/fx_hydro.h, FX_OPT_WENO_EPS): same tolerances, no fallback, no flag."""
    cfg = inputs.config(4, nb=(2, 2, 2))
    oplan, neigh, coords = oracle_plan_for(cfg)
    gplan, _, _ = gpu_plan_for(cfg, path=path)
    Ui = inputs.block_interiors(cfg, coords).numpy().copy()
    sr, sp = 1e7, 1e25
    sv = np.sqrt(sp / sr)
    Ui[0] *= sr
    Ui[1:4] *= sr * sv
    Ui[4] *= sp
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = inputs.dx_array(cfg)
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    for step in range(3):
        dt = oplan.compute_dt(Uo, dx, cfg.cfl)
        dtg = float(gplan.fx_hydro_compute_dt(Ud, dxd, cfg.cfl).item())
        assert abs(dtg - dt) <= TOL_DT * dt
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-11
    assert oplan.status()[0] == 0 and gplan.fx_hydro_status()[0] == 0


def test_device_dt_path_equals_host_dt_path():
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 2))
    dxd = torch.from_numpy(dx).cuda()
    A, B = Uh.cuda(), Uh.cuda()
    for _ in range(3):
        dt = gplan.fx_hydro_compute_dt(A, dxd, cfg.cfl)
        gplan.fx_hydro_advance(A, dxd, dt)  # device-resident dt
        dth = float(gplan.fx_hydro_compute_dt(B, dxd, cfg.cfl).item())
        gplan.fx_hydro_advance(B, dxd, dth)
    assert torch.equal(gplan.interior(A), gplan.interior(B))


@pytest.mark.parametrize("number,nb,kw", [(5, (2, 2, 2), {}), (4, (2, 2, 2), {}), (3, (2, 2, 2), dict(rk=3, bc="outflow")), (2, None, {})])
def test_step_with_fused_dt_equals_compute_dt_then_advance(number, nb, kw):
    """fx_hydro_step: same state as advance with the same dt (bitwise), and the dt it leaves behind is the CFL step of
    the advanced state (<= 1e-14 relative to the oracle's, and to the library's own reduction pass)."""
    cfg, oplan, gplan, Uh, dx = setup(number, nb, **kw)
    dxd = torch.from_numpy(dx).cuda()
    A, B = Uh.cuda(), Uh.cuda()
    dt = gplan.fx_hydro_compute_dt(A, dxd, cfg.cfl).clone()
    for _ in range(3):
        dt_used = dt.clone()
        gplan.fx_hydro_step(A, dxd, cfg.cfl, dt)
        gplan.fx_hydro_advance(B, dxd, dt_used)
        assert torch.equal(gplan.interior(A), gplan.interior(B))
        dt_lib = float(gplan.fx_hydro_compute_dt(B, dxd, cfg.cfl).item())
        dt_ora = oplan.compute_dt(B.cpu().numpy(), dx, cfg.cfl)
        assert abs(float(dt.item()) - dt_lib) <= TOL_DT * dt_lib
        assert abs(float(dt.item()) - dt_ora) <= TOL_DT * dt_ora
    fg, _ = gplan.fx_hydro_status()
    assert fg == 0


@pytest.mark.parametrize("nguard,recon,dims", [(2, 0, (16, 16, 16)), (3, 0, (16, 16, 16)), (3, 1, (16, 16, 16)), (4, 0, (16, 16, 6)),
                                               (4, 1, (16, 16, 5))])
def test_fused_kernel_other_guard_depths_and_block_heights(nguard, recon, dims):
    """Guard depths other than 4 and block heights other than 16: the fused kernel where it applies (a TMA box must start
    on a 16-byte boundary, so an odd guard depth goes to the generic path), parity with the oracle either way."""
    for bc in ("periodic", "outflow"):
        cfg = inputs.config(5, nb=(2, 2, 2))
        cfg.nguard, cfg.block_dims = nguard, dims
        oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon)
        gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon)
        assert gplan.path == (1 if nguard % 2 == 0 else 0)
        rng = np.random.default_rng(11)
        shape = (8,) + tuple(reversed(dims))
        rho = 1.0 + 0.3 * rng.random(shape)
        vel = 0.4 * rng.standard_normal((3,) + shape)
        p = 1.0 + 0.3 * rng.random(shape)
        Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], p / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
        Uh = inputs.embed(cfg, torch.from_numpy(Ui))
        dx = np.full((8, 3), 1.0 / 32)
        Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
        for step in range(3):
            dt = oplan.compute_dt(Uo, dx, 0.3)
            oplan.advance(Uo, dx, dt)
            gplan.fx_hydro_advance(Ud, dxd, dt)
        assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-11


@pytest.mark.parametrize("recon,rk,nzb", [(0, 2, 16), (1, 3, 16), (0, 3, 4)])
def test_z_chains_irregular_topology_bitwise_and_parity(recon, rk, nzb):
    """The fused kernel marches one CTA through up to FX_OPT_ZCHAIN z-neighbour blocks.  On a topology whose chains are a
    periodic ring of 5, with one block's +x link cut (outflow on one side only), one z link that is not mutual (the chain
    must break there) and a different dx per block: the result does not depend on the chain length, bit for bit, the
    fused time step neither, and both agree with the oracle on the same neighbour table."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 1, 5))
    cfg.block_dims = (16, 16, nzb)
    per, out = fx.TOPO_PERIODIC, fx.TOPO_OUTFLOW
    neigh, coords = fx.fx_topology_cartesian((2, 1, 5), (out, per, per), (out, per, per), inputs.ORDER_LEX)
    neigh = np.array(neigh, np.int32).copy()
    nbk = neigh.shape[0]
    mid = int(np.flatnonzero((coords[:, 0] == 0) & (coords[:, 2] == 2))[0])
    neigh[mid, 1] = fx.BC_OUTFLOW                       # x = 0 column: block 2 of the chain has no +x neighbour
    a = int(np.flatnonzero((coords[:, 0] == 1) & (coords[:, 2] == 1))[0])
    c = int(np.flatnonzero((coords[:, 0] == 1) & (coords[:, 2] == 3))[0])
    neigh[a, 5] = c                                     # x = 1 column: block 1 sees block 3 above it, block 2 still names 1 below
    neigh[c, 2] = fx.BC_OUTFLOW                         # and block 3 has outflow at -y
    oplan = fxo.OraclePlan(cfg.block_dims, cfg.nguard, nbk, cfg.gamma, recon, cfg.riemann, rk)
    oplan.set_topology(neigh)
    rng = np.random.default_rng(5)
    shape = (nbk, nzb, 16, 16)
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    pr = 1.0 + 0.3 * rng.random(shape)
    Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = rng.uniform(1.0 / 40, 1.0 / 24, size=(nbk, 3))
    Uo = Uh.numpy().copy()
    dts_o = []
    for step in range(2):
        dts_o.append(oplan.compute_dt(Uo, dx, 0.3))
        oplan.advance(Uo, dx, dts_o[-1])
    dts_o.append(oplan.compute_dt(Uo, dx, 0.3))
    results = []
    for zc in (1, 2, 3, 8):
        gplan, _, _ = gpu_plan_for(cfg, recon=recon, rk=rk, neigh=neigh, zchain=zc)
        assert gplan.path == 1
        Ud, dxd = Uh.cuda(), torch.from_numpy(dx).cuda()
        dt = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
        dts = [float(dt.item())]
        for step in range(2):
            gplan.fx_hydro_step(Ud, dxd, 0.3, dt)
            dts.append(float(dt.item()))
        results.append((gplan.interior(Ud).cpu().numpy(), dts))
    for got, dts in results[1:]:
        assert np.array_equal(got, results[0][0]) and dts == results[0][1]
    assert rel_err(cfg, results[0][0], oplan.interior(Uo)) <= 1e-11
    assert all(abs(g - o) <= 1e-12 * o for g, o in zip(results[0][1], dts_o))


@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_walls_all_round_chain_lengths_bitwise_and_conservation(recon, rk):
    """[B9] A closed box (reflecting walls on all six sides, 1 x 2 x 3 blocks): the fused kernel's image cells (x / y
    halos in the producer warp, z image planes in the prologue and the z loop) against the oracle's filled guard cells;
    the same bits for chain lengths 1, 2 and 8; and nothing leaves a closed box: total mass and energy are conserved
    to rounding."""
    cfg = inputs.config(5, nb=(1, 2, 3))
    oplan, neigh, coords = oracle_plan_for(cfg, bc="reflect", recon=recon, rk=rk)
    rng = np.random.default_rng(23)
    shape = (6, 16, 16, 16)
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    pr = 1.0 + 0.3 * rng.random(shape)
    Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = np.full((6, 3), 1.0 / 32)
    Uo = Uh.numpy().copy()
    dts = []
    for step in range(3):
        dts.append(oplan.compute_dt(Uo, dx, 0.3))
        oplan.advance(Uo, dx, dts[-1])
    results = []
    for zc in (1, 2, 8):
        gplan, _, _ = gpu_plan_for(cfg, bc="reflect", recon=recon, rk=rk, zchain=zc)
        assert gplan.path == 1
        Ud, dxd = Uh.cuda(), torch.from_numpy(dx).cuda()
        for dt in dts:
            gplan.fx_hydro_advance(Ud, dxd, dt)
        results.append(gplan.interior(Ud).cpu().numpy())
    assert np.array_equal(results[1], results[0]) and np.array_equal(results[2], results[0])
    assert rel_err(cfg, results[0], oplan.interior(Uo)) <= 1e-11
    for v in (0, 4):
        assert abs(results[0][v].sum() - Ui[v].sum()) <= 1e-12 * Ui[v].sum()


@pytest.mark.parametrize("path", [None, 1])
@pytest.mark.parametrize("recon,rk,bc", [(0, 2, "periodic"), (1, 3, "reflect")])
def test_constant_gravity_parity_and_free_fall(recon, rk, bc, path):
    """[B10] The gravity source in both stage kernels: parity with the oracle on general data (fused dt included), and
    the free-fall closed form m = m0 + rho g t, E = E0 + g.m0 t + rho |g|^2 t^2 / 2 for a uniform gas."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 2))
    grav = (0.7, -1.1, 0.4)
    oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, rk=rk)
    gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk, path=path)
    assert gplan.path == (1 if path is None else 0)
    for d in range(3):
        oplan.set_option(fxo.OPT_GRAVITY_X + d, grav[d])
        gplan.fx_hydro_plan_set_option(fx.OPT_GRAVITY_X + d, grav[d])
    rng = np.random.default_rng(31)
    shape = (8, 16, 16, 16)
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    pr = 1.0 + 0.3 * rng.random(shape)
    Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = np.full((8, 3), 1.0 / 32)
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    dt = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
    for step in range(3):
        dto = oplan.compute_dt(Uo, dx, 0.3)
        assert abs(float(dt.item()) - dto) <= 1e-12 * dto
        oplan.advance(Uo, dx, dto)
        gplan.fx_hydro_step(Ud, dxd, 0.3, dt)
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-11
    # free fall (periodic box only: a wall would stop the gas)
    if bc == "periodic":
        r0, v0, p0 = 1.3, np.array([0.2, 0.1, -0.4]), 0.9
        m0, E0 = r0 * v0, p0 / (cfg.gamma - 1) + 0.5 * r0 * (v0 ** 2).sum()
        U = torch.full(Uh.shape, float("nan"), dtype=torch.float64)
        I = inputs.interior_view(cfg, U)
        for v, val in enumerate((r0, m0[0], m0[1], m0[2], E0)):
            I[v] = val
        U = U.cuda()
        t = 0.0
        for dts in (0.01, 0.003, 0.02):
            gplan.fx_hydro_advance(U, dxd, dts)
            t += dts
        I = gplan.interior(U).cpu().numpy()
        g = np.array(grav)
        assert np.max(np.abs(I[0] - r0)) <= 1e-15
        for d in range(3):
            assert np.max(np.abs(I[1 + d] - (m0[d] + r0 * g[d] * t))) <= 1e-14
        assert np.max(np.abs(I[4] - (E0 + g @ m0 * t + 0.5 * r0 * (g ** 2).sum() * t * t))) <= 1e-14


@pytest.mark.parametrize("recon,rk,bc,path", [(0, 2, "periodic", None), (1, 3, "outflow", None), (0, 3, "reflect", None), (0, 2, "periodic", 1)])
def test_x_guard_depth_8_layout(recon, rk, bc, path):
    """FX_OPT_GUARD_X = 8: 256-byte row pitch.  Same interiors as the oracle (which keeps its own 4-deep layout) after
    three fused steps, on an array placed by alloc_state and on one deliberately misplaced by 16 bytes (placement
    changes the DRAM traffic, never the result: the two agree bit for bit); the filled guard zones equal the oracle's
    8-deep fill cropped to (8, 4, 4); and the option is refused once the workspace exists."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 2))
    oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, rk=rk)
    code = {"periodic": fx.TOPO_PERIODIC, "outflow": fx.TOPO_OUTFLOW, "reflect": fx.TOPO_REFLECT}[bc]
    gplan = fx.HydroPlan(cfg.block_dims, cfg.nguard, 8, cfg.gamma, recon, cfg.riemann, rk)
    if path is not None:
        gplan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
    gplan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 8)
    assert gplan.np == (32, 24, 24) and gplan.gd == (8, 4, 4) and gplan.S_j == 32
    gplan.fx_hydro_plan_set_topology(neigh)
    gplan.fx_hydro_plan_set_workspace()
    assert gplan.path == (1 if path is None else 0)
    with pytest.raises(fx.FxError):
        gplan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 4)
    for key in (fx.OPT_PATH, fx.OPT_ZCHAIN, fx.OPT_OWNED_BLOCKS):  # what the topology call builds its tables from
        with pytest.raises(fx.FxError):
            gplan.fx_hydro_plan_set_option(key, 1)
    gplan.fx_hydro_plan_set_option(fx.OPT_WAVESPEED, 0)  # a physics option may still change
    rng = np.random.default_rng(41)
    shape = (8, 16, 16, 16)
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    pr = 1.0 + 0.3 * rng.random(shape)
    Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
    Uo = inputs.embed(cfg, torch.from_numpy(Ui)).numpy()
    Ud = gplan.embed(Ui)
    assert (Ud.data_ptr() + 8 * 8) % 128 == 0
    n = int(np.prod(gplan.shape))
    buf = torch.full((n + 16,), float("nan"), dtype=torch.float64, device="cuda")
    Um = buf[2:2 + n].view(gplan.shape)  # interior rows at 80 mod 128
    gplan.interior(Um).copy_(torch.from_numpy(Ui))
    dx = np.full((8, 3), 1.0 / 32)
    dxd = torch.from_numpy(dx).cuda()
    dt = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
    dtm = dt.clone()
    for step in range(3):
        dto = oplan.compute_dt(Uo, dx, 0.3)
        assert abs(float(dt.item()) - dto) <= 1e-12 * dto
        oplan.advance(Uo, dx, dto)
        gplan.fx_hydro_step(Ud, dxd, 0.3, dt)
        gplan.fx_hydro_step(Um, dxd, 0.3, dtm)
    assert torch.equal(gplan.interior(Ud), gplan.interior(Um)) and torch.equal(dt, dtm)
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-11
    # guard fill in the wide layout against the oracle with 8 guard zones everywhere
    o8 = fxo.OraclePlan(cfg.block_dims, 8, 8, cfg.gamma, recon, cfg.riemann, rk)
    o8.set_topology(neigh)
    V = np.full(o8.shape, np.nan)
    o8.interior(V)[...] = gplan.interior(Ud).cpu().numpy()
    o8.fill_guardcells(V)
    gplan.fx_fill_guardcells(Ud)
    assert np.array_equal(Ud.cpu().numpy(), V[:, :, 4:-4, 4:-4, :])


@pytest.mark.parametrize("number,nb", [(2, None), (5, (2, 2, 2))])
def test_step_is_capturable_in_a_cuda_graph(number, nb):
    """fx_hydro_step only enqueues work on the caller's stream (tensor maps travel as kernel parameters, dt stays on the
    device), so a loop of steps can be captured once and replayed: same bits as the eager loop, on the generic path
    (5 launches per step: launch-bound on small problems) and on the fused one."""
    cfg, oplan, gplan, Uh, dx = setup(number, nb)
    dxd = torch.from_numpy(dx).cuda()
    A, B = Uh.cuda(), Uh.cuda()
    dta = gplan.fx_hydro_compute_dt(A, dxd, cfg.cfl).clone()
    dtb = dta.clone()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        gplan.fx_hydro_step(A, dxd, cfg.cfl, dta, stream=s)  # warm-up outside the capture (first-launch set-up)
        s.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=s):
            for _ in range(4):
                gplan.fx_hydro_step(A, dxd, cfg.cfl, dta, stream=torch.cuda.current_stream())
    torch.cuda.synchronize()
    g.replay()
    g.replay()
    torch.cuda.synchronize()
    for _ in range(1 + 8):
        gplan.fx_hydro_step(B, dxd, cfg.cfl, dtb)
    torch.cuda.synchronize()
    assert torch.equal(gplan.interior(A), gplan.interior(B)) and torch.equal(dta, dtb)
    fg, _ = gplan.fx_hydro_status()
    assert fg == 0


@pytest.mark.parametrize("recon,rk,bc", [(0, 2, "periodic"), (1, 3, "reflect"), (0, 3, "outflow")])
def test_repeated_runs_are_bitwise_identical(recon, rk, bc):
    """compute-sanitizer's racecheck is closed on this pool, so the shared-memory protocol of the fused kernel (ring and
    halo slots, two barriers per plane, three warp roles) is also checked by determinism: 512 blocks (more segments than
    resident CTAs, so slots are reused under every interleaving the scheduler produces), 3 steps, 12 repeats from the
    same state -- every repeat must give the same bits, state and dt."""
    cfg = inputs.config(5, nb=(8, 8, 8))
    gplan, neigh, coords = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk)
    assert gplan.path == 1
    U0 = gplan.embed(inputs.block_interiors(cfg, coords, "cuda"))
    dxd = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    ref = None
    for rep in range(12):
        U = U0.clone()
        dt = gplan.fx_hydro_compute_dt(U, dxd, cfg.cfl).clone()
        for _ in range(3):
            gplan.fx_hydro_step(U, dxd, cfg.cfl, dt)
        got = (gplan.interior(U).clone(), dt.clone())
        if ref is None:
            ref = got
        else:
            assert torch.equal(got[0], ref[0]) and torch.equal(got[1], ref[1]), rep
    assert torch.isfinite(ref[0]).all()


@pytest.mark.parametrize("dims,nb,nguard,recon,rk,bc,grav", [
    ((8, 8, 8), (3, 2, 2), 4, 0, 2, "periodic", False), ((8, 8, 8), (2, 2, 3), 4, 1, 3, "reflect", True),
    ((8, 8, 8), (2, 3, 2), 2, 0, 3, "outflow", False), ((8, 6, 5), (2, 2, 2), 3, 1, 2, "periodic", False),
    ((32, 32, 1), (2, 2, 1), 4, 0, 2, "reflect", True), ((256, 1, 1), (2, 1, 1), 4, 1, 3, "outflow", False)])
def test_tile_kernel_small_blocks(dims, nb, nguard, recon, rk, bc, grav):
    """The shared-memory tile kernel (path 2: blocks whose padded zones fit a CTA's shared memory -- 8^3 blocks, 2-D and
    1-D blocks): parity with the oracle after 1 and 5 steps, the same status flags, agreement with the generic kernel to
    rounding, walls, gravity, odd guard depths and non-cubic blocks included."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=nb)
    cfg.block_dims, cfg.nguard = dims, nguard
    oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, rk=rk)
    gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk, path=2)  # 2: prefer the tile kernel (3-D PLM blocks default to the generic one)
    gen, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk, path=1)
    auto, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk)
    assert gplan.path == 2 and gen.path == 0 and auto.path == (0 if (recon == 0 and min(dims) > 1) else 2)
    g = (0.7, -1.1 if dims[1] > 1 else 0.0, 0.4 if dims[2] > 1 else 0.0)
    if grav:
        for d in range(3):
            oplan.set_option(fxo.OPT_GRAVITY_X + d, g[d])
            gplan.fx_hydro_plan_set_option(fx.OPT_GRAVITY_X + d, g[d])
            gen.fx_hydro_plan_set_option(fx.OPT_GRAVITY_X + d, g[d])
    nblk = nb[0] * nb[1] * nb[2]
    rng = np.random.default_rng(77)
    shape = (nblk, dims[2], dims[1], dims[0])
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    for d in (1, 2):
        if dims[d] == 1:
            vel[d] = 0.0
    pr = 1.0 + 0.3 * rng.random(shape)
    Ui = np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = np.full((nblk, 3), 1.0 / 64)
    Uo, Ud, Ug, dxd = Uh.numpy().copy(), Uh.cuda(), Uh.cuda(), torch.from_numpy(dx).cuda()
    for step in range(5):
        dt = oplan.compute_dt(Uo, dx, 0.3)
        oplan.advance(Uo, dx, dt)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        gen.fx_hydro_advance(Ug, dxd, dt)
        err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
        assert err <= (1e-12 if step == 0 else 1e-10), (step, err)
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), gen.interior(Ug).cpu().numpy()) <= 1e-11
    assert oplan.status()[0] == gplan.fx_hydro_status()[0]
    # the step call (dt of the advanced state by the reduction pass) on the tile path
    dtd = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
    gplan.fx_hydro_step(Ud, dxd, 0.3, dtd)
    dto = oplan.compute_dt(Uo, dx, 0.3)
    oplan.advance(Uo, dx, dto)
    assert abs(float(dtd.item()) - oplan.compute_dt(Uo, dx, 0.3)) <= 1e-12 * dto


@pytest.mark.parametrize("path", [None, 1])
def test_status_flags_floors_and_nonfinite(path):
    """A7/A27: primitive floors and non-finite states raise the same status bits as in the oracle, the floored step
    still agrees with it, and nothing traps or hangs."""
    from paper_2208_11630_b200 import binding as fx
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 2), path=path)
    Ui = inputs.interior_view(cfg, Uh)
    Ui[4, 3, 5, 6, 7] = 1e-3          # energy below the kinetic energy: negative pressure -> p floor
    Ui[0, 5, 9, 2, 11] = -0.5         # negative density (at rest, so that the floored state stays finite) -> rho floor
    Ui[1:4, 5, 9, 2, 11] = 0.0
    Uo, Ud, dxd = Uh.numpy().copy(), Uh.cuda(), torch.from_numpy(dx).cuda()
    oplan.advance(Uo, dx, 1e-6)
    gplan.fx_hydro_advance(Ud, dxd, 1e-6)
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fo == fg and (fg & fx.STATUS_P_FLOOR) and (fg & fx.STATUS_RHO_FLOOR) and not (fg & fx.STATUS_NONFINITE)
    got, ref = gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)
    ok = np.ones(got.shape[1:], dtype=bool)
    ok[3, 3:8, 4:9, 5:10] = False     # the neighbourhoods of the two bad zones hold huge floored-state values
    ok[5, 7:12, 0:5, 9:14] = False
    scale = np.abs(ref[:, ok]).max()
    assert np.max(np.abs(got[:, ok] - ref[:, ok])) <= 1e-12 * scale
    assert np.all(np.isfinite(got[:, ~ok]) == np.isfinite(ref[:, ~ok]))
    # a NaN zone: flagged, not trapped
    gplan.fx_hydro_status_reset()
    Ud2 = Uh.cuda()
    gplan.interior(Ud2)[1, 2, 4, 4, 4] = float("nan")
    gplan.fx_hydro_advance(Ud2, dxd, 1e-6)
    torch.cuda.synchronize()
    fg2, _ = gplan.fx_hydro_status()
    assert fg2 & fx.STATUS_NONFINITE


def test_advance_host_equals_device_path():
    cfg, oplan, gplan, Uh, dx = setup(3, (2, 2, 2))
    dxd = torch.from_numpy(dx).cuda()
    A = Uh.cuda()
    for _ in range(2):
        gplan.fx_hydro_advance(A, dxd, gplan.fx_hydro_compute_dt(A, dxd, cfg.cfl))
    Hh = Uh.clone().pin_memory()
    dxh = torch.from_numpy(dx).pin_memory()
    stage, dstage = torch.empty_like(A), torch.empty_like(dxd)
    dt_last = gplan.fx_hydro_advance_host(Hh, dxh, cfg.cfl, 2, stage, dstage)
    assert np.isfinite(dt_last) and dt_last > 0
    assert torch.equal(gplan.interior(Hh), gplan.interior(A).cpu())
    # the interior-only host call: same bits, a staging state whose guard zones are NaN, both layouts
    for gx, number in ((4, 3), (8, 5), (4, 2)):
        cfg2, _, g2, Uh2, dx2 = setup(number, (2, 2, 2) if number != 2 else None)
        if gx == 8:
            from paper_2208_11630_b200 import binding as fx
            g2 = fx.HydroPlan(cfg2.block_dims, cfg2.nguard, g2.nblocks, cfg2.gamma, cfg2.recon, cfg2.riemann, cfg2.rk_order)
            g2.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 8)
            g2.fx_hydro_plan_set_topology(gpu_plan_for(cfg2)[1])
            g2.fx_hydro_plan_set_workspace()
        Ui = inputs.interior_view(cfg2, Uh2).contiguous()
        B = g2.embed(Ui)
        dxd2 = torch.from_numpy(dx2).cuda()
        for _ in range(2):
            g2.fx_hydro_advance(B, dxd2, g2.fx_hydro_compute_dt(B, dxd2, cfg2.cfl))
        Hi = Ui.clone().pin_memory()
        assert tuple(Hi.shape) == g2.interior_shape
        stage = g2.alloc_state(fill=float("nan"))
        packed = torch.empty(Hi.numel(), dtype=torch.float64, device="cuda")
        dt2 = g2.fx_hydro_advance_host_interior(Hi, torch.from_numpy(dx2).pin_memory(), cfg2.cfl, 2, stage, packed,
                                                torch.empty_like(dxd2))
        assert np.isfinite(dt2) and dt2 > 0
        assert torch.equal(Hi, g2.interior(B).cpu())


@pytest.mark.parametrize("recon,riemann,rk", [(0, 0, 2), (0, 1, 3), (1, 0, 3), (1, 1, 2)])
def test_uniform_state_preserved_bitwise(recon, riemann, rk):
    for dims, nb in (((16, 16, 16), (2, 2, 2)), ((6, 5, 4), (2, 1, 2)), ((16, 16, 1), (2, 2, 1))):
        cfg = inputs.config(3, nb=nb)
        cfg.block_dims = dims
        for bc in ("periodic", "outflow"):
            gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk)
            W = (1.3, 0.7, -0.4, 0.2, 2.2)
            E = W[4] / (cfg.gamma - 1) + 0.5 * W[0] * (W[1] ** 2 + W[2] ** 2 + W[3] ** 2)
            U = torch.full(gplan.shape, float("nan"), dtype=torch.float64, device="cuda")
            for v, val in enumerate((W[0], W[0] * W[1], W[0] * W[2], W[0] * W[3], E)):
                gplan.interior(U)[v] = val
            U0 = gplan.interior(U).clone()
            dx = torch.tensor([[0.1, 0.2, 0.15]] * gplan.nblocks, dtype=torch.float64, device="cuda")
            for _ in range(10):
                gplan.fx_hydro_advance(U, dx, 0.01)
            assert torch.equal(gplan.interior(U), U0)


def test_guard_contents_do_not_matter_and_bad_dt_is_refused():
    from paper_2208_11630_b200 import binding as fx
    cfg, oplan, gplan, Uh, dx = setup(5, (2, 2, 2))
    dxd = torch.from_numpy(dx).cuda()
    Ui = inputs.interior_view(cfg, Uh)
    A = inputs.embed(cfg, Ui, float("nan")).cuda()
    B = inputs.embed(cfg, Ui, 123.0).cuda()
    gplan.fx_hydro_advance(A, dxd, 1e-4)
    gplan.fx_hydro_advance(B, dxd, 1e-4)
    assert torch.equal(gplan.interior(A), gplan.interior(B))
    for bad in (0.0, -1.0, float("nan"), float("inf")):
        with pytest.raises(fx.FxError) as e:
            gplan.fx_hydro_advance(A, dxd, bad)
        assert e.value.code == fx.ERR_INVALID_ARG


def test_block_permutation_invariance_bitwise():
    cfg = inputs.config(5, nb=(3, 2, 2))
    gplan, neigh, coords = gpu_plan_for(cfg)
    Uh = inputs.embed(cfg, inputs.block_interiors(cfg, coords))
    perm = np.random.default_rng(3).permutation(12)
    inv = np.argsort(perm)
    neigh_p = neigh[perm].copy()
    neigh_p[neigh_p >= 0] = inv[neigh_p[neigh_p >= 0]]
    gplan_p, _, _ = gpu_plan_for(cfg, neigh=neigh_p)
    A = Uh.cuda()
    B = Uh[:, perm].contiguous().cuda()
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    for _ in range(2):
        gplan.fx_hydro_advance(A, dx, 2e-4)
        gplan_p.fx_hydro_advance(B, dx, 2e-4)
    assert torch.equal(gplan.interior(A)[:, perm], gplan_p.interior(B))


def test_sod_mirror_symmetry_and_run_to_time():
    cfg, oplan, gplan, Uh, dx = setup(1)
    dxd = torch.from_numpy(dx).cuda()
    A = Uh.cuda()
    M = Uh.flip(-1).clone()
    M[1] *= -1
    M = M.cuda()
    gplan.fx_hydro_advance(A, dxd, 0.0026411070460266143)
    gplan.fx_hydro_advance(M, dxd, 0.0026411070460266143)
    a, m = gplan.interior(A).cpu().numpy(), gplan.interior(M).cpu().numpy()[..., ::-1]
    assert np.max(np.abs(a[0] - m[0])) <= 1e-13 and np.max(np.abs(a[4] - m[4])) <= 1e-13 * 2.5
    assert np.max(np.abs(a[1] + m[1])) <= 1e-13
    # whole run to t = 0.2 with the GPU's own dt, last step clipped; compare with the oracle's run
    Uo = Uh.numpy().copy()
    Ud = Uh.cuda()
    t = 0.0
    n = 0
    while t < 0.2:
        dt = float(gplan.fx_hydro_compute_dt(Ud, dxd, cfg.cfl).item())
        dto = oplan.compute_dt(Uo, dx, cfg.cfl)
        assert abs(dt - dto) <= 1e-11 * dto  # states drift apart by rounding only
        dt = min(dto, 0.2 - t)
        gplan.fx_hydro_advance(Ud, dxd, dt)
        oplan.advance(Uo, dx, dt)
        t += dt
        n += 1
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-9
