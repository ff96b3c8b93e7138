"""Parity at BASELINE.json's full size (config 5: 32768 blocks of 16^3) in the launch configuration bench.py times
(Morton block order, auto path = fused kernel, the wide layout FX_OPT_GUARD_X = 8 stepped with fx_hydro_step; and the
compact layout stepped with compute_dt + advance), on sampled blocks the oracle can compute one by one, plus properties
that hold at any size (conservation, dt = global min, index maps).

After n RK2 steps a zone depends on zones at most 4n away (2 stages x 2 cells), so the interior of a sampled
block equals that of an oracle run on its (2r+1)^3-block neighbourhood alone when 4n <= 16 r."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import rel_err

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module", params=[8, 4], ids=["wide-layout-step", "compact-layout-advance"])
def full(request):
    from paper_2208_11630_b200 import binding as fx
    gx = request.param
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 60e9:
        pytest.skip("needs 60 GB of free HBM")
    cfg = inputs.config(5)
    bcs = [fx.TOPO_PERIODIC] * 3
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order)
    if gx != cfg.nguard:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, gx)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    assert plan.path == 1  # the fused TMA stage kernel is what runs
    U = plan.alloc_state(fill=float("nan"))  # as bench.py places it
    Ui = plan.interior(U)
    for b0 in range(0, cfg.nblocks, 1024):
        Ui[:, b0:b0 + 1024] = inputs.block_interiors(cfg, coords[b0:b0 + 1024], "cuda")
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    id_of = {tuple(int(x) for x in c): b for b, c in enumerate(coords)}
    yield cfg, plan, U, dx, neigh, coords, id_of, gx
    del U, plan
    torch.cuda.empty_cache()


def neighbourhood_oracle(cfg, plan, U, id_of, centre, radius):
    """Oracle plan over the (2r+1)^3 blocks around `centre` (outflow outside) with the bytes the GPU holds."""
    nbc, shape = inputs.neighbourhood(cfg, centre, radius)
    ids = [id_of[tuple(int(x) for x in c)] for c in nbc]
    sub = inputs.config(5, nb=shape)
    neigh, _ = fxo.topology_cartesian(shape, [fxo.TOPO_OUTFLOW] * 3, [fxo.TOPO_OUTFLOW] * 3, fxo.ORDER_LEX)
    oplan = fxo.OraclePlan(sub.block_dims, sub.nguard, len(ids), sub.gamma, sub.recon, sub.riemann, sub.rk_order)
    oplan.set_topology(neigh)
    Uo = np.full(oplan.shape, np.nan)  # the oracle's own (compact) layout; guard zones are filled by its advance
    oplan.interior(Uo)[...] = plan.interior(U[:, torch.as_tensor(ids, device=U.device)]).cpu().numpy()
    return oplan, Uo, ids, len(ids) // 2  # the centre block is the middle one in lexicographic offset order


def test_full_size_sampled_blocks_dt_and_conservation(full):
    cfg, plan, U, dx, neigh, coords, id_of, gx = full
    if gx == cfg.nguard:
        # guard-cell index map of sampled blocks, bit-exact against the oracle on the full topology (same layout)
        oplan_full = fxo.OraclePlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order)
        oplan_full.set_topology(neigh)
        for b0 in (0, 12345, cfg.nblocks - 3):
            assert np.array_equal(plan.fx_guardcell_index_map(b0, 3).cpu().numpy(), oplan_full.index_map(b0, 3))
    Ui = plan.interior(U)
    tot0 = [float(Ui[v].sum(dtype=torch.float64)) for v in range(5)]
    # dt: the global minimum is attained in some block; the oracle's dt on that block alone must equal it
    dt = float(plan.fx_hydro_compute_dt(U, dx, cfg.cfl).item())
    rho = Ui[0]
    u = [Ui[d] / rho for d in (1, 2, 3)]
    p = (cfg.gamma - 1) * (Ui[4] - 0.5 * rho * (u[0] ** 2 + u[1] ** 2 + u[2] ** 2))
    cs = torch.sqrt(cfg.gamma * p / rho)
    per_block = torch.stack([(cfg.dx[d] / (u[d].abs() + cs)).amin(dim=(1, 2, 3)) for d in range(3)]).amin(dim=0)
    bmin = int(per_block.argmin())
    del rho, u, p, cs
    op1 = fxo.OraclePlan(cfg.block_dims, cfg.nguard, 1, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order)
    U1 = np.full(op1.shape, np.nan)
    op1.interior(U1)[...] = plan.interior(U[:, bmin:bmin + 1]).cpu().numpy()
    dt_o = op1.compute_dt(U1, inputs.dx_array(cfg, 1), cfg.cfl)
    assert abs(dt - dt_o) <= 1e-14 * dt_o
    assert abs(dt - cfg.cfl * float(per_block.min())) <= 1e-13 * dt
    # sampled blocks: a corner block (periodic wrap in all directions), an interior one, the last one
    samples = [(0, 0, 0), (17, 5, 30), (31, 31, 31)]
    oracles = [neighbourhood_oracle(cfg, plan, U, id_of, c, 1) for c in samples]
    long_run = neighbourhood_oracle(cfg, plan, U, id_of, (9, 22, 14), 3)
    dts = []
    dt_dev = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    for step in range(10):
        if gx == cfg.nguard:
            dts.append(float(plan.fx_hydro_compute_dt(U, dx, cfg.cfl).item()))
            plan.fx_hydro_advance(U, dx, dts[-1])
        else:  # bench.py's step: the dt of the advanced state comes out of the last stage
            dts.append(float(dt_dev.item()))
            plan.fx_hydro_step(U, dx, cfg.cfl, dt_dev)
        if step == 0:
            for oplan, Uo, ids, mid in oracles:
                oplan.advance(Uo, inputs.dx_array(cfg, len(ids)), dts[0])
                got = plan.interior(U[:, ids[mid]:ids[mid] + 1]).cpu().numpy()
                assert rel_err(cfg, got, oplan.interior(Uo)[:, mid:mid + 1]) <= 1e-12
            tot1 = [float(plan.interior(U)[v].sum(dtype=torch.float64)) for v in range(5)]
    oplan, Uo, ids, mid = long_run
    for d in dts:
        oplan.advance(Uo, inputs.dx_array(cfg, len(ids)), d)
    got = plan.interior(U[:, ids[mid]:ids[mid] + 1]).cpu().numpy()
    assert rel_err(cfg, got, oplan.interior(Uo)[:, mid:mid + 1]) <= 1e-9
    # conservation on the periodic domain [A22]: momentum is scaled by sum rho(|u|+c) ~ 2.4 sum rho
    tot10 = [float(plan.interior(U)[v].sum(dtype=torch.float64)) for v in range(5)]
    for tot in (tot1, tot10):
        assert abs(tot[0] - tot0[0]) <= 1e-13 * tot0[0] and abs(tot[4] - tot0[4]) <= 1e-13 * tot0[4]
        for v in (1, 2, 3):
            assert abs(tot[v] - tot0[v]) <= 1e-13 * 2.0 * tot0[0]
    flags, counts = plan.fx_hydro_status()
    assert not (flags & 1)  # nothing non-finite
