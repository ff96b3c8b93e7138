"""Passive mass scalars (reading B11) at BASELINE.json's full size: config 5 (32768 blocks of 16^3) with two
scalars, in the launch configuration `bench.py --scalars 2` times (Morton block order, wide layout, generic path,
fx_hydro_step), checked on sampled blocks the oracle computes from their 3^3-block neighbourhoods (after n RK2 steps a
zone depends on zones at most 4n away, so n <= 4 steps are exact on the centre block), plus conservation."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import rel_err

pytestmark = pytest.mark.gpu

NS = 2


def test_full_size_scalars_sampled_blocks_and_conservation():
    from paper_2208_11630_b200 import binding as fx
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 90e9:
        pytest.skip("needs 90 GB of free HBM")
    cfg = inputs.config(5)
    bcs = [fx.TOPO_PERIODIC] * 3
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order,
                        nvars=5 + NS)
    plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 8)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    assert plan.path == 1  # fused kernel + scalar pass (config 5 is periodic, PLM)
    U = plan.alloc_state(fill=float("nan"))
    Ui = plan.interior(U)
    for b0 in range(0, cfg.nblocks, 1024):
        c = coords[b0:b0 + 1024]
        Ui[:, b0:b0 + 1024] = inputs.with_scalars(cfg, c, inputs.block_interiors(cfg, c, "cuda"), NS)
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    id_of = {tuple(int(x) for x in c): b for b, c in enumerate(coords)}
    tot0 = [float(Ui[v].sum(dtype=torch.float64)) for v in range(5 + NS)]

    def neighbourhood_oracle(centre):
        nbc, shape = inputs.neighbourhood(cfg, centre, 1)
        ids = [id_of[tuple(int(x) for x in c)] for c in nbc]
        sub = inputs.config(5, nb=shape)
        on, _ = fxo.topology_cartesian(shape, [fxo.TOPO_OUTFLOW] * 3, [fxo.TOPO_OUTFLOW] * 3, fxo.ORDER_LEX)
        oplan = fxo.OraclePlan(sub.block_dims, sub.nguard, len(ids), sub.gamma, sub.recon, sub.riemann, sub.rk_order,
                               nvars=5 + NS)
        oplan.set_topology(on)
        Uo = np.full(oplan.shape, np.nan)
        oplan.interior(Uo)[...] = plan.interior(U[:, torch.as_tensor(ids, device=U.device)]).cpu().numpy()
        return oplan, Uo, ids, len(ids) // 2

    # a corner block (periodic wrap), a block on the composition interface of scalar 1 (x = N/4), an interior one
    oracles = [neighbourhood_oracle(c) for c in ((0, 0, 0), (8, 13, 21), (17, 5, 30))]
    dt_dev = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    dts = []
    for step in range(3):
        dts.append(float(dt_dev.item()))
        plan.fx_hydro_step(U, dx, cfg.cfl, dt_dev)
        for oplan, Uo, ids, mid in oracles:
            oplan.advance(Uo, inputs.dx_array(cfg, len(ids)), dts[-1])
            got = plan.interior(U[:, ids[mid]:ids[mid] + 1]).cpu().numpy()
            ref = oplan.interior(Uo)[:, mid:mid + 1]
            tol = 1e-12 if step == 0 else 1e-9
            assert rel_err(cfg, got[:5], ref[:5]) <= tol
            assert float((np.abs(got[5:] - ref[5:]) / ref[0]).max()) <= tol
    # the interface block's scalar did change
    oplan, Uo, ids, mid = oracles[1]
    assert np.abs(oplan.interior(Uo)[6, mid]).max() > 0
    tot = [float(plan.interior(U)[v].sum(dtype=torch.float64)) for v in range(5 + NS)]
    for v in (0, 4, 5, 6):
        assert abs(tot[v] - tot0[v]) <= 1e-13 * max(abs(tot0[v]), tot0[0])
    flags, _ = plan.fx_hydro_status()
    assert not (flags & 1)
    del U, plan
    torch.cuda.empty_cache()
