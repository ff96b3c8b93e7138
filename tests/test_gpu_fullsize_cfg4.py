"""Parity of config 4 at its own size (BASELINE.json configs[3]: 4096 blocks of 16^3 tiling a periodic 256^3 cube, WENO5 +
HLLC, SSP-RK3) in the launch configuration bench.py --config 4 times: Morton block order, the wide layout
(FX_OPT_GUARD_X = 8), the automatic path (fused TMA kernel, automatic chain length) and fx_hydro_step with the time step
left on the device by the last stage.

The oracle runs the WHOLE domain (16.8 M zones, 10 RK3 steps: about a minute on the box's host cores), so every zone is
compared, the field is the smooth one [CFG4] specifies (no reduced tiling, no jump at the wrap [B5]) and nothing is
sampled: <= 1e-12 after one step, <= 1e-9 after ten [NS], dt <= 1e-14 every step."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import rel_err

pytestmark = pytest.mark.gpu


def test_config4_whole_domain_1_and_10_steps():
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(4)
    assert cfg.nblocks == 4096 and cfg.block_dims == (16, 16, 16)
    bcs = [fx.TOPO_PERIODIC] * 3
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order)
    plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 8)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    assert plan.path == 1
    U = plan.alloc_state(fill=float("nan"))
    Ui = plan.interior(U)
    for b0 in range(0, cfg.nblocks, 1024):
        Ui[:, b0:b0 + 1024] = inputs.block_interiors(cfg, coords[b0:b0 + 1024], "cuda")
    dxh = inputs.dx_array(cfg)
    dx = torch.from_numpy(dxh).cuda()
    # the oracle on the same bytes, same neighbour table (its own compact layout)
    oplan = fxo.OraclePlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order)
    oplan.set_topology(neigh)
    Uo = np.full(oplan.shape, np.nan)
    oplan.interior(Uo)[...] = Ui.cpu().numpy()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    for step in range(10):
        dto = oplan.compute_dt(Uo, dxh, cfg.cfl)
        dtg = float(dt.item())
        assert abs(dtg - dto) <= 1e-14 * dto, (step, dtg, dto)
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)      # advances by the device-resident dt, leaves the next one
        oplan.advance(Uo, dxh, dtg)                 # same dt on both sides: the step is what is compared
        if step in (0, 9):
            err = rel_err(cfg, plan.interior(U).cpu().numpy(), oplan.interior(Uo))
            assert err <= (1e-12 if step == 0 else 1e-9), (step, err)
    fo, _ = oplan.status()
    fg, _ = plan.fx_hydro_status()
    assert fo == 0 and fg == 0  # no floor, no fallback on the smooth field [A6, A7]
