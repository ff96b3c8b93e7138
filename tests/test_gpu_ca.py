"""fx_hydro_advance_ca (communication-avoiding step, B17) on the GPU: parity with the oracle's
fxo_hydro_advance_ca element by element (<= 1e-12 after one step, <= 1e-9 after ten [NS]), and -- the variant's defining
property -- the SAME BITS as fx_hydro_advance on the generic path (FX_OPT_PATH = 1), whose kernels it shares: an extended
zone is the neighbour's interior zone, updated with the same instructions from the same numbers."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for, oracle_plan_for, rel_err

pytestmark = pytest.mark.gpu

PLM, WENO = 0, 1
CASES = [
    (5, (3, 3, 3), PLM, 2, 4, "periodic", {}),      # several blocks per dimension, Morton order below
    (5, (2, 2, 2), PLM, 3, 6, "periodic", {}),
    (4, (2, 2, 2), WENO, 2, 6, "periodic", {}),
    (4, (2, 1, 2), WENO, 3, 9, "periodic", {}),
    (5, (2, 2, 2), PLM, 2, 4, "outflow", {}),
    (5, (2, 2, 1), PLM, 3, 6, "reflect", {}),
    (5, (2, 2, 2), PLM, 2, 5, "reflect", dict(riemann=0, wavespeed=1)),
    (2, (4, 4, 1), PLM, 2, 4, "periodic", {}),      # 2-D
    (2, (2, 2, 1), PLM, 3, 6, "outflow", {}),
    (1, (1, 1, 1), PLM, 2, 4, "outflow", {}),       # 1-D
]


@pytest.mark.parametrize("number,nb,recon,rk,g,bc,kw", CASES)
def test_ca_parity_with_the_oracle_and_bitwise_with_the_standard_step(number, nb, recon, rk, g, bc, kw):
    cfg = inputs.config(number, nb=nb)
    cfg.nguard = g
    order = inputs.ORDER_MORTON if number == 5 and bc == "periodic" else inputs.ORDER_LEX
    oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, rk=rk, order=order, **kw)
    gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, rk=rk, order=order, path=1, **kw)   # generic path
    assert gplan.path == 0
    Uh = inputs.embed(cfg, inputs.block_interiors(cfg, coords))
    dx = inputs.dx_array(cfg)
    dxd = torch.from_numpy(dx).cuda()
    Uo = Uh.numpy().copy()
    Uca, Ustd = Uh.cuda(), Uh.cuda()
    Uca[...] = float("nan")                                   # the step must not depend on guard zones on entry
    gplan.interior(Uca).copy_(gplan.interior(Ustd))
    for step in range(10):
        dto = oplan.compute_dt(Uo, dx, cfg.cfl)
        dtg = float(gplan.fx_hydro_compute_dt(Ustd, dxd, cfg.cfl).item())
        assert abs(dtg - dto) <= 1e-12 * dto
        oplan.advance_ca(Uo, dx, dto)
        gplan.fx_hydro_advance_ca(Uca, dxd, dto)
        gplan.fx_hydro_advance(Ustd, dxd, dto)
        assert torch.equal(gplan.interior(Uca), gplan.interior(Ustd)), step
        if step in (0, 9):
            err = rel_err(cfg, gplan.interior(Uca).cpu().numpy(), oplan.interior(Uo))
            assert err <= (1e-12 if step == 0 else 1e-9), (step, err)
    fo, _ = oplan.status()
    fg, _ = gplan.fx_hydro_status()
    assert fg == fo


def test_ca_with_device_dt_and_gravity():
    cfg = inputs.config(5, nb=(2, 2, 2))
    oplan, neigh, coords = oracle_plan_for(cfg, bc="reflect")
    gplan, _, _ = gpu_plan_for(cfg, bc="reflect", path=1)
    for pl, mod in ((oplan, fxo), (gplan, None)):
        if mod:
            pl.set_option(fxo.OPT_GRAVITY_Z, -0.7)
        else:
            from paper_2208_11630_b200 import binding as fx
            pl.fx_hydro_plan_set_option(fx.OPT_GRAVITY_Z, -0.7)
    Uh = inputs.embed(cfg, inputs.block_interiors(cfg, coords))
    dx = inputs.dx_array(cfg)
    dxd = torch.from_numpy(dx).cuda()
    Uo, Ud = Uh.numpy().copy(), Uh.cuda()
    for step in range(3):
        dt = gplan.fx_hydro_compute_dt(Ud, dxd, cfg.cfl)      # stays on the device
        dto = oplan.compute_dt(Uo, dx, cfg.cfl)
        gplan.fx_hydro_advance_ca(Ud, dxd, dt)
        oplan.advance_ca(Uo, dx, float(dt.item()))
        assert abs(float(dt.item()) - dto) <= 1e-12 * dto
    assert rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo)) <= 1e-11


def test_ca_refusals():
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(4, nb=(2, 2, 2))                      # WENO5 + RK3 with 4 guard zones: needs 9
    gplan, neigh, coords = gpu_plan_for(cfg)
    U = gplan.alloc_state(fill=1.0)
    dxd = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    with pytest.raises(fx.FxError, match="nguard"):
        gplan.fx_hydro_advance_ca(U, dxd, 1e-4)
    cfg = inputs.config(5, nb=(2, 2, 2))
    gplan, neigh, coords = gpu_plan_for(cfg, nvars=7)
    with pytest.raises(fx.FxError, match="scalars"):
        gplan.fx_hydro_advance_ca(gplan.alloc_state(fill=1.0), dxd, 1e-4)
    gplan, neigh, coords = gpu_plan_for(cfg)
    with pytest.raises(fx.FxError, match="dt"):
        gplan.fx_hydro_advance_ca(gplan.alloc_state(fill=1.0), dxd, -1.0)


def test_ca_at_config3_size_against_the_fused_path():
    """Config 3's tiling (512 blocks of 16^3, RK2 + PLM + HLLC as it is run) with config 5's smooth field: the CA step
    against the default (fused) path, which differs from the generic kernels by rounding only."""
    cfg = inputs.config(5, nb=(8, 8, 8))
    gca, neigh, coords = gpu_plan_for(cfg, path=1, order=inputs.ORDER_MORTON)
    gfu, _, _ = gpu_plan_for(cfg, order=inputs.ORDER_MORTON)
    assert gfu.path == 1 and gca.path == 0
    Ui = inputs.block_interiors(cfg, coords, "cuda")
    A, B = gca.embed(Ui), gfu.embed(Ui)
    dxd = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    for step in range(5):
        dt = gfu.fx_hydro_compute_dt(B, dxd, cfg.cfl).clone()
        gca.fx_hydro_advance_ca(A, dxd, dt)
        gfu.fx_hydro_advance(B, dxd, dt)
    assert rel_err(cfg, gca.interior(A).cpu().numpy(), gfu.interior(B).cpu().numpy()) <= 1e-10
