"""Blocks of 8 x 8 x nz zones on the fused kernel: 2 x 2 bundles of x / y neighbours march as one 16 x 16 cross-section
(csrc/fx_stage_bundle.cu, fx_hydro_plan_path = 4).  Parity with the oracle to the [NS] tolerances, the fused time step,
results independent of the chain length bit for bit, outflow boundaries, per-block dx, uniform state bit for bit,
agreement with the generic kernel, and the cases that must NOT bundle."""
import numpy as np
import pytest
import torch

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for, oracle_plan_for, rel_err

pytestmark = pytest.mark.gpu


def random_state(cfg, nblk, dims, seed):
    rng = np.random.default_rng(seed)
    shape = (nblk, dims[2], dims[1], dims[0])
    rho = 1.0 + 0.3 * rng.random(shape)
    vel = 0.4 * rng.standard_normal((3,) + shape)
    pr = 1.0 + 0.3 * rng.random(shape)
    return np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], pr / (cfg.gamma - 1) + 0.5 * rho * (vel ** 2).sum(0)])


@pytest.mark.parametrize("nb,dims,recon,riemann,rk,bc,order,kw", [
    ((4, 4, 4), (8, 8, 8), 0, 1, 2, "periodic", 1, {}), ((2, 4, 3), (8, 8, 8), 1, 1, 3, "periodic", 0, {}),
    ((4, 2, 2), (8, 8, 8), 0, 0, 3, "outflow", 1, {}), ((2, 2, 5), (8, 8, 4), 1, 0, 2, "outflow", 0, {}),
    ((4, 4, 2), (8, 8, 16), 0, 1, 2, "periodic", 1, dict(wavespeed=1)), ((2, 2, 2), (8, 8, 8), 0, 1, 2, "periodic", 0, {}),
    ((2, 2, 12), (8, 8, 8), 0, 1, 2, "periodic", 0, {}), ((2, 2, 20), (8, 8, 4), 1, 1, 3, "outflow", 0, {})])
def test_bundle_parity_chain_lengths_and_generic(nb, dims, recon, riemann, rk, bc, order, kw):
    cfg = inputs.config(5, nb=nb)
    cfg.block_dims = dims
    oplan, neigh, coords = oracle_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk, order=order, **kw)
    nblk = neigh.shape[0]
    Ui = random_state(cfg, nblk, dims, 3)
    Uh = inputs.embed(cfg, torch.from_numpy(Ui))
    dx = np.random.default_rng(9).uniform(1.0 / 40, 1.0 / 24, size=(nblk, 3))  # a different dx per block
    dxd = torch.from_numpy(dx).cuda()
    Uo = Uh.numpy().copy()
    results = []
    for zc in (None, 1, 3, 16):  # 16: the longest chain (a column of 12 or 20 layers is marched as one or two segments)
        gplan, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk, order=order, zchain=zc, **kw)
        assert gplan.path == 4
        Ud = Uh.cuda()
        dt = gplan.fx_hydro_compute_dt(Ud, dxd, 0.3).clone()
        dts = []
        for step in range(10):
            dts.append(float(dt.item()))
            if zc is None:
                dto = oplan.compute_dt(Uo, dx, 0.3)
                assert abs(dts[-1] - dto) <= 1e-13 * dto, (step, dts[-1], dto)
                oplan.advance(Uo, dx, dts[-1])
            gplan.fx_hydro_step(Ud, dxd, 0.3, dt)
            if zc is None and step in (0, 9):
                err = rel_err(cfg, gplan.interior(Ud).cpu().numpy(), oplan.interior(Uo))
                assert err <= (1e-12 if step == 0 else 1e-9), (step, err)
        results.append((gplan.interior(Ud).clone(), dts))
        fg, _ = gplan.fx_hydro_status()
        assert fg == oplan.status()[0]
    for got, dts in results[1:]:
        assert torch.equal(got, results[0][0]) and dts == results[0][1]
    gen, _, _ = gpu_plan_for(cfg, bc=bc, recon=recon, riemann=riemann, rk=rk, order=order, path=1, **kw)
    assert gen.path == 0
    A, B = Uh.cuda(), Uh.cuda()
    gplan.fx_hydro_advance(A, dxd, 1e-3)
    gen.fx_hydro_advance(B, dxd, 1e-3)
    assert rel_err(cfg, gplan.interior(A).cpu().numpy(), gen.interior(B).cpu().numpy()) <= 1e-12


def test_bundle_uniform_state_bitwise_and_determinism():
    cfg = inputs.config(5, nb=(4, 4, 4))
    cfg.block_dims = (8, 8, 8)
    gplan, neigh, coords = gpu_plan_for(cfg, order=1)
    assert gplan.path == 4
    U = torch.full(inputs.padded_shape(cfg), float("nan"), dtype=torch.float64)
    I = inputs.interior_view(cfg, U)
    for v, val in enumerate((1.3, 0.4, -0.7, 0.2, 5.9485)):
        I[v] = val
    U = U.cuda()
    U0 = gplan.interior(U).clone()
    dxd = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    for _ in range(10):
        gplan.fx_hydro_advance(U, dxd, 1e-4)
    assert torch.equal(gplan.interior(U), U0)
    Uh = inputs.embed(cfg, torch.from_numpy(random_state(cfg, 64, (8, 8, 8), 5)))
    ref = None
    for rep in range(6):
        A = Uh.cuda()
        dt = gplan.fx_hydro_compute_dt(A, dxd, 0.3).clone()
        for _ in range(3):
            gplan.fx_hydro_step(A, dxd, 0.3, dt)
        got = gplan.interior(A).clone()
        assert torch.isfinite(got).all()
        if ref is None:
            ref = got
        assert torch.equal(got, ref), rep


@pytest.mark.parametrize("nb,bc,nvars,why", [((3, 2, 2), "periodic", 5, "odd count in x"), ((2, 2, 2), "reflect", 5, "walls"),
                                              ((2, 2, 2), "periodic", 7, "passive scalars"), ((1, 2, 2), "periodic", 5, "one block wide")])
def test_plans_that_do_not_bundle_keep_their_path(nb, bc, nvars, why):
    cfg = inputs.config(5, nb=nb)
    cfg.block_dims = (8, 8, 8)
    gplan, _, _ = gpu_plan_for(cfg, bc=bc, nvars=nvars)
    assert gplan.path in (0, 2), why
