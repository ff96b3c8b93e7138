"""Refinement jumps at the size and in the launch configuration `bench.py --amr` times (config 5's domain as 16^3 coarse blocks,
the central 8^3 of them refined: 7680 blocks of 16^3 zones, 1736 with a jump face; Morton order, wide layout, fx_hydro_step):
the fused path (fx_hydro_plan_path = 5) against the all-generic path on every zone, conservation of the volume-weighted
totals through the jumps [B14], and the status word.  (The oracle checks the same path element by element on the small
two-level grids of tests/test_gpu_amr_hybrid.py; here the properties that hold at any size.)"""
import types

import numpy as np
import pytest
import torch

pytestmark = pytest.mark.gpu


def test_full_size_two_level_grid_fused_against_generic_and_conservation():
    import bench
    from tests.helpers import rel_err
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 40e9:
        pytest.skip("needs 40 GB of free HBM")
    base = dict(order="morton", guard_x=-1, zchain=0)
    cfg, plan, U, dx, _ = bench.build_amr_workload(types.SimpleNamespace(path=0, **base), torch.device("cuda:0"))
    _, gen, V, _, _ = bench.build_amr_workload(types.SimpleNamespace(path=1, **base), torch.device("cuda:0"))
    assert plan.path == 5 and gen.path == 0 and plan.nblocks == 7680 and cfg.jump_blocks == 1736
    assert torch.equal(plan.interior(U), gen.interior(V))
    vol = (dx[:, 0] * dx[:, 1] * dx[:, 2]).view(1, -1, 1, 1, 1)  # a coarse zone is eight fine ones

    def totals(P, A):
        return [float((P.interior(A)[v:v + 1] * vol).sum(dtype=torch.float64)) for v in range(5)]

    T0 = totals(plan, U)
    dt, dtg = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone(), gen.fx_hydro_compute_dt(V, dx, cfg.cfl).clone()
    assert torch.equal(dt, dtg)

    class G:
        gamma = cfg.gamma
    for step in range(2):
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)
        gen.fx_hydro_step(V, dx, cfg.cfl, dtg)
        a, b = plan.interior(U), gen.interior(V)
        worst = 0.0
        for b0 in range(0, plan.nblocks, 1920):  # (the error metric A21 block range by block range: it runs on the host)
            worst = max(worst, rel_err(G, a[:, b0:b0 + 1920].cpu().numpy(), b[:, b0:b0 + 1920].cpu().numpy()))
        assert worst <= (1e-12 if step == 0 else 1e-11), (step, worst)
        assert abs(float(dt.item()) - float(dtg.item())) <= 1e-13 * float(dtg.item())
    T1 = totals(plan, U)
    scale = [T0[0], 2.4 * T0[0], 2.4 * T0[0], 2.4 * T0[0], T0[4]]
    for v in range(5):
        assert abs(T1[v] - T0[v]) <= 1e-13 * scale[v], (v, T1[v] - T0[v], scale[v])
    flags, _ = plan.fx_hydro_status()
    assert not (flags & 1)
    del U, V, plan, gen
    torch.cuda.empty_cache()
