"""The sharded path at the size and in the launch configuration `bench.py --gpus 8` gives one rank: rank 0 of an 8-way
partition of the 64^3-block tiling (32 768 owned blocks of 16^3 and 6144 ghost blocks, Morton order, wide layout), alone on
this GPU.  A stage launched in two parts side by side on two streams -- as ShardedHydro.step launches it -- equals the
undivided stage bit for bit, time step included, and no stage writes a ghost block."""
import types

import pytest
import torch

pytestmark = pytest.mark.gpu


def test_rank0_of_8_two_part_stage_equals_the_whole_stage_bitwise():
    import bench
    from paper_2208_11630_b200 import binding as fx
    torch.cuda.empty_cache()
    free, _ = torch.cuda.mem_get_info()
    if free < 110e9:
        pytest.skip("needs 110 GB of free HBM")
    args = types.SimpleNamespace(config=5, nb=None, block=None, order="morton", guard_x=-1, scalars=0, zchain=0, wavespeed=0,
                                 no_overlap=False)
    cfg, sh, U, dx = bench.build_sharded_workload(args, torch.device("cuda:0"), 0, 8)[:4]
    plan = sh.plan
    inner, boundary = plan.fx_hydro_plan_stage_parts()
    assert (sh.n_owned, sh.shard.n_ghost, inner, boundary) == (32768, 6144, 27000, 5768) and sh.overlap
    # ghost blocks: this rank's own slabs stand in for the peers' (same bytes, same shapes)
    n = min(sh.send_elems, sh.recv_elems)
    X, _ = plan.fx_hydro_stage_arrays(U, 0)
    sh.pack(X)
    sh.recv_buf[:n].copy_(sh.send_buf[:n])
    sh.unpack(X)
    ghosts0 = plan.interior(U)[:, sh.n_owned:].clone()
    V = U.clone()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    dtv = dt.clone()
    side, main = torch.cuda.Stream(), torch.cuda.current_stream()
    assert cfg.rk_order == 2
    plan.fx_hydro_advance_stage(U, dx, dt, 0)
    # (the plan holds ONE set of stage copies: run the undivided step on U to its end, then the two-part step on V)
    plan.fx_hydro_advance_stage(U, dx, dt, 1, cfl_next=cfg.cfl, dt_next=dt)
    torch.cuda.synchronize()
    for s in range(cfg.rk_order):
        kwv = dict(cfl_next=cfg.cfl, dt_next=dtv) if s == cfg.rk_order - 1 else {}
        side.wait_stream(main)
        with torch.cuda.stream(side):
            plan.fx_hydro_advance_stage_part(V, dx, dtv, s, fx.PART_BOUNDARY, **kwv)
        plan.fx_hydro_advance_stage_part(V, dx, dtv, s, fx.PART_INNER, **kwv)
        main.wait_stream(side)
    torch.cuda.synchronize()
    assert torch.equal(dt, dtv)
    assert torch.equal(plan.interior(U)[:, :sh.n_owned], plan.interior(V)[:, :sh.n_owned])
    bits = lambda t: t.contiguous().view(torch.int64)  # (the ghost blocks' cores are NaN: compare bit patterns)
    assert torch.equal(bits(plan.interior(U)[:, sh.n_owned:]), bits(ghosts0)) and torch.equal(bits(plan.interior(V)[:, sh.n_owned:]), bits(ghosts0))
    flags, _ = plan.fx_hydro_status()
    assert not (flags & 1)
    del U, V, ghosts0, sh, plan
    torch.cuda.empty_cache()
