"""Sharded runs on ONE GPU: the ranks of a 2- and a 3-way partition are emulated in one process (every rank's plan lives on
the same device, the all_to_all is replaced by copies between the ranks' buffers), so that the pack / unpack kernels, the
owned / ghost split of the plans (FX_OPT_OWNED_BLOCKS) and the stage-by-stage API are exercised: the union of the ranks'
owned blocks after RK steps equals the single-plan result BIT FOR BIT, the time step too, and the ghost blocks are
never written by a stage.  (The rank-to-rank transfer itself is torch.distributed; the host logic is covered with two
gloo ranks in tests/test_multirank_host.py.)"""
import numpy as np
import pytest
import torch

from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for

pytestmark = pytest.mark.gpu


def run_sharded(cfg, neigh, coords, world, steps, recon, rk, guard_x, path, nvars=5):
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200.sharded import ShardedHydro
    ranks = [ShardedHydro(cfg.block_dims, cfg.nguard, cfg.gamma, recon, cfg.riemann, rk, neigh, r, world, guard_x=guard_x, nvars=nvars)
             for r in range(world)]
    for sh in ranks:
        sh.world = 1  # no process group here: transfer() is done by hand below
        if path is not None:
            assert sh.plan.path == path
    Ui = inputs.block_interiors(cfg, coords)
    if nvars > 5:
        Ui = inputs.with_scalars(cfg, coords, Ui, nvars - 5)
    Us, dxs = [], []
    dx_all = inputs.dx_array(cfg)
    for sh in ranks:
        U = sh.alloc_state(fill=float("nan"))  # ghost blocks start as NaN: only exchanged slabs are ever read
        gid = sh.shard.global_id[:sh.n_owned]
        sh.interior(U)[...] = Ui[:, gid].cuda()
        Us.append(U)
        dxl = np.ascontiguousarray(dx_all[sh.shard.global_id])
        dxs.append(torch.from_numpy(dxl).cuda())

    def exchange(stage):
        for sh, U in zip(ranks, Us):
            X, _ = sh.plan.fx_hydro_stage_arrays(U, stage)
            sh.pack(X)
        torch.cuda.synchronize()
        for q, sh in enumerate(ranks):  # what all_to_all_single does: rank q's piece of p's send buffer, in rank order
            ro = 0
            for p, src in enumerate(ranks):
                n = sh.recv_splits[p]
                so = sum(src.send_splits[:q])
                assert n == src.send_splits[q]
                sh.recv_buf[ro:ro + n] = src.send_buf[so:so + n]
                ro += n
        for sh, U in zip(ranks, Us):
            X, _ = sh.plan.fx_hydro_stage_arrays(U, stage)
            sh.unpack(X)

    def global_min(dts):
        m = torch.stack(dts).min()
        for d in dts:
            d.copy_(m)

    dts = [sh.plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone() for sh, U, dx in zip(ranks, Us, dxs)]
    global_min(dts)
    history = [float(dts[0].item())]
    for _ in range(steps):
        for s in range(rk):
            exchange(s)
            for sh, U, dx, dt in zip(ranks, Us, dxs, dts):
                if s == rk - 1:
                    sh.plan.fx_hydro_advance_stage(U, dx, dt, s, cfl_next=cfg.cfl, dt_next=dt)
                else:
                    sh.plan.fx_hydro_advance_stage(U, dx, dt, s)
        global_min(dts)
        history.append(float(dts[0].item()))
    out = torch.empty((nvars,) + tuple(Ui.shape[1:]), dtype=torch.float64)
    for sh, U in zip(ranks, Us):
        out[:, sh.shard.global_id[:sh.n_owned]] = sh.interior(U).cpu()
    return out, history, ranks, Us


def test_sharded_with_passive_scalars_equals_single_plan():
    """Passive scalars in a sharded plan on the fused kernel + scalar pass: a zone's high-face data behind a cut are not the
    ghost block's (nobody computes those) but the fused kernel's own solve of that face, left in P.fqb -- owned blocks and
    time steps equal the single plan's bit for bit.  (The first sharded run with scalars had read the ghost block's.)"""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 4))
    bcs = [fx.TOPO_PERIODIC] * 3
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    got, hist, ranks, Us = run_sharded(cfg, neigh, coords, 2, 3, 0, 2, 4, 1, nvars=7)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, 0, cfg.riemann, 2, nvars=7)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    U = plan.alloc_state(fill=float("nan"))
    plan.interior(U)[...] = inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), 2).cuda()
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    ref_hist = [float(dt.item())]
    for _ in range(3):
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)
        ref_hist.append(float(dt.item()))
    assert plan.path == 1 and hist == ref_hist
    assert torch.equal(got, plan.interior(U).cpu())


@pytest.mark.parametrize("number,nb,block,recon,rk,guard_x,world,path", [
    (5, (2, 2, 4), None, 0, 2, 8, 2, 1), (5, (4, 2, 2), None, 1, 3, 4, 3, 1), (5, (2, 2, 2), (8, 8, 8), 0, 2, 4, 2, 4),
    (5, (2, 2, 2), (8, 8, 8), 1, 3, 4, 2, 4), (5, (3, 2, 2), (8, 8, 8), 0, 2, 4, 2, 0), (2, (4, 4, 1), None, 0, 2, 4, 3, 2)])
def test_sharded_equals_single_plan_bitwise(number, nb, block, recon, rk, guard_x, world, path):
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(number, nb=nb)
    if block:
        cfg.block_dims = block
    bcs = [fx.TOPO_PERIODIC if cfg.block_dims[d] > 1 else fx.TOPO_NONE for d in range(3)]
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    steps = 3
    got, hist, ranks, Us = run_sharded(cfg, neigh, coords, world, steps, recon, rk, guard_x, path)
    # single plan, same order, same layout
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, recon, cfg.riemann, rk)
    if guard_x != cfg.nguard:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    assert plan.path == path
    U = plan.alloc_state(fill=float("nan"))
    plan.interior(U)[...] = inputs.block_interiors(cfg, coords).cuda()
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    ref_hist = [float(dt.item())]
    for _ in range(steps):
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)
        ref_hist.append(float(dt.item()))
    assert hist == ref_hist
    assert torch.equal(got, plan.interior(U).cpu())
    # every rank has ghosts, they were never written by a stage beyond the exchanged slabs (their cores are still NaN
    # where no slab reaches: blocks of 16 with slabs of depth 2 or 3 from at most both sides of each dimension)
    for sh, Ur in zip(ranks, Us):
        assert sh.shard.n_ghost > 0
        if cfg.block_dims[0] == 16:
            core = sh.plan.interior(Ur)[:, sh.n_owned:, 4:12 if cfg.block_dims[2] > 1 else 0:1, 4:12, 4:12]
            assert torch.isnan(core).all()


@pytest.mark.parametrize("recon,rk,guard_x", [(0, 2, 8), (1, 3, 4)])
def test_stage_in_two_parts_inner_reads_no_ghost(recon, rk, guard_x):
    """fx_hydro_advance_stage_part: FX_PART_INNER runs BEFORE the exchange with every ghost block of the stage input full of
    NaN, FX_PART_BOUNDARY after it; the union of the ranks' owned blocks still equals the single plan bit for bit, and so
    does the time step (the fused reduction is finalised by the stage's last CTA, whichever launch it is in).  The tiling is
    cut in y with outflow there, so that each rank has blocks away from the cut."""
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200.sharded import ShardedHydro
    cfg = inputs.config(5, nb=(4, 4, 2))
    bcs = [fx.TOPO_PERIODIC, fx.TOPO_OUTFLOW, fx.TOPO_PERIODIC]
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    world, steps = 2, 3
    ranks = [ShardedHydro(cfg.block_dims, cfg.nguard, cfg.gamma, recon, cfg.riemann, rk, neigh, r, world, guard_x=guard_x) for r in range(world)]
    Ui = inputs.block_interiors(cfg, coords)
    dx_all = inputs.dx_array(cfg)
    Us, dxs = [], []
    for sh in ranks:
        sh.world = 1
        assert sh.plan.path == 1
        ni, nbd = sh.plan.fx_hydro_plan_stage_parts()
        assert ni > 0 and nbd > 0 and ni + nbd == sh.n_owned
        U = sh.alloc_state(fill=float("nan"))
        sh.interior(U)[...] = Ui[:, sh.shard.global_id[:sh.n_owned]].cuda()
        Us.append(U)
        dxs.append(torch.from_numpy(np.ascontiguousarray(dx_all[sh.shard.global_id])).cuda())
    dts = [sh.plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone() for sh, U, dx in zip(ranks, Us, dxs)]
    m = torch.stack(dts).min()
    for d in dts:
        d.copy_(m)
    hist = [float(m.item())]
    for _ in range(steps):
        for s in range(rk):
            last = s == rk - 1
            kw = [dict(cfl_next=cfg.cfl, dt_next=dt) if last else {} for dt in dts]
            for sh, U, dx, dt, k in zip(ranks, Us, dxs, dts, kw):
                X, _ = sh.plan.fx_hydro_stage_arrays(U, s)
                # poison the ghost blocks of the stage's input (the array at X: U itself or a stage copy inside the workspace)
                if X == U.data_ptr():
                    view = U
                else:
                    ws = sh.plan._ws
                    off = X - ws.data_ptr()
                    assert 0 < off < ws.numel() and off % 8 == 0
                    view = ws[off:off + U.numel() * 8].view(torch.float64).view(U.shape)
                view[:, sh.n_owned:] = float("nan")
                sh.plan.fx_hydro_advance_stage_part(U, dx, dt, s, fx.PART_INNER, **k)
            for sh, U in zip(ranks, Us):
                X, _ = sh.plan.fx_hydro_stage_arrays(U, s)
                sh.pack(X)
            torch.cuda.synchronize()
            for q, sh in enumerate(ranks):
                ro = 0
                for p, src in enumerate(ranks):
                    n = sh.recv_splits[p]
                    so = sum(src.send_splits[:q])
                    sh.recv_buf[ro:ro + n] = src.send_buf[so:so + n]
                    ro += n
            for sh, U, dx, dt, k in zip(ranks, Us, dxs, dts, kw):
                X, _ = sh.plan.fx_hydro_stage_arrays(U, s)
                sh.unpack(X)
                sh.plan.fx_hydro_advance_stage_part(U, dx, dt, s, fx.PART_BOUNDARY, **k)
        m = torch.stack(dts).min()
        for d in dts:
            d.copy_(m)
        hist.append(float(m.item()))
    got = torch.empty((5,) + tuple(Ui.shape[1:]), dtype=torch.float64)
    for sh, U in zip(ranks, Us):
        got[:, sh.shard.global_id[:sh.n_owned]] = sh.interior(U).cpu()
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, recon, cfg.riemann, rk)
    if guard_x != cfg.nguard:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    U = plan.alloc_state(fill=float("nan"))
    plan.interior(U)[...] = Ui.cuda()
    dx = torch.from_numpy(dx_all).cuda()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    ref_hist = [float(dt.item())]
    for _ in range(steps):
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)
        ref_hist.append(float(dt.item()))
    assert hist == ref_hist
    assert torch.equal(got, plan.interior(U).cpu())


def test_overlapped_step_of_two_ranks_in_two_threads():
    """ShardedHydro.step as the ranks run it -- the exchange on a stream of its own beside FX_PART_INNER, FX_PART_BOUNDARY behind
    the event -- with the two ranks of a partition driven by two host threads on this GPU (the rank-to-rank transfer and the
    time-step minimum are replaced by copies between the ranks' buffers at a host barrier; no kernel waits for another
    rank's): bit for bit the single plan's result and time steps."""
    import threading
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200.sharded import ShardedHydro
    cfg = inputs.config(5, nb=(4, 4, 2))
    bcs = [fx.TOPO_PERIODIC, fx.TOPO_OUTFLOW, fx.TOPO_PERIODIC]
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON)
    world, steps = 2, 4
    ranks = [ShardedHydro(cfg.block_dims, cfg.nguard, cfg.gamma, 0, cfg.riemann, 2, neigh, r, world, guard_x=8) for r in range(world)]
    assert all(sh.overlap for sh in ranks)
    Ui = inputs.block_interiors(cfg, coords)
    dx_all = inputs.dx_array(cfg)
    bar = threading.Barrier(world)
    shared_dt = [None] * world

    def make_transfer(q):
        sh = ranks[q]

        def transfer():
            torch.cuda.current_stream().synchronize()  # this rank's pack (on its exchange stream) is done
            bar.wait()
            ro = 0
            for p, src in enumerate(ranks):
                n = sh.recv_splits[p]
                so = sum(src.send_splits[:q])
                sh.recv_buf[ro:ro + n].copy_(src.send_buf[so:so + n])
                ro += n
            torch.cuda.current_stream().synchronize()
            bar.wait()  # nobody packs the next stage before everybody has copied this one
        return transfer

    def make_min(q):
        def global_min(dt):
            torch.cuda.synchronize()
            shared_dt[q] = float(dt.item())
            bar.wait()
            dt.fill_(min(shared_dt))
            bar.wait()
            return dt
        return global_min

    results, hists, errors = [None] * world, [None] * world, []

    def run(q):
        try:
            sh = ranks[q]
            sh.transfer, sh._global_min = make_transfer(q), make_min(q)
            with torch.cuda.stream(torch.cuda.Stream()):
                U = sh.alloc_state(fill=float("nan"))
                sh.interior(U)[...] = Ui[:, sh.shard.global_id[:sh.n_owned]].cuda()
                dx = torch.from_numpy(np.ascontiguousarray(dx_all[sh.shard.global_id])).cuda()
                dt = sh.compute_dt(U, dx, cfg.cfl)
                hist = [float(dt.item())]
                for _ in range(steps):
                    sh.step(U, dx, cfg.cfl, dt)
                    hist.append(float(dt.item()))
                torch.cuda.synchronize()
                results[q], hists[q] = sh.interior(U).cpu(), hist
        except Exception as e:  # a failing rank must not leave the other at the barrier
            errors.append(e)
            bar.abort()

    threads = [threading.Thread(target=run, args=(q,)) for q in range(world)]
    for t in threads:
        t.start()
    for t in threads:
        t.join(timeout=120)
    assert not errors, errors
    got = torch.empty((5,) + tuple(Ui.shape[1:]), dtype=torch.float64)
    for sh, r in zip(ranks, results):
        got[:, sh.shard.global_id[:sh.n_owned]] = r
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, 0, cfg.riemann, 2)
    plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, 8)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    U = plan.alloc_state(fill=float("nan"))
    plan.interior(U)[...] = Ui.cuda()
    dx = torch.from_numpy(dx_all).cuda()
    dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()
    ref_hist = [float(dt.item())]
    for _ in range(steps):
        plan.fx_hydro_step(U, dx, cfg.cfl, dt)
        ref_hist.append(float(dt.item()))
    assert hists[0] == ref_hist and hists[1] == ref_hist
    assert torch.equal(got, plan.interior(U).cpu())


@pytest.mark.parametrize("number,nb,block,recon,path", [(5, (2, 2, 2), None, 0, 1), (5, (2, 2, 2), (8, 8, 8), 1, 4), (2, (2, 2, 1), None, 0, 2),
                                                        (5, (2, 2, 2), (6, 5, 4), 0, 0)])
def test_stage_parts_on_every_path_equal_the_whole_stage(number, nb, block, recon, path):
    """fx_hydro_advance_stage_part on a plan of its own (no ghost block: everything is 'inner' on the fused path) and on the
    paths that are not split (FX_PART_INNER does nothing, FX_PART_BOUNDARY is the stage): both parts = fx_hydro_advance_stage."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(number, nb=nb)
    if block:
        cfg.block_dims = block
    n = cfg.nb[0] * cfg.nb[1] * cfg.nb[2]
    a, neigh, coords = gpu_plan_for(cfg, recon=recon, rk=2)
    b, _, _ = gpu_plan_for(cfg, recon=recon, rk=2)
    assert a.path == path
    ni, nbd = a.fx_hydro_plan_stage_parts()
    assert (ni, nbd) == ((n, 0) if path == 1 else (0, n))
    Uh = inputs.embed(cfg, inputs.block_interiors(cfg, coords))
    Ua, Ub = Uh.cuda(), Uh.cuda()
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dta, dtb = a.fx_hydro_compute_dt(Ua, dx, cfg.cfl).clone(), b.fx_hydro_compute_dt(Ub, dx, cfg.cfl).clone()
    for _ in range(2):
        for s in range(2):
            kwa = dict(cfl_next=cfg.cfl, dt_next=dta) if s == 1 else {}
            kwb = dict(cfl_next=cfg.cfl, dt_next=dtb) if s == 1 else {}
            a.fx_hydro_advance_stage(Ua, dx, dta, s, **kwa)
            b.fx_hydro_advance_stage_part(Ub, dx, dtb, s, fx.PART_BOUNDARY if s == 0 else fx.PART_INNER, **kwb)  # either order
            b.fx_hydro_advance_stage_part(Ub, dx, dtb, s, fx.PART_INNER if s == 0 else fx.PART_BOUNDARY, **kwb)
    assert torch.equal(dta, dtb) and torch.equal(a.interior(Ua), b.interior(Ub))
    with pytest.raises(fx.FxError):
        b.fx_hydro_advance_stage_part(Ub, dx, dtb, 0, 3)
