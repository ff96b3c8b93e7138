"""Sharded runs: one process per GPU, each advancing a contiguous run of the block order (DESIGN.md
section 8).  Argument marshalling and torch.distributed plumbing only: the partition is fx_shard_* (C++), the stages,
the CFL reduction and the pack / unpack of the cut-face slabs are kernels of libfxhydro.so, the bytes cross NVLink in
one grouped batch of torch.distributed sends and receives (NCCL) per RK stage and the time step in one 8-byte all_reduce(MIN) per step.

    sh = ShardedHydro(block_dims, nguard, gamma, recon, riemann, rk, neigh_global, rank, world)
    U = sh.alloc_state(); sh.interior(U)[...] = <this rank's owned blocks, sh.shard.global_id[:sh.n_owned]>
    dt = sh.compute_dt(U, dx, cfl)            # device scalar, the minimum over all ranks
    sh.step(U, dx, cfl, dt)                   # all RK stages; dt <- the next global time step

The ghost blocks of U need no initial data: every stage input's ghost slabs are exchanged before the stage runs.
"""
from __future__ import annotations

import numpy as np
import torch

from . import binding as fx


def exchange_buffers(send_buf, send_splits, recv_buf, recv_splits, rank, world, group=None):
    """Rank-to-rank transfer of the packed slabs: piece p of send_buf (send_splits[p] elements, in rank order) goes to rank
    p, piece p of recv_buf comes from rank p -- one grouped batch of point-to-point sends and receives (ncclSend / ncclRecv
    inside one group on GPUs: every peer is one NVLink hop through the switch; gloo on the CPU in the tests)."""
    import torch.distributed as dist
    ops, so, ro = [], 0, 0
    for p in range(world):
        ns, nr = send_splits[p], recv_splits[p]
        if p != rank and nr:
            ops.append(dist.P2POp(dist.irecv, recv_buf[ro:ro + nr], p, group))
        if p != rank and ns:
            ops.append(dist.P2POp(dist.isend, send_buf[so:so + ns], p, group))
        so += ns
        ro += nr
    if ops:
        for w in dist.batch_isend_irecv(ops):
            w.wait()


class ShardedHydro:
    def __init__(self, block_dims, nguard, gamma, recon, riemann, rk_order, neigh_global, rank, world, device="cuda",
                 guard_x=None, nvars=5, group=None, zchain=None, wavespeed=None, overlap=True):
        self.rank, self.world, self.group = rank, world, group
        self.shard = fx.Shard(neigh_global, world, rank)
        sd = self.shard
        self.n_owned, self.n_local = sd.n_owned, sd.n_local
        self.plan = fx.HydroPlan(block_dims, nguard, sd.n_local, gamma, recon, riemann, rk_order, nvars=nvars, device=device)
        self.plan.fx_hydro_plan_set_option(fx.OPT_OWNED_BLOCKS, sd.n_owned)
        if guard_x is not None and guard_x != nguard:
            self.plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
        if zchain:
            self.plan.fx_hydro_plan_set_option(fx.OPT_ZCHAIN, zchain)
        if wavespeed:
            self.plan.fx_hydro_plan_set_option(fx.OPT_WAVESPEED, wavespeed)
        self.plan.fx_hydro_plan_set_topology(sd.neigh_local)
        self.plan.fx_hydro_plan_set_workspace()
        self.rk_order = rk_order
        dev = self.plan.device
        elems = [self.plan.fx_halo_item_elems(s) for s in range(6)]

        def side(items, counts):
            sizes = np.array([elems[s] for s in items[:, 1]], np.int64)
            offsets = np.concatenate([[0], np.cumsum(sizes)[:-1]]).astype(np.int64) if len(sizes) else np.zeros(0, np.int64)
            bounds = np.concatenate([[0], np.cumsum(counts)]).astype(np.int64)
            splits = [int(sizes[bounds[p]:bounds[p + 1]].sum()) for p in range(world)]  # elements per peer
            return (torch.from_numpy(np.ascontiguousarray(items)).to(dev), torch.from_numpy(offsets).to(dev),
                    torch.empty(max(int(sizes.sum()), 1), dtype=torch.float64, device=dev), splits, int(sizes.sum()))

        self.send_items, self.send_offsets, self.send_buf, self.send_splits, self.send_elems = side(sd.send_items, sd.send_counts)
        self.recv_items, self.recv_offsets, self.recv_buf, self.recv_splits, self.recv_elems = side(sd.recv_items, sd.recv_counts)
        # a stage in two parts, the exchange on a stream of its own beside the first (fused kernel only; see step)
        inner, _ = self.plan.fx_hydro_plan_stage_parts()
        self.overlap = bool(overlap) and world > 1 and inner > 0 and torch.device(dev).type == "cuda"
        if self.overlap:
            self._comm = torch.cuda.Stream(device=dev)

    # ---- state helpers
    def alloc_state(self, fill=float("nan")):
        return self.plan.alloc_state(fill=fill)

    def interior(self, U):
        """Interior zones of the OWNED blocks [nvars, n_owned, nz, ny, nx]."""
        return self.plan.interior(U)[:, :self.n_owned]

    # ---- the exchange, in its three parts (a single-process test drives them by hand)
    def pack(self, X, stream=None):
        """Owned blocks' cut-face slabs of the array at X (tensor or device address) -> send_buf."""
        if self.send_items.shape[0]:
            self.plan.fx_halo_pack(X, self.send_items, self.send_offsets, self.send_buf, stream)

    def transfer(self):
        """send_buf -> the peers' recv_buf (exchange_buffers)."""
        if self.world > 1:
            exchange_buffers(self.send_buf, self.send_splits, self.recv_buf, self.recv_splits, self.rank, self.world, self.group)

    def unpack(self, X, stream=None):
        """recv_buf -> the ghost blocks' slabs of the array at X."""
        if self.recv_items.shape[0]:
            self.plan.fx_halo_unpack(X, self.recv_items, self.recv_offsets, self.recv_buf, stream)

    def exchange(self, X):
        self.pack(X)
        self.transfer()
        self.unpack(X)

    # ---- the path
    def _global_min(self, dt):
        if self.world > 1:
            import torch.distributed as dist
            dist.all_reduce(dt, op=dist.ReduceOp.MIN, group=self.group)
        return dt

    def compute_dt(self, U, dx, cfl):
        return self._global_min(self.plan.fx_hydro_compute_dt(U, dx, cfl).clone())

    def step(self, U, dx, cfl, dt):
        """One SSP-RK step by the device-resident dt; dt receives the next step's global CFL time step.
        Where the plan runs the fused kernel, a stage is launched in two parts (fx_hydro_advance_stage_part): the owned blocks
        that touch no ghost block on the caller's stream WHILE pack, transfer and unpack of the cut-face slabs run on a second
        stream, followed there by the blocks next to the cut -- the two launches run side by side, the second filling the SMs
        as the first drains (measured on rank 0 of an 8-way partition of config 5 x 8, alone on one GPU: 11.5 ms per step,
        against 12.3 ms with the second launch behind the first on one stream and 11.8 - 12.1 ms for undivided stages)."""
        for s in range(self.rk_order):
            X, _ = self.plan.fx_hydro_stage_arrays(U, s)
            last = s == self.rk_order - 1
            kw = dict(cfl_next=cfl, dt_next=dt) if last else {}  # the next time step comes out of the last stage
            if self.overlap:
                main = torch.cuda.current_stream(self.plan.device)
                self._comm.wait_stream(main)  # the stage's input is complete
                with torch.cuda.stream(self._comm):
                    self.exchange(X)
                    self.plan.fx_hydro_advance_stage_part(U, dx, dt, s, fx.PART_BOUNDARY, **kw)
                self.plan.fx_hydro_advance_stage_part(U, dx, dt, s, fx.PART_INNER, **kw)
                main.wait_stream(self._comm)  # the stage is complete when both launches are
            else:
                self.exchange(X)
                self.plan.fx_hydro_advance_stage(U, dx, dt, s, **kw)
        return self._global_min(dt)
