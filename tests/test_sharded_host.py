"""The sharded path's host logic with TWO gloo ranks on the CPU: the partition and the send / receive
lists of fx_shard_* (C++, no GPU needed), the meaning of an item (written out again here in numpy), the rank-to-rank
transfer (sharded.exchange_buffers, the code the GPU path runs over NCCL) and the per-stage protocol -- with the ORACLE as
each rank's engine.  Pins: the owned blocks of the two ranks after three RK2 steps, composed from the oracle's own Euler
step with an exchange before each, equal the single-domain run bit for bit; the time step is the minimum of the ranks';
every owned block's face guard zones resolve, through the ghost blocks, to the zones the single-domain index map names."""
import json
import os
import subprocess
import sys

from tests.test_multirank_host import ROOT, free_port

WORKER = r"""
import os, sys, json
sys.path.insert(0, %r)
import numpy as np, torch
import torch.distributed as dist
from oracle import fxoracle as fxo
from paper_2208_11630_b200 import binding as fx, inputs
from paper_2208_11630_b200.sharded import exchange_buffers
dist.init_process_group("gloo", rank=int(os.environ["RANK"]), world_size=int(os.environ["WORLD_SIZE"]))
rank, world = dist.get_rank(), dist.get_world_size()
dims, g, R, nb = (8, 8, 8), 2, 2, (2, 2, 4)
cfg = inputs.config(5, nb=nb); cfg.block_dims = dims; cfg.nguard = g
per = fx.TOPO_PERIODIC
neigh, coords = fx.fx_topology_cartesian(nb, [per] * 3, [per] * 3, fx.ORDER_MORTON)
N = neigh.shape[0]
sd = fx.Shard(neigh, world, rank)
# the partition covers every block exactly once
owned = torch.zeros(N, dtype=torch.int64); owned[sd.global_id[:sd.n_owned]] = 1
dist.all_reduce(owned); assert bool((owned == 1).all())
assert sd.n_ghost > 0 and len(sd.send_items) == len(sd.recv_items) > 0

def slab(plan, U, block, side):  # an item [include/fx_hydro.h]: the R-deep slab of the block's interior behind face `side`
    I = plan.interior(U)[:, block]            # [v, k, j, i]
    ax = 3 - side // 2
    n = I.shape[ax]
    sl = [slice(None)] * 4
    sl[ax] = slice(n - R, n) if side & 1 else slice(0, R)
    return I[tuple(sl)]

def exchange(plan, U):
    send = np.concatenate([slab(plan, U, b, s).ravel() for b, s in sd.send_items])
    sizes = lambda items: [slab(plan, U, b, s).size for b, s in items]
    cs, cr = np.cumsum([0] + list(sd.send_counts)), np.cumsum([0] + list(sd.recv_counts))
    ss, rs = sizes(sd.send_items), sizes(sd.recv_items)
    send_splits = [int(sum(ss[cs[p]:cs[p + 1]])) for p in range(world)]
    recv_splits = [int(sum(rs[cr[p]:cr[p + 1]])) for p in range(world)]
    sb, rb = torch.from_numpy(send.copy()), torch.empty(sum(recv_splits), dtype=torch.float64)
    exchange_buffers(sb, send_splits, rb, recv_splits, rank, world)
    o = 0
    for b, s in sd.recv_items:
        v = slab(plan, U, b, s)
        v[...] = rb[o:o + v.size].numpy().reshape(v.shape)
        o += v.size

def rk2(plan, U, dx, dt, ex):  # SSP-RK2 from the oracle's Euler step: U <- (U + E(E(U))) / 2, an exchange before each E
    U0 = U.copy()
    ex(plan, U); plan.euler_step(U, dx, dt)
    ex(plan, U); plan.euler_step(U, dx, dt)
    U[...] = 0.5 * U0 + 0.5 * U

Ui = inputs.block_interiors(cfg, coords).numpy()
dxg = inputs.dx_array(cfg)
# single domain
ref = fxo.OraclePlan(dims, g, N, cfg.gamma, 0, 1, 2); ref.set_topology(neigh)
Ur = np.full(ref.shape, np.nan); ref.interior(Ur)[...] = Ui
# this rank
loc = fxo.OraclePlan(dims, g, sd.n_local, cfg.gamma, 0, 1, 2); loc.set_topology(sd.neigh_local)
own = fxo.OraclePlan(dims, g, sd.n_owned, cfg.gamma, 0, 1, 2)  # for the time step of the owned blocks alone
Ul = np.full(loc.shape, np.nan); loc.interior(Ul)[:, :sd.n_owned] = Ui[:, sd.global_id[:sd.n_owned]]
dxl = np.ascontiguousarray(dxg[sd.global_id])
# face guard zones resolve to the same global zones
exchange(loc, Ul)
mg, ml = ref.index_map(), loc.index_map()
lb, off = np.divmod(ml[:sd.n_owned], loc.S_b)
as_global = sd.global_id[lb] * ref.S_b + off
k, j, i = np.meshgrid(*[np.arange(n + 2 * g) for n in dims[::-1]], indexing="ij")
outside = sum(((c < g) | (c >= g + n)).astype(int) for c, n in zip((k, j, i), dims[::-1]))
face = outside <= 1
assert np.array_equal(as_global[:, face], mg[sd.global_id[:sd.n_owned]][:, face])
dts = []
for step in range(3):
    Uo = np.full(own.shape, np.nan); own.interior(Uo)[...] = loc.interior(Ul)[:, :sd.n_owned]
    d = torch.tensor([own.compute_dt(Uo, dxl[:sd.n_owned], 0.3)], dtype=torch.float64)
    dist.all_reduce(d, op=dist.ReduceOp.MIN)
    dt = float(d.item()); dts.append(dt)
    assert dt == ref.compute_dt(Ur, dxg, 0.3)
    rk2(loc, Ul, dxl, dt, exchange)
    rk2(ref, Ur, dxg, dt, lambda p, U: None)
same = bool(np.array_equal(loc.interior(Ul)[:, :sd.n_owned], ref.interior(Ur)[:, sd.global_id[:sd.n_owned]]))
dist.barrier()
print(json.dumps({"rank": rank, "same": same, "owned": int(sd.n_owned), "ghost": int(sd.n_ghost), "dts": dts}), flush=True)
dist.destroy_process_group()
"""


def test_two_rank_partition_exchange_and_steps_equal_the_single_domain_bitwise():
    port = free_port()
    procs = []
    for rank in range(2):
        env = dict(os.environ, RANK=str(rank), WORLD_SIZE="2", MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), OMP_NUM_THREADS="2")
        procs.append(subprocess.Popen([sys.executable, "-c", WORKER % ROOT], env=env, stdout=subprocess.PIPE, stderr=subprocess.PIPE, text=True))
    res = [p.communicate(timeout=300) for p in procs]
    assert all(p.returncode == 0 for p in procs), [r[1][-2000:] for r in res]
    outs = [json.loads(r[0].strip().splitlines()[-1]) for r in res]
    assert all(o["same"] for o in outs)
    assert outs[0]["dts"] == outs[1]["dts"] and outs[0]["owned"] + outs[1]["owned"] == 16 and outs[0]["ghost"] > 0
