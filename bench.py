#!/usr/bin/env python
"""bench.py -- throughput of the batched block Euler update on B200 (one JSON line on stdout).

A "step" is one pass of the whole hot path over the workload: fx_hydro_step = all RK stages (a1..a6) with the
device-resident dt, and the CFL reduction (a7) of the advanced state, which the fused path forms inside the last
stage; the first dt comes from fx_hydro_compute_dt before the warm-up.  Metric: hydro zone-updates/s per RK
stage = interior zones x stages / time.  Workload at N = 1: BASELINE.json configs[4] (32768 blocks of 16^3,
PLM-minmod + HLLC, SSP-RK2; 24.2 GB per state copy in the wide layout bench.py picks for 16-wide blocks
(--guard-x, FX_OPT_GUARD_X; 18.1 GB in the compact one), far larger than the 126 MB L2, so nothing is served
from cache between timed iterations).  e2e: the same step through fx_hydro_advance_host_interior, the host
holding the interior zones in a pinned buffer (5.37 GB each way per step inside the timed region).  N > 1 (weak scaling):
the config's tiling grown N-fold (z, then y, then x doubled), cut into N contiguous Morton runs, one per rank
(paper_2208_11630_b200/sharded.py): before every stage the cut-face slabs of its input are packed,
exchanged (grouped NCCL send/recv) and unpacked into ghost blocks; dt is the all-reduced minimum.  Started plainly with
--gpus N (no WORLD_SIZE in the environment) bench.py launches its N ranks itself.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 5] [--nb a,b,c]

--impl reference times the CPU oracle (oracle/) on the box's host cores on a bounded sample of the same
workload; it is a deliberately slow program, reported as a baseline, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "hydro zone-updates/s per RK stage (fp64)"
UNIT = "zone-updates/s"
FP64_FMA_LANES_PER_SM = 64  # 64 DFMA lanes per SM (a warp-wide fp64 instruction per 2 cycles per sub-partition, measured)


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--nb", default=None, help="override blocks per dimension, e.g. 16,16,16")
    ap.add_argument("--block", default=None, help="override zones per block and dimension, e.g. 8,8,8 (with --nb 64,64,64: config 5's field "
                    "on 8^3 blocks; not a BASELINE config: the small-block workload of the tile kernel)")
    ap.add_argument("--path", type=int, default=0, help="FX_OPT_PATH: 0 auto (fused TMA stage kernel when supported), 1 generic, 2 tile, 3 the fused kernel's two-zones-per-thread variant")
    ap.add_argument("--zchain", type=int, default=0, help="FX_OPT_ZCHAIN: z-neighbour blocks per CTA of the fused kernel (0 = library default)")
    ap.add_argument("--guard-x", type=int, default=-1, help="FX_OPT_GUARD_X: x guard depth (layout); -1 = 8 for 16-wide blocks with 4 guard zones "
                    "(256-byte row pitch, interior rows on 128-byte lines), else the config's nguard")
    ap.add_argument("--order", default="morton", choices=["lex", "morton"])
    ap.add_argument("--scalars", type=int, default=0, help="passive mass scalars carried with the 5 hydro variables (DESIGN.md B11; "
                    "nvars = 5 + this; generic path)")
    ap.add_argument("--wavespeed", type=int, default=0, help="FX_OPT_WAVESPEED: 0 Einfeldt (the reading the configs are run with [A8]), 1 Davis")
    ap.add_argument("--shard", action="store_true", help="drive the step through ShardedHydro even on one rank (the N > 1 code path with an "
                    "empty exchange; N > 1 always uses it)")
    ap.add_argument("--one-rank-of", type=int, default=0, metavar="N", help="rank 0 of an N-way partition of the N-fold tiling, ALONE on this GPU: "
                    "its stage launches (two parts side by side), pack and unpack as the rank runs them, the transfer replaced by a device "
                    "copy of the same bytes and the dt all-reduce left out -- what one rank's kernels cost, not a multi-GPU measurement")
    ap.add_argument("--no-overlap", action="store_true", help="sharded runs: the exchange in front of an undivided stage instead of beside its first part")
    ap.add_argument("--amr", action="store_true", help="two-level grid of 16^3 blocks on config 5's domain (7680 blocks, 1736 of them with a "
                    "refinement jump): the fused kernel on every block (path 5; the blocks at the jumps read their own guard zones); --path 1 for all-generic")
    ap.add_argument("--ca", action="store_true", help="time the communication-avoiding step (fx_hydro_advance_ca, DESIGN.md B17: one guard fill "
                    "per step, generic kernels on a shrinking extension of the interior) + fx_hydro_compute_dt instead of fx_hydro_step")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=2)
    return ap.parse_args()


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.05] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0]))
                smax = float(f[1])
            except Exception:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(x: float, world: int, device="cpu") -> float:
    """Max of a per-rank scalar over all ranks (the multi-GPU timing rule); identity for one rank."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(zones_per_rank: int, stages: int, steps: int, ms_max: float, world: int) -> float:
    """Weak scaling: every rank advances its own share (equal shares of the grown tiling); value = all zone-updates / max time."""
    return world * zones_per_rank * stages * steps / (ms_max * 1e-3)


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def build_workload(args, device):
    """Config, plan, state resident in HBM (generated on the device), dx."""
    import torch
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200 import inputs
    nb = tuple(int(x) for x in args.nb.split(",")) if args.nb else None
    cfg = inputs.config(args.config, nb=nb)
    if args.block:
        import dataclasses
        cfg = dataclasses.replace(cfg, block_dims=tuple(int(x) for x in args.block.split(",")))
    order = fx.ORDER_MORTON if args.order == "morton" else fx.ORDER_LEX
    code = fx.TOPO_PERIODIC if cfg.bc == "periodic" else fx.TOPO_OUTFLOW
    bcs = [code if cfg.block_dims[d] > 1 else fx.TOPO_NONE for d in range(3)]
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, order)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order,
                        nvars=5 + args.scalars, device=device)
    plan.fx_hydro_plan_set_option(fx.OPT_PATH, args.path)
    if args.wavespeed:
        plan.fx_hydro_plan_set_option(fx.OPT_WAVESPEED, args.wavespeed)
    guard_x = args.guard_x if args.guard_x >= 0 else (8 if (cfg.block_dims[0] == 16 and cfg.nguard == 4) else cfg.nguard)
    if guard_x != cfg.nguard:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
    if args.zchain:
        plan.fx_hydro_plan_set_option(fx.OPT_ZCHAIN, args.zchain)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    U = plan.alloc_state(fill=float("nan"))  # interior rows on 128-byte lines where the pitch allows it
    Ui = plan.interior(U)
    chunk = 1024
    for b0 in range(0, cfg.nblocks, chunk):
        b1 = min(cfg.nblocks, b0 + chunk)
        Ui[:, b0:b1] = inputs.with_scalars(cfg, coords[b0:b1], inputs.block_interiors(cfg, coords[b0:b1], device), args.scalars)
    dx = torch.from_numpy(inputs.dx_array(cfg)).to(device)
    return cfg, plan, U, dx, coords


AMR_NBC, AMR_LO, AMR_HI = (16, 16, 16), (4, 4, 4), (12, 12, 12)  # --amr: coarse tiling and the refined box (coarse cells)


def amr_config(inputs, nbc, nblocks):
    """What the rest of bench.py reads from a config, for the two-level workload (config 5's scheme and field)."""
    import types
    fine = inputs.config(5, nb=tuple(2 * x for x in nbc))
    return fine, types.SimpleNamespace(
        number=5, name=f"two-level grid: {nbc[0]}x{nbc[1]}x{nbc[2]} coarse blocks, the central "
                       f"{AMR_HI[0] - AMR_LO[0]}x{AMR_HI[1] - AMR_LO[1]}x{AMR_HI[2] - AMR_LO[2]} of them refined 2x (config 5's field and scheme)",
        block_dims=fine.block_dims, nguard=fine.nguard, nb=nbc, bc="periodic", gamma=fine.gamma, recon=fine.recon,
        riemann=fine.riemann, rk_order=fine.rk_order, cfl=fine.cfl, nblocks=nblocks, ndim=3,
        interior_zones=nblocks * fine.block_dims[0] * fine.block_dims[1] * fine.block_dims[2])


def build_amr_workload(args, device):
    """--amr: a static two-level grid [DESIGN.md B12-B14] of 16^3 blocks on config 5's domain: 512^3 zones inside the refined
    box, 256^3 outside; fine blocks hold config 5's field, coarse blocks its 2 x 2 x 2 means."""
    import numpy as np
    import torch
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200 import inputs
    order = fx.ORDER_MORTON if args.order == "morton" else fx.ORDER_LEX
    grid = inputs.two_level_tiling(AMR_NBC, AMR_LO, AMR_HI, order)
    n = len(grid["level"])
    fine, cfg = amr_config(inputs, AMR_NBC, n)
    ns = getattr(args, "scalars", 0)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, n, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order, nvars=5 + ns, device=device)
    plan.fx_hydro_plan_set_option(fx.OPT_PATH, args.path)
    guard_x = args.guard_x if args.guard_x >= 0 else 8
    if guard_x != cfg.nguard:
        plan.fx_hydro_plan_set_option(fx.OPT_GUARD_X, guard_x)
    if args.zchain:
        plan.fx_hydro_plan_set_option(fx.OPT_ZCHAIN, args.zchain)
    plan.fx_hydro_plan_set_refinement(grid["jump"])
    plan.fx_hydro_plan_set_topology(grid["neigh"])
    plan.fx_hydro_plan_set_workspace()
    U = plan.alloc_state(fill=float("nan"))
    Ui = plan.interior(U)
    for b0 in range(0, n, 512):
        b1 = min(n, b0 + 512)
        Ui[:5, b0:b1] = inputs.two_level_interiors(fine, grid, b0, b1, device)
        for s in range(ns):  # --scalars: abundances that follow the density field (a throughput workload: any smooth bounded field does)
            Ui[5 + s, b0:b1] = Ui[0, b0:b1] * (0.5 + 0.4 * torch.sin((s + 1.0) * Ui[0, b0:b1]))
    dxf = fine.dx
    dxh = np.where(grid["level"][:, None] == 1, 1.0, 2.0) * np.array(dxf)[None, :]
    cfg.jump_blocks = int((grid["neigh"] <= inputs.NEIGH_COARSER).any(axis=1).sum())
    return cfg, plan, U, torch.from_numpy(np.ascontiguousarray(dxh)).to(device), None


def shard_factors(world):
    """How the config's tiling grows with the number of ranks (weak scaling): powers of two double z, then y, then x."""
    f, d, w = [1, 1, 1], 2, world
    while w % 2 == 0 and w > 1:
        f[d] *= 2
        d = (d - 1) % 3
        w //= 2
    f[2] *= w  # an odd remainder goes to z
    return tuple(f)


def build_sharded_workload(args, device, rank, world):
    """N > 1: the config's tiling grown by shard_factors(world) (its field continued periodically), cut into `world`
    contiguous Morton runs, one per rank; every rank holds its run plus the ghost blocks behind its cuts."""
    import numpy as np
    import torch
    from paper_2208_11630_b200 import binding as fx
    from paper_2208_11630_b200 import inputs
    from paper_2208_11630_b200.sharded import ShardedHydro
    base = inputs.config(args.config, nb=tuple(int(x) for x in args.nb.split(",")) if args.nb else None)
    f = shard_factors(world)
    cfg = inputs.config(args.config, nb=tuple(base.nb[d] * f[d] for d in range(3)))
    if args.block:
        import dataclasses
        cfg = dataclasses.replace(cfg, block_dims=tuple(int(x) for x in args.block.split(",")))
    code = fx.TOPO_PERIODIC if cfg.bc == "periodic" else fx.TOPO_OUTFLOW
    bcs = [code if cfg.block_dims[d] > 1 else fx.TOPO_NONE for d in range(3)]
    neigh, coords = fx.fx_topology_cartesian(cfg.nb, bcs, bcs, fx.ORDER_MORTON if args.order == "morton" else fx.ORDER_LEX)
    guard_x = args.guard_x if args.guard_x >= 0 else (8 if (cfg.block_dims[0] == 16 and cfg.nguard == 4) else cfg.nguard)
    sh = ShardedHydro(cfg.block_dims, cfg.nguard, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order, neigh, rank, world, device=device,
                      guard_x=guard_x, nvars=5 + args.scalars, zchain=args.zchain, wavespeed=args.wavespeed, overlap=not args.no_overlap)
    U = sh.alloc_state(fill=float("nan"))
    gid = sh.shard.global_id
    Ui = sh.interior(U)
    for b0 in range(0, sh.n_owned, 1024):
        b1 = min(sh.n_owned, b0 + 1024)
        c = coords[gid[b0:b1]]
        Ui[:, b0:b1] = inputs.with_scalars(cfg, c, inputs.block_interiors(cfg, c, device), args.scalars)
    dx = torch.from_numpy(np.ascontiguousarray(inputs.dx_array(cfg)[:sh.n_local])).to(device)
    return cfg, sh, U, dx


# ------------------------------------------------------------------ CPU oracle legs
def oracle_sample(args, target_seconds=15.0, steps=None, steps_single=0):
    """Times the oracle as it stands on a bounded sample of the workload: a 6x6x6-block sub-tiling of the
    same field (periodic wrap of the sub-tiling), all host threads OpenMP gives it."""
    import numpy as np
    from oracle import fxoracle as fxo
    from paper_2208_11630_b200 import inputs
    full = inputs.config(args.config)
    nb = tuple(min(6, full.nb[d]) for d in range(3))
    cfg = inputs.config(args.config, nb=nb)
    code = fxo.TOPO_PERIODIC if cfg.bc == "periodic" else fxo.TOPO_OUTFLOW
    bcs = [code if cfg.block_dims[d] > 1 else fxo.TOPO_NONE for d in range(3)]
    neigh, coords = fxo.topology_cartesian(cfg.nb, bcs, bcs, fxo.ORDER_LEX)
    plan = fxo.OraclePlan(cfg.block_dims, cfg.nguard, cfg.nblocks, cfg.gamma, cfg.recon, cfg.riemann, cfg.rk_order,
                          nvars=5 + args.scalars)
    plan.set_topology(neigh)
    U = inputs.embed(cfg, inputs.with_scalars(cfg, coords, inputs.block_interiors(cfg, coords), args.scalars)).numpy()
    dx = inputs.dx_array(cfg)
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)

    def one_step():
        t = time.perf_counter()
        dt = plan.compute_dt(U, dx, cfg.cfl)
        (plan.advance_ca if getattr(args, "ca", False) else plan.advance)(U, dx, dt)
        return time.perf_counter() - t

    t_first = one_step()  # also the warm-up
    if steps is None:
        steps = max(2, min(50, int(target_seconds / max(t_first, 1e-3))))
    times = [one_step() for _ in range(steps)]
    per_step = sum(times) / len(times)
    zs = cfg.interior_zones * cfg.rk_order
    single = None
    if steps_single:
        try:  # the same sample on ONE thread (SURVEY.md 8(d) asks for both figures)
            import ctypes
            gomp = ctypes.CDLL("libgomp.so.1")
            gomp.omp_set_num_threads(1)
            ts = [one_step() for _ in range(steps_single)]
            gomp.omp_set_num_threads(cores)
            single = {"value": zs / (sum(ts) / len(ts)), "unit": UNIT, "cores": 1, "steps": steps_single}
        except Exception:
            single = None
    return {"value": zs / per_step, "unit": UNIT, "cores": cores, "kind": "oracle", "single_thread": single,
            "sample": f"config {args.config} field on a {nb[0]}x{nb[1]}x{nb[2]}-block periodic sub-tiling "
                      f"({cfg.interior_zones} zones), {steps} steps of compute_dt + {'advance_ca' if getattr(args, 'ca', False) else 'advance'}, OpenMP over blocks",
            "ms_per_step": per_step * 1e3, "steps": steps}


def run_reference(args, rank, world):
    if rank != 0:
        return
    from paper_2208_11630_b200 import inputs
    cfg = inputs.config(args.config)
    # each step is one oracle step on the bounded sample; warm-up steps run first, untimed
    r = oracle_sample(args, steps=max(1, args.steps))
    line = {"impl": "reference", "metric": METRIC, "value": r["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": r["ms_per_step"], "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {args.config}: {cfg.name} (bounded sample: {r['sample']})"},
            "cpu_baseline": {"value": r["value"], "unit": UNIT, "cores": r["cores"], "kind": "oracle", "sample": r["sample"]},
            "e2e": {"value": r["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------ roofline inputs (files only; nothing under oracle/ runs here)
def aux_calls(plan, U, dx, cfg, zones, reps=5):
    """fx_hydro_compute_dt and fx_fill_guardcells, each alone: average of `reps` launches between CUDA events on the
    stream they are launched on (the state is larger than L2 at the bench sizes, so no flush), GB/s of algorithmic bytes."""
    import torch
    out = {}
    dt_tmp = torch.empty(1, dtype=torch.float64, device=U.device)
    guard_zones = plan.nblocks * (plan.np[0] * plan.np[1] * plan.np[2] - cfg.block_dims[0] * cfg.block_dims[1] * cfg.block_dims[2])
    for name, call, nbytes in (("fx_hydro_compute_dt", lambda: plan.fx_hydro_compute_dt(U, dx, cfg.cfl, dt_tmp), 40.0 * zones),
                               ("fx_fill_guardcells", lambda: plan.fx_fill_guardcells(U), 16.0 * plan.nvars * guard_zones)):
        call()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(reps):
            call()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / reps
        out[name] = {"ms": ms, "alg_bytes": nbytes, "GB/s": nbytes / (ms * 1e-3) / 1e9, "launches_timed": reps}
    return out


def algorithmic_flops(cfg, args):
    """Exact fp64 operations per zone and RK stage of this scheme from oracle/flop_counts.json, or None."""
    try:
        counts = json.load(open(os.path.join(ROOT, "oracle", "flop_counts.json")))["per_zone_stage"]
    except Exception:
        return None
    key = f"{cfg.ndim}d_{'weno5' if cfg.recon else 'plm'}_{'hllc' if cfg.riemann else 'hlle'}_rk{cfg.rk_order}"
    if args.wavespeed:
        key += "_davis"
    if cfg.ndim == 3 and cfg.block_dims == (8, 8, 8):
        key += "_8cubed"
    elif cfg.ndim == 3 and cfg.block_dims != (16, 16, 16):
        return None
    if args.scalars:
        return None  # the counts are for the five hydro variables
    return counts.get(key, {}).get("flops")


def committed_traffic(cfg, args, plan):
    """dram__bytes_read.sum + dram__bytes_write.sum per stage launch (mean over the stages of a step) from the committed
    `ncu --set full` capture of this workload and path under profiles/, read by metric name; (None, None) if there is none."""
    per_stage = 1  # captured launches that make up one stage
    if args.wavespeed or args.zchain or args.ca or args.amr:
        return None, None
    if args.block == "8,8,8" and args.nb == "64,64,32" and not args.scalars:
        name = f"r2_ncu_config{cfg.number}_8cubed_path{plan.path}_raw.csv"
    elif args.nb or args.block or plan.gd[0] != 8:
        return None, None
    elif args.scalars:
        name = f"r2_ncu_config{cfg.number}_scalars{args.scalars}_path{plan.path}_raw.csv"
        per_stage = 1 + (args.scalars + 3) // 4  # the stage kernel and one scalar-pass launch per four scalars
    else:
        name = f"r2_ncu_config{cfg.number}_path{plan.path}_raw.csv"
    path = os.path.join(ROOT, "profiles", name)
    if not os.path.exists(path):
        return None, None
    import csv
    rd = wr = None
    for row in csv.reader(open(path)):
        if not row:
            continue
        if row[0] in ("dram__bytes_read.sum", "dram__bytes_write.sum"):
            scale = {"Gbyte": 1e9, "Mbyte": 1e6, "Kbyte": 1e3, "byte": 1.0}.get(row[1], None)
            vals = [float(x) * scale for x in row[2:] if x]
            if row[0].startswith("dram__bytes_read"):
                rd = sum(vals) / len(vals)
            else:
                wr = sum(vals) / len(vals)
    if rd is None or wr is None:
        return None, None
    return (rd + wr) * per_stage, (f"profiles/{name}: dram__bytes_read.sum + dram__bytes_write.sum, mean over the captured launches"
                                    + (f" x {per_stage} launches per stage" if per_stage > 1 else ""))


# ------------------------------------------------------------------ CUDA arm
def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2208_11630_b200 import binding as fx

    fx.lib()  # fail loudly if the CUDA library is missing
    torch.cuda.set_device(local_rank)
    device = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=device)
    sh = None
    if world > 1 or args.shard or args.one_rank_of > 1:
        cfg, sh, U, dx = build_sharded_workload(args, device, rank, args.one_rank_of if args.one_rank_of > 1 else world)
        if args.one_rank_of > 1:
            n = min(sh.send_elems, sh.recv_elems)
            sh.transfer = lambda: sh.recv_buf[:n].copy_(sh.send_buf[:n])  # the slabs' bytes moved once, on the device
            sh._global_min = lambda d: d
        plan = sh.plan
        zones = sh.n_owned * cfg.block_dims[0] * cfg.block_dims[1] * cfg.block_dims[2]  # this rank's share
    else:
        cfg, plan, U, dx, coords = build_amr_workload(args, device) if args.amr else build_workload(args, device)
        zones = cfg.interior_zones
    stages = cfg.rk_order
    fused = plan.path in (1, 3, 4)
    # fused path: one launch per RK stage, the CFL reduction (a7) rides in the last one; tile and generic paths: one
    # stage kernel per stage, then the reduction pass; with passive scalars also their face fill per stage
    launches_per_step = stages if fused else (stages + 1 + (stages if args.scalars else 0))
    if args.amr:  # per stage: guard zones behind the jumps, the stage kernel (and the scalar pass), the flux correction; then the reduction pass
        launches_per_step = stages * (3 + (args.scalars + 3) // 4) + 1
    if sh is not None:
        launches_per_step += (int(sh.send_elems > 0) + int(sh.recv_elems > 0)) * stages  # pack + unpack of the cut-face slabs before every stage
        if sh.overlap:  # a stage in two launches: the blocks away from the cut beside the exchange, the others behind it
            launches_per_step += stages
        dt = sh.compute_dt(U, dx, cfg.cfl)  # the minimum over the ranks

        def step():
            sh.step(U, dx, cfg.cfl, dt)  # per stage: slab exchange, then the stage on the owned blocks; dt <- min over ranks
    elif args.ca:
        # fill (1 launch), the stages, the local re-imaging of physical boundaries after all but the last, the reduction
        launches_per_step = 1 + stages + (0 if cfg.bc == "periodic" else stages - 1) + 1
        dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()

        def step():
            plan.fx_hydro_advance_ca(U, dx, dt)          # one guard fill, then every stage without another
            plan.fx_hydro_compute_dt(U, dx, cfg.cfl, dt)  # a7 of the advanced state
    else:
        dt = plan.fx_hydro_compute_dt(U, dx, cfg.cfl).clone()  # the first step's dt; stays on the device from here on

        def step():
            plan.fx_hydro_step(U, dx, cfg.cfl, dt)  # a1..a6 with this dt, a7 of the advanced state into dt

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    plan.fx_hydro_plan_set_timing(True)
    sampler = ClockSampler(local_rank)
    sampler.start()
    time.sleep(0.3)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t0 = time.time()
    e0.record()
    for _ in range(args.steps):
        step()
    e1.record()
    barrier()
    t1 = time.time()
    clocks = sampler.stop(t0, t1)
    ms = e0.elapsed_time(e1)
    stage_ms, stage_launches = plan.fx_hydro_plan_get_timing()
    plan.fx_hydro_plan_set_timing(False)
    flags, counts = plan.fx_hydro_status()
    ms = max_over_ranks(ms, world, device)
    # whole job: every rank's owned zone-updates over the slowest rank's time (ranks own equal shares of the grown tiling)
    value = whole_job_value(zones, stages, args.steps, ms, world)

    # roofline of the dominant kernel (the stage kernel) [NS]: the slower of the minimum HBM bytes at the measured copy
    # bandwidth and the method's fp64 operations at the fp64 peak.  Both sides are ALGORITHMIC: bytes = read X (+ U0 in the
    # later stages) and write the result, 8 B per variable; flops = the exact count of the oracle built with a counting
    # number type (oracle/flop_counts.json, written by oracle/count_flops.py; + - * / sqrt compare = 1 each).
    peak, peak_src = measured_peaks()
    alg_bytes_stage = [16.0 * (5 + args.scalars)] + [24.0 * (5 + args.scalars)] * (stages - 1)
    bytes_per_zone = sum(alg_bytes_stage) / stages
    alg_bytes_per_launch = zones * bytes_per_zone
    stage_avg_ms = stage_ms / max(stage_launches, 1)
    stage_s = stage_avg_ms * 1e-3
    hbm = {"achieved": alg_bytes_per_launch / stage_s / 1e9, "peak": peak, "unit": "GB/s", "peak_source": peak_src,
           "alg_bytes_per_zone_stage": bytes_per_zone, "alg_bytes_per_launch": alg_bytes_per_launch}
    hbm["frac"] = hbm["achieved"] / peak
    props = torch.cuda.get_device_properties(device)
    sm_max_mhz = clocks.get("sm_max_mhz") or 1965.0
    # fp64 peak: SMs x 64 fp64 lanes x 2 flops (FMA) x the maximum SM clock (the guide's unit counts)
    fp64_peak = props.multi_processor_count * FP64_FMA_LANES_PER_SM * 2 * sm_max_mhz * 1e6
    flops = algorithmic_flops(cfg, args)
    fp64 = None
    if flops is not None:
        fp64 = {"achieved": zones * flops / stage_s / 1e12, "peak": fp64_peak / 1e12, "unit": "TFLOP/s",
                "peak_source": f"nominal: {props.multi_processor_count} SMs x {FP64_FMA_LANES_PER_SM} lanes x 2 x {sm_max_mhz:.0f} MHz",
                "flops_per_zone_stage": flops, "flops_source": "oracle/flop_counts.json (counting build of the oracle, no FMA)"}
        fp64["frac"] = fp64["achieved"] / fp64["peak"]
    t_hbm, t_fp = bytes_per_zone / (peak * 1e9), (flops / fp64_peak if flops is not None else 0.0)
    traffic, traffic_src = committed_traffic(cfg, args, plan)
    side = fp64 if t_fp > t_hbm else hbm
    roofline = {"bound": "alu" if side is fp64 else "hbm", "achieved": side["achieved"], "peak": side["peak"], "unit": side["unit"],
                "frac": side["frac"], "traffic": traffic, "traffic_source": traffic_src,
                "roof_ps_per_zone_stage": {"hbm": t_hbm * 1e12, "fp64": t_fp * 1e12 if flops is not None else None},
                "hbm": hbm, "fp64": fp64,
                "kernel": "generic stage kernel over the extended interior (communication-avoiding step)" if args.ca else {5: "fused stage kernel + generic stage kernel at the refinement jumps", 1: "fused stage kernel", 3: "fused stage kernel, pair variant", 4: "fused stage kernel on 2 x 2 bundles of 8 x 8 blocks", 2: "tile stage kernel", 0: "generic stage kernel"}[plan.path],
                "kernel_ms_avg": stage_avg_ms, "kernel_launches_timed": stage_launches,
                "kernel_share_of_step": stage_ms / ms if ms > 0 else None}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": max(args.warmup, 3), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config {cfg.number}: {cfg.name}, {cfg.nblocks} blocks of "
                                   f"{cfg.block_dims[0]}x{cfg.block_dims[1]}x{cfg.block_dims[2]} (+{cfg.nguard} guard), "
                                   f"{'WENO5' if cfg.recon else 'PLM-minmod'}+{'HLLC' if cfg.riemann else 'HLLE'}, SSP-RK{stages}"
                                   + (f", {args.scalars} passive mass scalars" if args.scalars else "")
                                   + (", Davis wave speeds" if args.wavespeed else ""),
                       "interior_zones": zones, "state_bytes": plan.bytes_per_state, "block_order": args.order,
                       "layout": f"x guard depth {plan.gd[0]} (row pitch {plan.S_j * 8} B), y/z guard depth {plan.gd[1]}/{plan.gd[2]}",
                       "path": "communication-avoiding step (one guard fill per step; generic kernels on the extended interior)" if args.ca else {0: "generic", 5: f"fused (TMA); the {getattr(cfg, 'jump_blocks', 0)} blocks with a refinement jump as single-block segments reading their own guard zones", 1: "fused (TMA)", 2: "tile (shared-memory block)", 3: "fused (TMA), two zones per thread", 4: "fused (TMA), 2 x 2 bundles of 8 x 8 blocks"}[plan.path], "l2": "inputs (state) larger than L2; no flush needed",
                       "multi_gpu": (f"sharded: tiling {cfg.nb[0]}x{cfg.nb[1]}x{cfg.nb[2]} blocks in {args.one_rank_of if args.one_rank_of > 1 else world} contiguous Morton runs, "
                                     f"{sh.shard.n_ghost} ghost blocks on rank 0, cut-face slabs exchanged before every stage "
                                     f"(grouped NCCL send/recv, {sh.send_elems * 8} B sent by rank 0 per stage"
                                     + (", on a stream of its own beside the stage's launch over the blocks away from the cut" if sh.overlap else "")
                                     + "), dt = all-reduce(min)"
                                     + (f"; ONE RANK OF {args.one_rank_of} ALONE on this GPU (transfer replaced by a device copy, no all-reduce): not a multi-GPU measurement" if args.one_rank_of > 1 else ""))
                       if sh is not None else "single"},
            "clocks": clocks, "gpu_launches": launches_per_step * args.steps, "roofline": roofline,
            "status_flags": flags}

    # the two calls of the boundary that are not part of the fused step, each timed alone [SURVEY 8(d)]: the CFL reduction
    # a7 (reads the 5 hydro variables of the interior zones once: 40 B per zone) and the standalone guard fill a1 (reads one
    # interior zone and writes one guard zone per guard zone and variable: 16 B per guard zone and variable)
    if sh is None and rank == 0:
        try:
            line["aux"] = aux_calls(plan, U, dx, cfg, zones)
        except Exception as ex:
            line["aux"] = {"error": repr(ex)[:200]}

    # end to end through the C ABI with HOST buffers (H2D + steps + D2H inside the timed region)
    if not args.no_e2e and sh is not None:
        try:  # H2D of the owned interiors from pinned memory, one sharded step, D2H of the result, per step
            Uh = torch.empty(tuple(sh.interior(U).shape), dtype=torch.float64, pin_memory=True)
            Uh.copy_(sh.interior(U))
            dth = torch.empty(1, dtype=torch.float64, pin_memory=True)

            def e2e_step():
                sh.interior(U).copy_(Uh, non_blocking=True)
                d = sh.compute_dt(U, dx, cfg.cfl)
                sh.step(U, dx, cfg.cfl, d)
                Uh.copy_(sh.interior(U), non_blocking=True)
                dth.copy_(d, non_blocking=True)
                torch.cuda.synchronize()

            e2e_step()
            barrier()
            tt = time.perf_counter()
            for _ in range(args.e2e_steps):
                e2e_step()
            es = max_over_ranks((time.perf_counter() - tt) / args.e2e_steps, world, device)
            line["e2e"] = {"value": world * zones * stages / es, "unit": UNIT, "h2d_bytes_per_step": Uh.numel() * 8,
                           "d2h_bytes_per_step": Uh.numel() * 8 + 8, "ms_per_step": es * 1e3, "steps": args.e2e_steps,
                           "api": "ShardedHydro: copy of the owned interiors from pinned host memory into the padded device state, "
                                  "compute_dt + step (exchange, stages, all-reduce), copy back; per rank, max over ranks"}
            del Uh
        except Exception as ex:
            line["e2e"] = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}
    elif not args.no_e2e:
        try:
            # the host holds the interior zones (guard zones carry no information): [5][nblocks][nz][ny][nx], pinned
            Uh = torch.empty(plan.interior_shape, dtype=torch.float64, pin_memory=True)
            Uh.copy_(plan.interior(U))
            dxh = dx.cpu().pin_memory()
            stage_dev, dxs = U, torch.empty_like(dx)  # reuse the resident state buffer as the padded staging state
            packed = torch.empty(Uh.numel(), dtype=torch.float64, device=device)
            plan.fx_hydro_advance_host_interior(Uh, dxh, cfg.cfl, 1, stage_dev, packed, dxs)  # warm-up
            barrier()
            tt = time.perf_counter()
            for _ in range(args.e2e_steps):
                plan.fx_hydro_advance_host_interior(Uh, dxh, cfg.cfl, 1, stage_dev, packed, dxs)
            torch.cuda.synchronize()
            es = (time.perf_counter() - tt) / args.e2e_steps
            es = max_over_ranks(es, world, device)
            line["e2e"] = {"value": world * zones * stages / es, "unit": UNIT,
                           "h2d_bytes_per_step": Uh.numel() * 8 + dx.numel() * 8,
                           "d2h_bytes_per_step": Uh.numel() * 8 + 8, "ms_per_step": es * 1e3,
                           "steps": args.e2e_steps,
                           "api": "fx_hydro_advance_host_interior (pinned host buffer of interior zones; scatter into / "
                                  "gather from the padded device state inside the call)"}
            del Uh, packed
        except Exception as ex:  # e.g. not enough pinnable host memory
            line["e2e"] = {"value": None, "unit": UNIT, "error": repr(ex)[:200]}

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        del U
        torch.cuda.empty_cache()
        line["cpu_baseline"] = {k: v for k, v in oracle_sample(args, steps_single=2).items()
                                if k in ("value", "unit", "cores", "kind", "sample", "single_thread")}
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.amr:
        args.no_cpu_baseline = True  # (the oracle's two-level runs are in tests/; its timed sample is the uniform workload's)
        if args.gpus > 1 or args.shard or args.ca or args.nb or args.block or args.config != 5:
            sys.exit("--amr: single plan, config 5's scheme and field")
        if args.scalars:
            args.no_e2e = True  # (the end-to-end line is the five-variable workload's)
    if args.ca:
        args.no_e2e = True  # the end-to-end call (fx_hydro_advance_host_interior) runs the standard step
        if args.gpus > 1 or args.shard or args.scalars:
            sys.exit("--ca: single plan, five variables (fx_hydro_advance_ca refuses sharded plans and passive scalars)")
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl != "reference":
        # started plainly with --gpus N: launch the N ranks ourselves (one process per GPU, NCCL), as the driver's torchrun would
        import socket
        import torch
        if torch.cuda.device_count() < args.gpus:
            sys.exit(f"bench.py --gpus {args.gpus}: this machine has {torch.cuda.device_count()} GPU(s); one process per GPU is needed "
                     "(`--one-rank-of N` times one rank of an N-way partition alone)")
        sk = socket.socket()
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
        sk.close()
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
