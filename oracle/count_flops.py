"""Exact floating-point operation counts of the method as the oracle states it.

Builds oracle/count_flops.cpp (the oracle with a counting number type), runs one fxo_hydro_advance per scheme on a
small periodic tiling of seeded smooth data, and writes oracle/flop_counts.json: operations per interior zone and RK
stage, by kind.  Calls only oracle/ (and the seeded input generators).  bench.py reads the json for the flop side of
the roofline; tests/test_flop_counts.py checks the file against a fresh count.

    python -m oracle.count_flops [--check]

Counting convention [NS]: +, -, *, /, sqrt and each comparison count 1 (the oracle has no fused multiply-add);
flops = add + mul + div + sqrt + cmp.  The count is per zone-STAGE: total of one advance / (interior zones x stages);
block-boundary faces are evaluated by both blocks that share them (17 faces per 16 zones and direction), which is
part of the block-by-block method [P L69] and is included.
"""
from __future__ import annotations

import ctypes as C
import json
import os
import subprocess
import sys

import numpy as np

HERE = os.path.dirname(os.path.abspath(__file__))
ROOT = os.path.dirname(HERE)
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)
SRC = os.path.join(HERE, "count_flops.cpp")
LIB = os.path.join(HERE, "libfxoracle_count.so")
OUT = os.path.join(HERE, "flop_counts.json")

CASES = [  # name, block dims, tiling, recon, riemann, rk, wavespeed
    ("3d_plm_hllc_rk2", (16, 16, 16), (2, 2, 2), 0, 1, 2, 0),
    ("3d_plm_hlle_rk2", (16, 16, 16), (2, 2, 2), 0, 0, 2, 0),
    ("3d_weno5_hllc_rk3", (16, 16, 16), (2, 2, 2), 1, 1, 3, 0),
    ("3d_plm_hllc_rk2_davis", (16, 16, 16), (2, 2, 2), 0, 1, 2, 1),
    ("3d_plm_hllc_rk2_8cubed", (8, 8, 8), (2, 2, 2), 0, 1, 2, 0),
    ("3d_weno5_hllc_rk3_8cubed", (8, 8, 8), (2, 2, 2), 1, 1, 3, 0),
    ("2d_plm_hllc_rk2", (16, 16, 1), (4, 4, 1), 0, 1, 2, 0),
    ("2d_weno5_hllc_rk3", (16, 16, 1), (4, 4, 1), 1, 1, 3, 0),
    ("1d_plm_hlle_rk2", (256, 1, 1), (1, 1, 1), 0, 0, 2, 0),
    ("1d_plm_hllc_rk2", (256, 1, 1), (1, 1, 1), 0, 1, 2, 0),
]


def build():
    if not os.path.exists(LIB) or os.path.getmtime(LIB) < max(os.path.getmtime(SRC), os.path.getmtime(os.path.join(HERE, "fxoracle.c"))):
        subprocess.check_call(["g++", "-O1", "-std=c++17", "-ffp-contract=off", "-shared", "-fPIC", "-Wno-unknown-pragmas",
                               "-o", LIB, SRC, "-lm"])
    return LIB


def count_all():
    from oracle import fxoracle as fxo
    lib_path = build()
    fxo._lib = None
    fxo.build = lambda force=False: lib_path  # the wrapper loads the counting build instead of the plain one
    L = fxo.lib()
    L.fxo_count_reset.restype = None
    L.fxo_count_get.restype = None
    L.fxo_count_get.argtypes = [C.POINTER(C.c_ulonglong)]
    out = {}
    rng = np.random.default_rng(220811630)
    for name, dims, nb, recon, riemann, rk, ws in CASES:
        per = fxo.TOPO_PERIODIC
        bcs = [per if dims[d] > 1 else fxo.TOPO_NONE for d in range(3)]
        neigh, _ = fxo.topology_cartesian(nb, bcs, bcs, fxo.ORDER_LEX)
        nblocks = neigh.shape[0]
        plan = fxo.OraclePlan(dims, 4, nblocks, 1.4, recon, riemann, rk)
        plan.set_topology(neigh)
        plan.set_option(fxo.OPT_WAVESPEED, ws)
        U = np.full(plan.shape, np.nan)
        I = plan.interior(U)
        shape = I.shape[1:]
        rho = 1.0 + 0.3 * rng.random(shape)
        vel = 0.4 * rng.standard_normal((3,) + shape)
        pr = 1.0 + 0.3 * rng.random(shape)
        I[0] = rho
        for d in range(3):
            I[1 + d] = rho * vel[d] if dims[d] > 1 else 0.0
        I[4] = pr / 0.4 + 0.5 * rho * sum(vel[d] ** 2 for d in range(3) if dims[d] > 1)
        dx = np.full((nblocks, 3), 1.0 / 32)
        L.fxo_count_reset()
        plan.advance(U, dx, 1e-3)
        c = (C.c_ulonglong * 5)()
        L.fxo_count_get(c)
        zones_stages = nblocks * dims[0] * dims[1] * dims[2] * rk
        kinds = dict(zip(("add", "mul", "div", "sqrt", "cmp"), (int(x) / zones_stages for x in c)))
        kinds["flops"] = sum(kinds.values())
        out[name] = {k: round(v, 3) for k, v in kinds.items()}
    return out


def main():
    counts = count_all()
    if "--check" in sys.argv:
        stored = json.load(open(OUT))["per_zone_stage"]
        assert stored == counts, (stored, counts)
        print("flop_counts.json is up to date")
        return
    doc = {"what": "floating-point operations per interior zone and RK stage of the method as oracle/fxoracle.c states it "
                   "(+ - * / sqrt compare = 1 each, no FMA); written by oracle/count_flops.py",
           "per_zone_stage": counts}
    with open(OUT, "w") as f:
        json.dump(doc, f, indent=1)
        f.write("\n")
    for k, v in counts.items():
        print(k, v)


if __name__ == "__main__":
    main()
