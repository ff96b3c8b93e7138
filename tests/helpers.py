"""Test helpers shared by the oracle pins and the GPU parity tests (no method arithmetic beyond the
textbook exact Riemann solver used as an external pin)."""
import math

import numpy as np

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs


def golden_rows(name):
    import os
    path = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", name)
    rows = []
    with open(path) as f:
        for line in f:
            if line.startswith("#") or not line.strip():
                continue
            rows.append(line.split())
    return rows


def oracle_plan_for(cfg, nblocks=None, order=inputs.ORDER_LEX, bc=None, nb=None, recon=None, riemann=None, rk=None,
                    nvars=5, wavespeed=None):
    """Oracle plan + topology for a config (regular tiling nb, default cfg.nb)."""
    nb = tuple(nb or cfg.nb)
    bc = bc or cfg.bc
    code = {"periodic": fxo.TOPO_PERIODIC, "outflow": fxo.TOPO_OUTFLOW, "reflect": fxo.TOPO_REFLECT}[bc]
    bcs = [code if cfg.block_dims[d] > 1 else fxo.TOPO_NONE for d in range(3)]
    neigh, coords = fxo.topology_cartesian(nb, bcs, bcs, order)
    plan = fxo.OraclePlan(cfg.block_dims, cfg.nguard, neigh.shape[0], cfg.gamma,
                          cfg.recon if recon is None else recon, cfg.riemann if riemann is None else riemann,
                          cfg.rk_order if rk is None else rk, nvars=nvars)
    plan.set_topology(neigh)
    if wavespeed is not None:
        plan.set_option(fxo.OPT_WAVESPEED, wavespeed)
    return plan, neigh, coords


def exact_riemann(WL, WR, gamma, xi):
    """Exact solution of the 1-D Riemann problem for a perfect gas sampled at xi = x/t (array).
    Textbook (Toro, Riemann Solvers..., ch. 4): Newton iteration on the star pressure.  States
    (rho, u, p).  Returns rho, u, p arrays."""
    rl, ul, pl = WL
    rr, ur, pr = WR
    g = gamma
    cl, cr = math.sqrt(g * pl / rl), math.sqrt(g * pr / rr)

    def f(p, rk, pk, ck):
        if p > pk:
            A, B = 2.0 / ((g + 1) * rk), (g - 1) / (g + 1) * pk
            q = math.sqrt(A / (p + B))
            return (p - pk) * q, q * (1 - 0.5 * (p - pk) / (p + B))
        return 2 * ck / (g - 1) * ((p / pk) ** ((g - 1) / (2 * g)) - 1), 1 / (rk * ck) * (p / pk) ** (-(g + 1) / (2 * g))

    p = 0.5 * (pl + pr)
    for _ in range(100):
        fl, dfl = f(p, rl, pl, cl)
        fr, dfr = f(p, rr, pr, cr)
        dp = (fl + fr + ur - ul) / (dfl + dfr)
        p = max(p - dp, 1e-14)
        if abs(dp) < 1e-15 * p:
            break
    fl, _ = f(p, rl, pl, cl)
    fr, _ = f(p, rr, pr, cr)
    us = 0.5 * (ul + ur) + 0.5 * (fr - fl)
    ps = p
    xi = np.asarray(xi, np.float64)
    rho, u, pp = np.empty_like(xi), np.empty_like(xi), np.empty_like(xi)
    gm = (g - 1) / (g + 1)
    for n, s in enumerate(xi):
        if s <= us:  # left of contact
            if ps > pl:  # left shock
                sl = ul - cl * math.sqrt((g + 1) / (2 * g) * ps / pl + (g - 1) / (2 * g))
                if s <= sl:
                    rho[n], u[n], pp[n] = rl, ul, pl
                else:
                    rho[n], u[n], pp[n] = rl * ((ps / pl + gm) / (gm * ps / pl + 1)), us, ps
            else:
                shl = ul - cl
                csl = cl * (ps / pl) ** ((g - 1) / (2 * g))
                stl = us - csl
                if s <= shl:
                    rho[n], u[n], pp[n] = rl, ul, pl
                elif s >= stl:
                    rho[n], u[n], pp[n] = rl * (ps / pl) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) * (cl + (g - 1) / 2 * (ul - s))
                    rho[n] = rl * (c / cl) ** (2 / (g - 1))
                    u[n] = 2 / (g + 1) * (cl + (g - 1) / 2 * ul + s)
                    pp[n] = pl * (c / cl) ** (2 * g / (g - 1))
        else:
            if ps > pr:
                sr = ur + cr * math.sqrt((g + 1) / (2 * g) * ps / pr + (g - 1) / (2 * g))
                if s >= sr:
                    rho[n], u[n], pp[n] = rr, ur, pr
                else:
                    rho[n], u[n], pp[n] = rr * ((ps / pr + gm) / (gm * ps / pr + 1)), us, ps
            else:
                shr = ur + cr
                csr = cr * (ps / pr) ** ((g - 1) / (2 * g))
                str_ = us + csr
                if s >= shr:
                    rho[n], u[n], pp[n] = rr, ur, pr
                elif s <= str_:
                    rho[n], u[n], pp[n] = rr * (ps / pr) ** (1 / g), us, ps
                else:
                    c = 2 / (g + 1) * (cr - (g - 1) / 2 * (ur - s))
                    rho[n] = rr * (c / cr) ** (2 / (g - 1))
                    u[n] = 2 / (g + 1) * (-cr + (g - 1) / 2 * ur + s)
                    pp[n] = pr * (c / cr) ** (2 * g / (g - 1))
    return rho, u, pp, ps, us


def run_to_time(plan, U, dx, cfl, t_end=None, steps=None):
    """O8 driver: dt from compute_dt, last step clipped at t_end."""
    t, n = 0.0, 0
    while True:
        if steps is not None and n >= steps:
            break
        if t_end is not None and t >= t_end:
            break
        dt = plan.compute_dt(U, dx, cfl)
        if t_end is not None and t + dt > t_end:
            dt = t_end - t
        plan.advance(U, dx, dt)
        t += dt
        n += 1
    return t, n


def rel_err(cfg, got, ref):
    """Max relative cellwise error over interior zones [A21]: |d rho|/rho, |d E|/E,
    |d m_d|/(rho(|u|+c)), denominators from the reference state.  got/ref: interiors [5,...]."""
    got = np.asarray(got)
    ref = np.asarray(ref)
    rho, E = ref[0], ref[4]
    m2 = ref[1] ** 2 + ref[2] ** 2 + ref[3] ** 2
    p = np.maximum((cfg.gamma - 1.0) * (E - 0.5 * m2 / rho), 1e-300)
    scale_m = np.sqrt(m2) + rho * np.sqrt(cfg.gamma * p / rho)
    e = np.abs(got[0] - rho) / rho
    e = np.maximum(e, np.abs(got[4] - E) / E)
    for d in (1, 2, 3):
        e = np.maximum(e, np.abs(got[d] - ref[d]) / scale_m)
    if not np.all(np.isfinite(got)):
        return float("inf")
    return float(e.max())


def gpu_plan_for(cfg, order=inputs.ORDER_LEX, bc=None, nb=None, recon=None, riemann=None, rk=None, path=None,
                 neigh=None, nblocks=None, zchain=None, nvars=5, wavespeed=None):
    """CUDA-side plan + topology + workspace for a config (uses the library's own topology helper)."""
    from paper_2208_11630_b200 import binding as fx
    nb = tuple(nb or cfg.nb)
    bc = bc or cfg.bc
    code = {"periodic": fx.TOPO_PERIODIC, "outflow": fx.TOPO_OUTFLOW, "reflect": fx.TOPO_REFLECT}[bc]
    bcs = [code if cfg.block_dims[d] > 1 else fx.TOPO_NONE for d in range(3)]
    coords = None
    if neigh is None:
        neigh, coords = fx.fx_topology_cartesian(nb, bcs, bcs, order)
    plan = fx.HydroPlan(cfg.block_dims, cfg.nguard, neigh.shape[0], cfg.gamma,
                        cfg.recon if recon is None else recon, cfg.riemann if riemann is None else riemann,
                        cfg.rk_order if rk is None else rk, nvars=nvars)
    if path is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_PATH, path)
    if zchain is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_ZCHAIN, zchain)
    if wavespeed is not None:
        plan.fx_hydro_plan_set_option(fx.OPT_WAVESPEED, wavespeed)
    plan.fx_hydro_plan_set_topology(neigh)
    plan.fx_hydro_plan_set_workspace()
    return plan, neigh, coords


def cliff_state(cfg, coords, axis, high=1e6):
    """Conserved block interiors [5, nb, nz, ny, nx] of the config's own field with a density cliff and a pressure cliff
    along `axis` in every block -- a ramp (5.5, 3, 0.5) running into a plateau `high`, the profile whose WENO5 face
    value is negative on the ramp side (tests/test_oracle_pins_r2.py) -- so that the positivity fallback [A6] is taken
    on one side of some faces, in rho at one place and in p at another."""
    Ui = inputs.block_interiors(cfg, coords).numpy().copy()
    g = cfg.gamma
    rho = Ui[0]
    vel = Ui[1:4] / rho
    p = (g - 1) * (Ui[4] - 0.5 * rho * (vel ** 2).sum(0))
    ax = 3 - axis  # axis of rho[b, k, j, i]
    n = rho.shape[ax]
    lo_r, lo_p = (1, n - 7) if n >= 14 else (1, 1)
    for lo, arr, vals in ((lo_r, rho, (5.5, 3.0, 0.5, high, high, high)), (lo_p, p, (high, high, high, 0.5, 3.0, 5.5))):
        s = [slice(None)] * 4
        s[ax] = slice(lo, lo + 6)
        shape = [1, 1, 1, 1]
        shape[ax] = 6
        arr[tuple(s)] = np.array(vals).reshape(shape)
    return np.stack([rho, rho * vel[0], rho * vel[1], rho * vel[2], p / (g - 1) + 0.5 * rho * (vel ** 2).sum(0)])


def two_level_grid(nbc, refined, block_dims, periodic=True):
    """A static 2-level block grid [B12]: the coarse tiling nbc = (cx, cy, cz) of a unit-width-per-coarse-zone domain, the
    coarse cells in `refined` (a set of (X, Y, Z)) replaced by their 2^ndim children.  Written in numpy from the
    definition of the tables (include/fx_hydro.h, fxo_plan_set_refinement); used for both sides.
    Returns dict(neigh int32 [n,6], jump int32 [n,6,4], level int [n], origin float [n,3] (lower corner in coarse zones),
    dxrel float [n] (zone width in coarse zones: 1 or 1/2), cell [n,3], child [n,3])."""
    dims = [d for d in range(3) if block_dims[d] > 1]
    refined = set(tuple(r) for r in refined)
    blocks = []  # (level, cell, child)
    for Z in range(nbc[2]):
        for Y in range(nbc[1]):
            for X in range(nbc[0]):
                if (X, Y, Z) in refined:
                    for cz in range(2 if 2 in dims else 1):
                        for cy in range(2 if 1 in dims else 1):
                            for cx in range(2 if 0 in dims else 1):
                                blocks.append((1, (X, Y, Z), (cx, cy, cz)))
                else:
                    blocks.append((0, (X, Y, Z), (0, 0, 0)))
    ident = {(lv, cell, ch): i for i, (lv, cell, ch) in enumerate(blocks)}
    n = len(blocks)
    neigh = np.full((n, 6), -2, np.int32)
    jump = np.full((n, 6, 4), -1, np.int32)
    for b, (lv, cell, ch) in enumerate(blocks):
        for d in dims:
            tr = [e for e in range(3) if e != d]
            for side in (0, 1):
                f = 2 * d + side
                if lv == 1 and ch[d] == 1 - side:  # the sibling inside the same parent
                    sib = list(ch)
                    sib[d] = side
                    neigh[b, f] = ident[(1, cell, tuple(sib))]
                    continue
                nc = list(cell)
                nc[d] += 1 if side else -1
                if nc[d] < 0 or nc[d] >= nbc[d]:
                    if not periodic:
                        neigh[b, f] = -1  # outflow
                        continue
                    nc[d] %= nbc[d]
                nc = tuple(nc)
                if lv == 0:
                    if nc not in refined:
                        neigh[b, f] = ident[(0, nc, (0, 0, 0))]
                    else:
                        neigh[b, f] = -5
                        for q in range(4):
                            kid = [0, 0, 0]
                            kid[d] = 0 if side else 1
                            ok = True
                            for t, e in enumerate(tr):
                                bit = (q >> t) & 1
                                if e in dims:
                                    kid[e] = bit
                                elif bit:
                                    ok = False
                            if ok:
                                jump[b, f, q] = ident[(1, nc, tuple(kid))]
                else:
                    if nc in refined:
                        kid = list(ch)
                        kid[d] = 0 if side else 1
                        neigh[b, f] = ident[(1, nc, tuple(kid))]
                    else:
                        neigh[b, f] = -4
                        jump[b, f, 0] = ident[(0, nc, (0, 0, 0))]
                        jump[b, f, 1] = sum(ch[e] << t for t, e in enumerate(tr) if e in dims)
    level = np.array([lv for lv, _, _ in blocks])
    origin = np.array([[cell[d] * block_dims[d] + (ch[d] * block_dims[d] / 2 if lv else 0) for d in range(3)] for lv, cell, ch in blocks], float)
    return dict(neigh=neigh, jump=jump, level=level, origin=origin, dxrel=np.where(level == 1, 0.5, 1.0),
                cell=np.array([c for _, c, _ in blocks]), child=np.array([c for _, _, c in blocks]))


def amr_zone_centres(grid, block_dims):
    """Zone-centre coordinates (in coarse zones) of every interior zone: [n, 3, nz, ny, nx]."""
    n = len(grid["level"])
    out = np.zeros((n, 3, block_dims[2], block_dims[1], block_dims[0]))
    for b in range(n):
        h = grid["dxrel"][b]
        ax = [grid["origin"][b, d] + (np.arange(block_dims[d]) + 0.5) * (h if block_dims[d] > 1 else 1.0) for d in range(3)]
        K, J, I = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
        out[b, 0], out[b, 1], out[b, 2] = I, J, K
    return out
