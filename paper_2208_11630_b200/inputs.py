"""Seeded synthetic inputs for the five BASELINE.json configs.

A module of its own, shared by the oracle-side tests and the CUDA-side tests/bench.  It holds none
of the method's arithmetic (no reconstruction, no Riemann solver, no update): it only defines the
initial primitive fields of each workload, converts them to the conserved variables the state array
stores, and places block interiors into the padded SoA layout U[v][b][k][j][i].  It imports neither
oracle/ nor the CUDA binding.  Recipes: DESIGN.md "Input recipe".

All generation is done with torch float64 tensor ops so the same code runs on the host (tests) and on
the device (bench, config 5 is 18 GB); whichever device made the bytes, the *same bytes* are handed
to the oracle and to the CUDA path.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np
import torch

BASE_SEED = 220811630

RECON_PLM_MINMOD, RECON_WENO5 = 0, 1
RIEMANN_HLLE, RIEMANN_HLLC = 0, 1
ORDER_LEX, ORDER_MORTON = 0, 1


@dataclasses.dataclass
class Config:
    number: int
    name: str
    block_dims: tuple  # (nx, ny, nz) interior zones per block
    nguard: int
    nb: tuple  # blocks per dimension (nbx, nby, nbz)
    bc: str  # "periodic" | "outflow"
    gamma: float
    recon: int
    riemann: int
    rk_order: int
    cfl: float
    steps: int | None  # fixed step count, or None when run to t_end
    t_end: float | None
    full_nb: tuple = None  # blocks per dimension of the full-size config (field definition domain)

    @property
    def nblocks(self):
        return self.nb[0] * self.nb[1] * self.nb[2]

    @property
    def ndim(self):
        return sum(1 for d in self.block_dims if d > 1)

    @property
    def domain_zones(self):
        """Global zone counts (NX, NY, NZ) of the domain the fields are defined on."""
        f = self.full_nb or self.nb
        return tuple(self.block_dims[d] * f[d] for d in range(3))

    @property
    def dx(self):
        """Zone width per dimension; the domain is the unit interval/square/cube."""
        N = self.domain_zones
        return tuple(1.0 / N[d] for d in range(3))

    @property
    def interior_zones(self):
        return self.nblocks * self.block_dims[0] * self.block_dims[1] * self.block_dims[2]


def config(number: int, nb=None) -> Config:
    """Config `number` (1..5) of BASELINE.json.  `nb` overrides the number of blocks per dimension
    (a smaller tiling of the same blocks, for CPU-sized tests and sampled neighbourhoods).  For configs 4
    and 5 the field and dx stay those of the full-size domain, evaluated on the global zones the reduced
    tiling covers (so a periodic wrap of the reduced tiling sees a jump); configs 1-3 are re-defined on the
    reduced domain."""
    P, W, E, C = RECON_PLM_MINMOD, RECON_WENO5, RIEMANN_HLLE, RIEMANN_HLLC
    if number == 1:
        c = Config(1, "sod-1d", (256, 1, 1), 4, (1, 1, 1), "outflow", 1.4, P, E, 2, 0.8, None, 0.2)
    elif number == 2:
        c = Config(2, "kelvin-helmholtz-2d", (16, 16, 1), 4, (8, 8, 1), "periodic", 1.4, P, C, 2, 0.4, 100, None)
    elif number == 3:
        c = Config(3, "sedov-3d", (16, 16, 16), 4, (8, 8, 8), "periodic", 1.4, P, C, 2, 0.3, 50, None)
    elif number == 4:
        c = Config(4, "smooth-random-3d-weno5", (16, 16, 16), 4, (16, 16, 16), "periodic", 5.0 / 3.0, W, C, 3, 0.3, 20, None)
    elif number == 5:
        c = Config(5, "large-batch-3d", (16, 16, 16), 4, (32, 32, 32), "periodic", 1.4, P, C, 2, 0.3, 10, None)
    else:
        raise ValueError("config number must be 1..5")
    if nb is not None:
        # configs 4 and 5 keep the full-size field (smooth on the scale of the full domain) and its dx;
        # configs 1-3 are re-defined on the reduced domain (the Sedov deposit must stay inside it)
        c = dataclasses.replace(c, nb=tuple(nb), full_nb=c.nb if number in (4, 5) else tuple(nb))
    return c


# ----------------------------------------------------------------- block bookkeeping

def _morton_key(c):
    key = np.zeros(c.shape[0], np.uint64)
    for b in range(21):
        for d in range(3):
            key |= ((c[:, d].astype(np.uint64) >> np.uint64(b)) & np.uint64(1)) << np.uint64(3 * b + d)
    return key


def block_coords(nb, order=ORDER_LEX) -> np.ndarray:
    """Block coordinates [nblocks, 3] (bx, by, bz) in id order: lexicographic (bx fastest) or Morton."""
    bz, by, bx = np.meshgrid(np.arange(nb[2]), np.arange(nb[1]), np.arange(nb[0]), indexing="ij")
    c = np.stack([bx.ravel(), by.ravel(), bz.ravel()], axis=1).astype(np.int32)
    if order == ORDER_MORTON:
        c = c[np.argsort(_morton_key(c), kind="stable")]
    return np.ascontiguousarray(c)


def dx_array(cfg: Config, nblocks=None) -> np.ndarray:
    n = cfg.nblocks if nblocks is None else nblocks
    return np.ascontiguousarray(np.tile(np.asarray(cfg.dx, np.float64), (n, 1)))


def padded_shape(cfg: Config, nblocks=None, nvars=5):
    g = [cfg.nguard if d > 1 else 0 for d in cfg.block_dims]
    n = cfg.nblocks if nblocks is None else nblocks
    return (nvars, n, cfg.block_dims[2] + 2 * g[2], cfg.block_dims[1] + 2 * g[1], cfg.block_dims[0] + 2 * g[0])


def embed(cfg: Config, interior: torch.Tensor, guard_value=float("nan")) -> torch.Tensor:
    """Place interiors [nvars][nsel][nz][ny][nx] into a padded state array; guard zones get guard_value
    (NaN by default: fx_hydro_advance must not depend on them [A15])."""
    g = [cfg.nguard if d > 1 else 0 for d in cfg.block_dims]
    nx, ny, nz = cfg.block_dims
    U = torch.full(padded_shape(cfg, interior.shape[1], interior.shape[0]), guard_value, dtype=torch.float64, device=interior.device)
    U[:, :, g[2]:g[2] + nz, g[1]:g[1] + ny, g[0]:g[0] + nx] = interior
    return U


def interior_view(cfg: Config, U):
    g = [cfg.nguard if d > 1 else 0 for d in cfg.block_dims]
    nx, ny, nz = cfg.block_dims
    return U[:, :, g[2]:g[2] + nz, g[1]:g[1] + ny, g[0]:g[0] + nx]


# ----------------------------------------------------------------- field definitions

def _global_index(cfg, coords, device):
    """Global zone indices of every zone of the selected blocks: three int64 tensors
    [nsel, n_d] (I, J, K)."""
    out = []
    for d in range(3):
        base = torch.as_tensor(np.asarray(coords)[:, d].astype(np.int64), device=device) * cfg.block_dims[d]
        out.append(base[:, None] + torch.arange(cfg.block_dims[d], device=device, dtype=torch.int64)[None, :])
    return out


def _prim_to_cons(rho, u, v, w, p, gamma):
    E = p / (gamma - 1.0) + 0.5 * rho * (u * u + v * v + w * w)
    return torch.stack([rho, rho * u, rho * v, rho * w, E], dim=0)


def _modes(seed_words, nmodes, kmax, kmin_inf=1):
    """Distinct (up to sign) non-zero integer wave vectors with |k|_inf in [kmin_inf, kmax], isotropic
    unit vectors and phases."""
    rng = np.random.default_rng(seed_words)
    ks, seen = [], set()
    while len(ks) < nmodes:
        k = rng.integers(-kmax, kmax + 1, size=3)
        if np.abs(k).max() < kmin_inf:
            continue
        t, tn = tuple(int(x) for x in k), tuple(int(-x) for x in k)
        if t in seen or tn in seen:
            continue
        seen.add(t)
        ks.append(k)
    ks = np.asarray(ks, np.int64)
    e = rng.normal(size=(nmodes, 3))
    e /= np.linalg.norm(e, axis=1, keepdims=True)
    phi = rng.uniform(0.0, 2.0 * math.pi, size=nmodes)
    return ks, e, phi


def _mode_sum(cfg, idx, ks, amp, phi, device):
    """sum_m amp[m] * cos(2 pi k_m . x + phi_m) at zone centres x = (I + 1/2)/N of the selected blocks,
    built from separable 1-D complex tables.  amp may be [nmodes] or [nmodes, ncomp].
    Returns [ncomp][nsel][nz][ny][nx] (ncomp = 1 for 1-D amp)."""
    N = cfg.domain_zones
    amp = np.asarray(amp, np.float64)
    if amp.ndim == 1:
        amp = amp[:, None]
    tabs = []
    for d in range(3):
        k = torch.as_tensor(ks[:, d], device=device)  # [m]
        # theta = pi * k * (2I+1) / N, with the integer product reduced mod 2N first
        prod = (k[:, None, None] * (2 * idx[d][None, :, :] + 1)) % (2 * N[d])  # [m, nsel, n_d]
        th = prod.to(torch.float64) * (math.pi / N[d])
        tabs.append(torch.complex(torch.cos(th), torch.sin(th)))
    c = torch.as_tensor(amp, device=device).to(torch.complex128) * torch.as_tensor(
        np.exp(1j * phi), device=device)[:, None]  # [m, ncomp]
    out = torch.einsum("mc,mbk,mbj,mbi->cbkji", c, tabs[2], tabs[1], tabs[0])
    return out.real.contiguous()


def block_interiors(cfg: Config, coords, device="cpu") -> torch.Tensor:
    """Conserved variables [5][nsel][nz][ny][nx] (float64) of the interiors of the blocks whose block
    coordinates are `coords` [nsel, 3], for config cfg."""
    coords = np.asarray(coords)
    dev = torch.device(device)
    nx, ny, nz = cfg.block_dims
    nsel = coords.shape[0]
    I, J, K = _global_index(cfg, coords, dev)
    N = cfg.domain_zones
    shape = (nsel, nz, ny, nx)
    ones = torch.ones(shape, dtype=torch.float64, device=dev)
    n = cfg.number
    if n == 1:
        # x < 0.5: (rho,u,p) = (1,0,1); else (0.125,0,0.1)   [CFG1]
        left = (2 * I + 1 < N[0])[:, None, None, :].expand(shape)
        rho = torch.where(left, 1.0 * ones, 0.125 * ones)
        p = torch.where(left, 1.0 * ones, 0.1 * ones)
        z = torch.zeros_like(ones)
        return _prim_to_cons(rho, z, z, z, p, cfg.gamma)
    if n == 2:
        # rho = 2, u = +0.5 where |y - 0.5| < 0.25, else rho = 1, u = -0.5; p = 2.5;
        # v = 0.01 sin(4 pi x) + 1e-3 (2 xi - 1), xi ~ U[0,1) per zone in (j,i) order   [CFG2]
        y = (J.to(torch.float64) + 0.5) / N[1]
        x = (I.to(torch.float64) + 0.5) / N[0]
        inner = (torch.abs(y - 0.5) < 0.25)[:, None, :, None].expand(shape)
        rho = torch.where(inner, 2.0 * ones, 1.0 * ones)
        u = torch.where(inner, 0.5 * ones, -0.5 * ones)
        xi = torch.as_tensor(np.random.default_rng([BASE_SEED, 2]).random((N[1], N[0])), device=dev)
        noise = xi[J[:, :, None], I[:, None, :]]  # [nsel, ny, nx]
        v = 0.01 * torch.sin(4.0 * math.pi * x)[:, None, None, :] + 1e-3 * (2.0 * noise[:, None, :, :] - 1.0)
        v = v.expand(shape).contiguous()
        return _prim_to_cons(rho, u, v, torch.zeros_like(ones), 2.5 * ones, cfg.gamma)
    if n == 3:
        # rho = 1, u = 0, p = 1e-5; the 32 zones whose centre lies within 2 dx of the centre get
        # E = 1/(32 dx^3)   [CFG3]; integer test: (2I+1-N)^2 + ... <= 16
        ox = (2 * I + 1 - N[0])[:, None, None, :]
        oy = (2 * J + 1 - N[1])[:, None, :, None]
        oz = (2 * K + 1 - N[2])[:, :, None, None]
        hot = (ox * ox + oy * oy + oz * oz) <= 16
        dxs = cfg.dx
        E = torch.where(hot, ones / (32.0 * dxs[0] * dxs[1] * dxs[2]), ones * (1e-5 / (cfg.gamma - 1.0)))
        z = torch.zeros_like(ones)
        return torch.stack([ones, z, z, z, E], dim=0)
    if n == 4:
        # rho = 1 + 0.1/4 sum_16 cos(.), u = A sum_16 e_m cos(.), rms |u| = 0.3 sqrt(gamma), p = 1   [CFG4]
        ks, _, phi = _modes([BASE_SEED, 4, 0], 16, 8)
        rho = 1.0 + _mode_sum(cfg, (I, J, K), ks, np.full(16, 0.1 * 0.25), phi, dev)[0]
        ks2, e2, phi2 = _modes([BASE_SEED, 4, 1], 16, 8)
        # analytic grid rms of sum_m e_m cos(.) with distinct (up to sign) modes below Nyquist: sqrt(16/2)
        A = 0.3 * math.sqrt(cfg.gamma) / math.sqrt(16 * 0.5)
        vel = _mode_sum(cfg, (I, J, K), ks2, A * e2, phi2, dev)
        return _prim_to_cons(rho, vel[0], vel[1], vel[2], ones, cfg.gamma)
    if n == 5:
        # u = A sum_64 |k|^-2 e_m cos(.), rms Mach 1 w.r.t. c0 = sqrt(gamma); rho = exp(s - sigma^2/2),
        # s a 64-mode sum with grid std sigma = 0.5; p = 1   [CFG5]
        ks, e, phi = _modes([BASE_SEED, 5, 0], 64, 16)
        a = 1.0 / (ks.astype(np.float64) ** 2).sum(axis=1)
        A = math.sqrt(cfg.gamma) / math.sqrt(0.5 * (a * a).sum())
        vel = _mode_sum(cfg, (I, J, K), ks, (A * a)[:, None] * e, phi, dev)
        ks2, _, phi2 = _modes([BASE_SEED, 5, 1], 64, 16)
        a2 = 1.0 / (ks2.astype(np.float64) ** 2).sum(axis=1)
        sigma = 0.5
        s = _mode_sum(cfg, (I, J, K), ks2, a2 * (sigma / math.sqrt(0.5 * (a2 * a2).sum())), phi2, dev)[0]
        rho = torch.exp(s - 0.5 * sigma * sigma)
        return _prim_to_cons(rho, vel[0], vel[1], vel[2], ones, cfg.gamma)
    raise ValueError(n)


def with_scalars(cfg: Config, coords, interior: torch.Tensor, ns: int) -> torch.Tensor:
    """Append ns passive mass scalars rho*X_s to interiors [5][nsel][nz][ny][nx] -> [5+ns][...] (reading B11; the
    stand-in for a multispecies composition).  Even s: a smooth abundance X_s = 0.5 + 0.4 cos(2 pi
    k_s.x + phi_s), integer k_s with 1 <= |k_s|_inf <= 3 in the active dimensions, seeded; odd s: a composition
    interface, X_s = 1 where N/4 <= I_d < 3N/4 along the active dimension d = (s // 2) % ndim, else 0.
    N_d counts the zones of the tiling cfg.nb (not of the full-size field), so reduced tilings keep both features."""
    if ns == 0:
        return interior
    coords = np.asarray(coords)
    dev = interior.device
    idx = _global_index(cfg, coords, dev)
    N = tuple(cfg.block_dims[d] * cfg.nb[d] for d in range(3))  # the tiling actually run (periodic on it)
    active = [d for d in range(3) if cfg.block_dims[d] > 1]
    rho = interior[0]
    view = [(slice(None), None, None, slice(None)), (slice(None), None, slice(None), None),
            (slice(None), slice(None), None, None)]
    out = [interior]
    rng = np.random.default_rng([BASE_SEED, cfg.number, 100])
    for s in range(ns):
        k = rng.integers(-3, 4, size=3)
        phi = rng.random()
        if s % 2 == 0:
            if all(k[d] == 0 for d in active):
                k[active[0]] = 1
            theta = torch.zeros(rho.shape, dtype=torch.float64, device=dev)
            for d in active:
                theta = theta + (int(k[d]) * (2 * idx[d] + 1) % (2 * N[d])).to(torch.float64)[view[d]] / N[d]
            X = 0.5 + 0.4 * torch.cos(math.pi * theta + 2.0 * math.pi * phi)
        else:
            d = active[(s // 2) % len(active)]
            inside = ((4 * idx[d] >= N[d]) & (4 * idx[d] < 3 * N[d]))[view[d]]
            X = torch.where(inside, torch.ones_like(rho), torch.zeros_like(rho))
        out.append((rho * X)[None])
    return torch.cat(out, dim=0)


def initial_state(cfg: Config, order=ORDER_LEX, device="cpu", chunk_blocks=2048, guard_value=float("nan")):
    """Padded state U[5][nblocks][nzp][nyp][nxp] of the whole config and the block coordinates."""
    coords = block_coords(cfg.nb, order)
    U = torch.full(padded_shape(cfg), guard_value, dtype=torch.float64, device=device)
    Ui = interior_view(cfg, U)
    for b0 in range(0, cfg.nblocks, chunk_blocks):
        b1 = min(cfg.nblocks, b0 + chunk_blocks)
        Ui[:, b0:b1] = block_interiors(cfg, coords[b0:b1], device)
    return U, coords


def neighbourhood(cfg: Config, centre, radius: int):
    """Block coordinates of the (2r+1)^ndim cube of blocks around `centre` (wrapped periodically in
    the full domain), in lexicographic order of the offset, and the sub-tiling shape.  Used to check
    sampled blocks of a full-size run with an oracle run on the neighbourhood only."""
    rng = [range(-radius, radius + 1) if cfg.block_dims[d] > 1 else range(0, 1) for d in range(3)]
    out = []
    for oz in rng[2]:
        for oy in rng[1]:
            for ox in rng[0]:
                out.append([(centre[0] + ox) % cfg.nb[0], (centre[1] + oy) % cfg.nb[1], (centre[2] + oz) % cfg.nb[2]])
    return np.asarray(out, np.int32), tuple(len(r) for r in rng)


# ------------------------------------------------------------------ static two-level grids (B12; bench.py --amr)
NEIGH_COARSER, NEIGH_FINER = -4, -5


def two_level_tiling(nbc, lo, hi, order=ORDER_MORTON):
    """A 3-D periodic two-level block grid: the coarse tiling nbc = (cx, cy, cz), the coarse cells of the box [lo, hi)
    replaced by their 8 children.  Tables as include/fx_hydro.h defines them: neigh int32 [n, 6] (same-level id,
    NEIGH_COARSER or NEIGH_FINER), jump int32 [n, 6, 4] (behind NEIGH_FINER the four children that touch the face, index =
    first transverse half + 2 x second transverse half, transverse dimensions ascending; behind NEIGH_COARSER the coarse
    block and the index of the quarter of its face this block covers).  Block order: the coarse cells in `order`, a refined
    cell's children in place, x fastest.  Returns dict(neigh, jump, level [n], fine [n, 3]: the block's coordinates in the
    FINE tiling (a coarse block: those of its first child))."""
    nbc, lo, hi = tuple(nbc), tuple(lo), tuple(hi)
    refined = lambda c: all(lo[d] <= c[d] < hi[d] for d in range(3))  # noqa: E731
    ident, level, fine = {}, [], []
    for c in block_coords(nbc, order):
        c = tuple(int(x) for x in c)
        if refined(c):
            for cz in range(2):
                for cy in range(2):
                    for cx in range(2):
                        ident[(c, (cx, cy, cz))] = len(level)
                        level.append(1)
                        fine.append((2 * c[0] + cx, 2 * c[1] + cy, 2 * c[2] + cz))
        else:
            ident[(c, None)] = len(level)
            level.append(0)
            fine.append((2 * c[0], 2 * c[1], 2 * c[2]))
    n = len(level)
    neigh = np.empty((n, 6), np.int32)
    jump = np.full((n, 6, 4), -1, np.int32)
    for (c, ch), b in ident.items():
        for d in range(3):
            t1, t2 = [e for e in range(3) if e != d]
            for side in (0, 1):
                f = 2 * d + side
                if ch is not None and ch[d] != side:  # the sibling inside the same parent
                    sib = list(ch)
                    sib[d] = side
                    neigh[b, f] = ident[(c, tuple(sib))]
                    continue
                nc = list(c)
                nc[d] = (nc[d] + (1 if side else -1)) % nbc[d]
                nc = tuple(nc)
                if ch is None:
                    if not refined(nc):
                        neigh[b, f] = ident[(nc, None)]
                    else:
                        neigh[b, f] = NEIGH_FINER
                        for q in range(4):
                            kid = [0, 0, 0]
                            kid[d] = 1 - side  # the children that touch our face
                            kid[t1], kid[t2] = q & 1, q >> 1
                            jump[b, f, q] = ident[(nc, tuple(kid))]
                else:
                    if refined(nc):
                        kid = list(ch)
                        kid[d] = 1 - side
                        neigh[b, f] = ident[(nc, tuple(kid))]
                    else:
                        neigh[b, f] = NEIGH_COARSER
                        jump[b, f, 0] = ident[(nc, None)]
                        jump[b, f, 1] = ch[t1] + 2 * ch[t2]
    return dict(neigh=neigh, jump=jump, level=np.array(level, np.int32), fine=np.array(fine, np.int32))


def two_level_interiors(cfg_fine: Config, grid, b0, b1, device="cpu") -> torch.Tensor:
    """Conserved interiors [5, b1 - b0, nz, ny, nx] of blocks [b0, b1) of a two_level_tiling whose FINE tiling is cfg_fine's:
    a fine block holds cfg_fine's field, a coarse block the plain means over the 2 x 2 x 2 fine zones each of its zones
    covers (input recipe only: a coarse field consistent with the fine one)."""
    n = cfg_fine.block_dims
    out = torch.empty((5, b1 - b0, n[2], n[1], n[0]), dtype=torch.float64, device=device)
    lev, fine = grid["level"][b0:b1], grid["fine"][b0:b1]
    isf = np.nonzero(lev == 1)[0]
    if len(isf):
        out[:, torch.as_tensor(isf, device=device)] = block_interiors(cfg_fine, fine[isf], device)
    isc = np.nonzero(lev == 0)[0]
    if len(isc):
        acc = torch.zeros((5, len(isc), n[2], n[1], n[0]), dtype=torch.float64, device=device)
        h = [m // 2 for m in n]
        for cz in range(2):
            for cy in range(2):
                for cx in range(2):
                    kids = block_interiors(cfg_fine, fine[isc] + np.array([cx, cy, cz], np.int32), device)
                    pooled = kids.reshape(5, len(isc), h[2], 2, h[1], 2, h[0], 2).sum(dim=(3, 5, 7))
                    acc[:, :, cz * h[2]:(cz + 1) * h[2], cy * h[1]:(cy + 1) * h[1], cx * h[0]:(cx + 1) * h[0]] = pooled
        out[:, torch.as_tensor(isc, device=device)] = acc * 0.125
    return out
