"""Oracle pins for the fine-coarse boundary services [B12-B14] ("fine-coarse boundary resolution related API
functions of the Grid unit"): restriction and conservative limited prolongation into the face guard zones behind a
refinement jump, and the flux correction of the coarse face flux -- on static two-level grids (tests.helpers.two_level_grid)."""
import math

import numpy as np
import pytest

from oracle import fxoracle as fxo
from tests.helpers import amr_zone_centres, two_level_grid

GAMMA = 1.4


def amr_plan(grid, dims, g=4, recon=0, riemann=1, rk=2, nvars=5):
    n = len(grid["level"])
    plan = fxo.OraclePlan(dims, g, n, GAMMA, recon, riemann, rk, nvars=nvars)
    plan.set_refinement(grid["jump"])
    plan.set_topology(grid["neigh"])
    return plan


def cons(rho, u, v, w, p):
    return np.stack([rho, rho * u, rho * v, rho * w, p / (GAMMA - 1.0) + 0.5 * rho * (u * u + v * v + w * w)])


def state_from(plan, fields):
    """fields: [5, n, nz, ny, nx] conserved interiors -> padded state with NaN guards."""
    U = np.full(plan.shape, np.nan)
    plan.interior(U)[...] = fields
    return U


def smooth_field(grid, dims, L):
    """Smooth periodic data on the grid, point values at the zone centres (domain extent L in coarse zones)."""
    X = amr_zone_centres(grid, dims)
    ph = [2 * np.pi * X[:, d] / L[d] if dims[d] > 1 else 0.0 * X[:, d] for d in range(3)]
    rho = 1.0 + 0.2 * np.sin(ph[0]) * np.cos(ph[1]) + 0.1 * np.cos(ph[2] + 0.3)
    u = 0.3 * np.cos(ph[0] + 0.5) if dims[0] > 1 else 0.0 * rho
    v = 0.2 * np.sin(ph[1] + ph[0]) if dims[1] > 1 else 0.0 * rho
    w = 0.25 * np.sin(ph[2] - ph[1]) if dims[2] > 1 else 0.0 * rho
    p = 1.0 + 0.1 * np.cos(ph[0] - ph[1] + ph[2])
    return cons(rho, u, v, w, p)


def dx_of(grid, base=1.0 / 32):
    return np.repeat((grid["dxrel"] * base)[:, None], 3, axis=1).copy()


def totals(plan, grid, U, ndim):
    I = plan.interior(U)
    wgt = grid["dxrel"] ** ndim
    return np.array([math.fsum((I[v] * wgt[:, None, None, None]).ravel()) for v in range(I.shape[0])])


GRIDS = [((4, 1, 1), {(1, 0, 0)}, (16, 1, 1)), ((4, 4, 1), {(1, 1, 0), (2, 1, 0)}, (8, 8, 1)),
         ((3, 3, 3), {(1, 1, 1)}, (8, 8, 8)), ((3, 3, 2), {(0, 0, 0), (1, 0, 0), (2, 2, 1)}, (8, 8, 8))]


@pytest.mark.parametrize("nbc,refined,dims", GRIDS)
@pytest.mark.parametrize("recon,riemann,rk", [(0, 1, 2), (1, 0, 3)])
def test_uniform_state_is_preserved_bitwise_across_jumps(nbc, refined, dims, recon, riemann, rk):
    grid = two_level_grid(nbc, refined, dims)
    plan = amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk)
    n = len(grid["level"])
    shape = (n, dims[2], dims[1], dims[0])
    W = (1.3, 0.4 if dims[0] > 1 else 0.0, -0.7 if dims[1] > 1 else 0.0, 0.2 if dims[2] > 1 else 0.0, 0.9)
    U = state_from(plan, cons(*[np.full(shape, x) for x in W]))
    U0 = plan.interior(U).copy()
    dx = dx_of(grid)
    for _ in range(5):
        plan.advance(U, dx, plan.compute_dt(U, dx, 0.3))
    assert np.array_equal(plan.interior(U), U0)


@pytest.mark.parametrize("nbc,refined,dims", [((5, 1, 1), {(2, 0, 0)}, (16, 1, 1)), ((5, 5, 1), {(2, 2, 0)}, (8, 8, 1)),
                                               ((5, 5, 5), {(2, 2, 2)}, (8, 8, 8))])
def test_linear_data_are_prolonged_and_restricted_exactly(nbc, refined, dims):
    """q = a + b.x at the zone centres: the limited slopes are the slope itself, so every prolonged fine guard zone and
    every restricted coarse guard zone holds the linear function at its own centre; and the 2^ndim children of a coarse
    zone average to it (restriction o prolongation = identity)."""
    grid = two_level_grid(nbc, refined, dims, periodic=False)
    plan = amr_plan(grid, dims)
    X = amr_zone_centres(grid, dims)
    ndim = sum(1 for d in dims if d > 1)
    coef = np.array([0.7, -0.4, 0.25])
    lin = lambda x, y, z, v: (v + 2.0) + 0.01 * (v + 1) * (coef[0] * x + coef[1] * y + coef[2] * z)
    U = state_from(plan, np.stack([lin(X[:, 0], X[:, 1], X[:, 2], v) for v in range(5)]))
    plan.fill_guardcells(U)
    g = 4
    checked = 0
    for b in range(len(grid["level"])):
        h = grid["dxrel"][b]
        for f in range(6):
            code = grid["neigh"][b, f]
            if code not in (fxo.NEIGH_COARSER, fxo.NEIGH_FINER):
                continue
            d, side = f // 2, f % 2
            for m in range(g):
                idx = [slice(g, g + dims[2]) if dims[2] > 1 else slice(0, 1), slice(g, g + dims[1]) if dims[1] > 1 else slice(0, 1),
                       slice(g, g + dims[0])]
                pos = g + dims[d] + m if side else g - 1 - m
                idx[2 - d] = slice(pos, pos + 1)
                ax = [grid["origin"][b, e] + (np.arange(dims[e]) + 0.5) * (h if dims[e] > 1 else 1.0) for e in range(3)]
                ax[d] = np.array([grid["origin"][b, d] + (pos - g + 0.5) * h])
                K, J, I = np.meshgrid(ax[2], ax[1], ax[0], indexing="ij")
                for v in range(5):
                    got = U[v, b][tuple(idx)]
                    assert np.allclose(got, lin(I, J, K, v), rtol=0, atol=2e-15 * 3), (b, f, m, v)
                checked += 1
    assert checked >= 2 * g
    # children average to the parent: the fine block's guard zones behind a coarser face, in 2^ndim groups
    for b in np.flatnonzero(grid["level"] == 1):
        for f in range(6):
            if grid["neigh"][b, f] != fxo.NEIGH_COARSER:
                continue
            d, side = f // 2, f % 2
            cb, qd = grid["jump"][b, f, 0], grid["jump"][b, f, 1]
            tr = [e for e in range(3) if e != d]
            Ic = plan.interior(U)[:, cb]
            for pm in range(2):  # parent depth
                sl = [slice(g, g + dims[2]) if dims[2] > 1 else slice(0, 1), slice(g, g + dims[1]) if dims[1] > 1 else slice(0, 1),
                      slice(g, g + dims[0])]
                lo = g + dims[d] + 2 * pm if side else g - 2 - 2 * pm
                sl[2 - d] = slice(lo, lo + 2)
                kids = U[:, b][(slice(None),) + tuple(sl)]
                shp = kids.shape[1:]
                new = []
                for e, s_ in zip((2, 1, 0), shp):
                    new += [s_ // 2, 2] if (dims[e] > 1) else [s_, 1]
                mean = kids.reshape((5,) + tuple(new)).mean(axis=(2, 4, 6))
                csl = [slice(None)] * 3
                for t, e in enumerate(tr):
                    if dims[e] > 1:
                        a = (qd >> t) & 1
                        csl[2 - e] = slice(a * dims[e] // 2, (a + 1) * dims[e] // 2)
                cpos = pm if side else dims[d] - 1 - pm
                csl[2 - d] = slice(cpos, cpos + 1)
                assert np.allclose(mean, Ic[(slice(None),) + tuple(csl)], rtol=4e-16, atol=0)


@pytest.mark.parametrize("nbc,refined,dims", GRIDS)
@pytest.mark.parametrize("recon,rk", [(0, 2), (1, 3)])
def test_conservation_across_jumps(nbc, refined, dims, recon, rk):
    """Volume-weighted totals over a periodic two-level grid, 10 steps: <= 1e-13 relative [NS, A22] -- what the flux
    correction [B14] is for (without it the coarse and the fine side of a jump book different fluxes)."""
    grid = two_level_grid(nbc, refined, dims)
    plan = amr_plan(grid, dims, recon=recon, rk=rk)
    ndim = sum(1 for d in dims if d > 1)
    L = [nbc[d] * dims[d] for d in range(3)]
    U = state_from(plan, smooth_field(grid, dims, L))
    dx = dx_of(grid)
    T0 = totals(plan, grid, U, ndim)
    for _ in range(10):
        plan.advance(U, dx, plan.compute_dt(U, dx, 0.3))
    T1 = totals(plan, grid, U, ndim)
    scale = np.array([T0[0], 2.4 * T0[0], 2.4 * T0[0], 2.4 * T0[0], T0[4]])
    assert np.isfinite(T1).all()
    assert np.max(np.abs(T1 - T0) / scale) <= 1e-13, (T1 - T0) / scale
    assert plan.status()[0] == 0


def test_jump_table_without_jumps_changes_nothing():
    dims = (8, 8, 8)
    grid = two_level_grid((2, 2, 2), set(), dims)
    L = [16, 16, 16]
    a = amr_plan(grid, dims)
    b = fxo.OraclePlan(dims, 4, 8, GAMMA, 0, 1, 2)
    b.set_topology(grid["neigh"])
    Ua = state_from(a, smooth_field(grid, dims, L))
    Ub = Ua.copy()
    dx = dx_of(grid)
    for _ in range(3):
        a.advance(Ua, dx, 1e-3)
        b.advance(Ub, dx, 1e-3)
    assert np.array_equal(a.interior(Ua), b.interior(Ub))


def test_refined_sod_is_between_the_coarse_and_the_fine_uniform_runs():
    """1-D Sod on 8 coarse blocks of 32 zones with the middle four refined, to t = 0.2 (the shock has crossed the jump
    at x = 0.75 by then): its density error against the exact solution lies between the all-fine and the all-coarse
    run's; mass and energy conserved to rounding through the jump."""
    from tests.helpers import exact_riemann
    dims, nbc = (32, 1, 1), (8, 1, 1)

    def run(refined):
        grid = two_level_grid(nbc, refined, dims, periodic=False)
        plan = amr_plan(grid, dims, riemann=0)
        X = amr_zone_centres(grid, dims)[:, 0] / (nbc[0] * dims[0])
        rho = np.where(X < 0.5, 1.0, 0.125)
        p = np.where(X < 0.5, 1.0, 0.1)
        z = np.zeros_like(rho)
        U = state_from(plan, cons(rho, z, z, z, p))
        dx = dx_of(grid, 1.0 / (nbc[0] * dims[0]))
        T0 = totals(plan, grid, U, 1)
        t = 0.0
        while t < 0.2:
            dt = min(plan.compute_dt(U, dx, 0.8), 0.2 - t)
            plan.advance(U, dx, dt)
            t += dt
        T1 = totals(plan, grid, U, 1)
        assert abs(T1[0] - T0[0]) <= 1e-13 * T0[0] and abs(T1[4] - T0[4]) <= 1e-13 * T0[4]
        ex = exact_riemann((1, 0, 1), (0.125, 0, 0.1), GAMMA, ((X - 0.5) / 0.2).ravel())[0].reshape(X.shape)
        err = math.fsum((np.abs(plan.interior(U)[0] - ex) * grid["dxrel"][:, None, None, None]).ravel()) / (nbc[0] * dims[0])
        return err

    coarse, amr = run(set()), run({(2, 0, 0), (3, 0, 0), (4, 0, 0), (5, 0, 0)})
    fine = run({(i, 0, 0) for i in range(8)})
    assert fine < amr < coarse, (coarse, amr, fine)


def test_mirror_symmetric_patch_gives_mirror_symmetric_flow():
    dims, nbc = (8, 8, 1), (4, 4, 1)
    grid = two_level_grid(nbc, {(1, 1, 0), (2, 1, 0), (1, 2, 0), (2, 2, 0)}, dims)
    plan = amr_plan(grid, dims)
    X = amr_zone_centres(grid, dims)
    x, y = X[:, 0] / 32 - 0.5, X[:, 1] / 32 - 0.5
    rho = 1.0 + 0.5 * np.exp(-40 * (x * x + y * y))
    p = 1.0 + 2.0 * np.exp(-40 * (x * x + y * y))
    z = np.zeros_like(rho)
    U = state_from(plan, cons(rho, z, z, z, p))
    dx = dx_of(grid)
    for _ in range(8):
        plan.advance(U, dx, plan.compute_dt(U, dx, 0.4))
    I = plan.interior(U)
    # the block holding the mirror image in x: same level, cell and child mirrored
    key = {(int(l), tuple(c), tuple(ch)): i for i, (l, c, ch) in enumerate(zip(grid["level"], grid["cell"], grid["child"]))}
    for b, (l, c, ch) in enumerate(zip(grid["level"], grid["cell"], grid["child"])):
        m = key[(int(l), (3 - c[0], c[1], c[2]), ((1 - ch[0]) if l else 0, ch[1], ch[2]))]
        assert np.allclose(I[0, b], I[0, m][..., ::-1], rtol=1e-13, atol=0)
        assert np.allclose(I[1, b], -I[1, m][..., ::-1], rtol=0, atol=1e-13)
        assert np.allclose(I[4, b], I[4, m][..., ::-1], rtol=1e-13, atol=0)


# ---- passive mass scalars through refinement jumps [B11 with B12-B14]: the scalars are conserved variables like the rest,
# so restriction, prolongation and the flux correction act on rho X_s as they act on a momentum component
def with_scalars(fields, X):
    """fields [5, ...] conserved; X: list of abundance arrays -> [5 + ns, ...]."""
    return np.concatenate([fields, np.stack([fields[0] * x for x in X])])


@pytest.mark.parametrize("recon,riemann,rk", [(0, 1, 2), (0, 0, 3), (1, 1, 3)])
def test_scalar_equal_to_w_is_the_out_of_plane_momentum_bitwise_through_jumps(recon, riemann, rk):
    """2-D two-level grid, w a smooth field: a scalar with X = w is advected, restricted, prolonged and flux-corrected
    exactly as m_z is -- rho X stays equal to m_z BIT FOR BIT; and the hydro variables are those of the run without scalars."""
    dims = (8, 8, 1)
    grid = two_level_grid((4, 4, 1), {(1, 1, 0), (2, 1, 0)}, dims)
    f5 = smooth_field(grid, dims, [32, 32, 1])
    X = amr_zone_centres(grid, dims)
    w = 0.3 * np.sin(2 * np.pi * X[:, 0] / 32) * np.cos(2 * np.pi * X[:, 1] / 32 + 0.4)
    f5[3] = f5[0] * w
    f5[4] = f5[4] + 0.5 * f5[0] * w * w
    plan5 = amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk)
    plan7 = amr_plan(grid, dims, recon=recon, riemann=riemann, rk=rk, nvars=7)
    U5 = state_from(plan5, f5)
    U7 = state_from(plan7, with_scalars(f5, [w, np.full_like(w, 0.25)]))
    dx = dx_of(grid)
    for _ in range(6):
        dt = plan5.compute_dt(U5, dx, 0.4)
        assert dt == plan7.compute_dt(U7, dx, 0.4)
        plan5.advance(U5, dx, dt)
        plan7.advance(U7, dx, dt)
    I5, I7 = plan5.interior(U5), plan7.interior(U7)
    assert np.array_equal(I7[:5], I5)
    assert np.array_equal(I7[5], I7[3]) and np.abs(I7[3]).max() > 0.01
    assert np.max(np.abs(I7[6] - 0.25 * I7[0])) <= 2e-15  # a uniform abundance stays uniform
    fo, _ = plan7.status()
    assert fo == 0


@pytest.mark.parametrize("nbc,refined,dims,periodic", [((3, 3, 3), {(1, 1, 1)}, (8, 8, 8), True),
                                                        ((3, 3, 2), {(0, 0, 0), (1, 0, 0), (2, 2, 1)}, (8, 8, 8), True)])
def test_scalar_mass_is_conserved_through_jumps(nbc, refined, dims, periodic):
    grid = two_level_grid(nbc, refined, dims, periodic=periodic)
    L = [nbc[d] * dims[d] for d in range(3)]
    f5 = smooth_field(grid, dims, L)
    X = amr_zone_centres(grid, dims)
    xa = 0.5 + 0.4 * np.sin(2 * np.pi * X[:, 0] / L[0]) * np.cos(2 * np.pi * X[:, 2] / L[2])
    xb = (np.abs(X[:, 1] - 0.5 * L[1]) < 0.2 * L[1]).astype(float)  # a slab that crosses the refined region
    plan = amr_plan(grid, dims, nvars=7)
    U = state_from(plan, with_scalars(f5, [xa, xb]))
    dx = dx_of(grid)
    T0 = totals(plan, grid, U, 3)
    for _ in range(10):
        plan.advance(U, dx, plan.compute_dt(U, dx, 0.3))
    T1 = totals(plan, grid, U, 3)
    for v in (0, 4, 5, 6):
        assert abs(T1[v] - T0[v]) <= 1e-13 * T0[0], (v, T1[v] - T0[v])
    I = plan.interior(U)
    assert np.abs(I[6] - xb * I[0]).max() > 1e-3  # the slab moved
