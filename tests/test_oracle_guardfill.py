"""O1 guard fill: the hop definition must equal the global wrap/clamp definition on regular tilings
(SURVEY.md 8(c)-i O1, 8(c)-iii row 'O1').  The global definition is written here in numpy and shares
nothing with oracle/fxoracle.c."""
import itertools

import numpy as np
import pytest

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import inputs


def global_definition_map(dims, g, nb, bc_lo, bc_hi, coords):
    """For each padded zone of each block: flat var-0 index of the interior zone that owns the global
    index origin(b) + (i,j,k) - g mapped per dimension by wrap (periodic), clamp (outflow) or mirror about the
    domain face (reflecting wall [B9]: global index -1-m images m, N+m images N-1-m)."""
    nblocks = coords.shape[0]
    gd = [g if dims[d] > 1 else 0 for d in range(3)]
    npd = [dims[d] + 2 * gd[d] for d in range(3)]
    S_j, S_k = npd[0], npd[0] * npd[1]
    S_b = S_k * npd[2]
    id_of = {tuple(int(x) for x in coords[b]): b for b in range(nblocks)}
    out = np.empty((nblocks, npd[2], npd[1], npd[0]), np.int64)
    for b in range(nblocks):
        for k, j, i in itertools.product(range(npd[2]), range(npd[1]), range(npd[0])):
            loc = [i, j, k]
            blk, cell = [0, 0, 0], [0, 0, 0]
            for d in range(3):
                N = dims[d] * nb[d]
                G = int(coords[b, d]) * dims[d] + loc[d] - gd[d]
                if G < 0:
                    G = G % N if bc_lo[d] == fxo.TOPO_PERIODIC else (-1 - G if bc_lo[d] == fxo.TOPO_REFLECT else 0)
                elif G >= N:
                    G = G % N if bc_hi[d] == fxo.TOPO_PERIODIC else (2 * N - 1 - G if bc_hi[d] == fxo.TOPO_REFLECT else N - 1)
                blk[d], cell[d] = G // dims[d], G % dims[d] + gd[d]
            out[b, k, j, i] = id_of[tuple(blk)] * S_b + cell[2] * S_k + cell[1] * S_j + cell[0]
    return out


CASES = [
    ((4, 4, 4), 2, (2, 2, 2), "ppp", fxo.ORDER_LEX),
    ((4, 4, 4), 4, (2, 2, 2), "ppp", fxo.ORDER_MORTON),  # nguard == block size
    ((6, 4, 5), 3, (3, 1, 2), "pop", fxo.ORDER_LEX),      # single block in a periodic direction... and outflow in y
    ((5, 4, 4), 4, (3, 1, 2), "opo", fxo.ORDER_MORTON),   # a block that is its own periodic neighbour (y)
    ((8, 6, 1), 3, (2, 3, 1), "po-", fxo.ORDER_LEX),      # 2-D
    ((12, 1, 1), 4, (3, 1, 1), "o--", fxo.ORDER_LEX),     # 1-D outflow
    ((12, 1, 1), 4, (1, 1, 1), "p--", fxo.ORDER_LEX),     # 1-D, one block, periodic with itself
    ((12, 1, 1), 4, (2, 1, 1), "r--", fxo.ORDER_LEX),     # 1-D between two reflecting walls
    ((4, 4, 4), 4, (2, 1, 2), "rpr", fxo.ORDER_MORTON),   # walls in x and z, nguard == block size
    ((6, 4, 5), 3, (2, 2, 1), "orr", fxo.ORDER_LEX),      # outflow in x, walls in y and z (one block between two walls)
]


def bcs(spec, hi_spec=None):
    m = {"p": fxo.TOPO_PERIODIC, "o": fxo.TOPO_OUTFLOW, "-": fxo.TOPO_NONE, "r": fxo.TOPO_REFLECT}
    return [m[c] for c in spec]


@pytest.mark.parametrize("dims,g,nb,spec,order", CASES)
def test_hop_map_equals_global_definition(dims, g, nb, spec, order):
    bc = bcs(spec)
    neigh, coords = fxo.topology_cartesian(nb, bc, bc, order)
    # the inputs module's block ordering agrees with the oracle's helper
    assert np.array_equal(coords, inputs.block_coords(nb, order))
    plan = fxo.OraclePlan(dims, g, neigh.shape[0], 1.4, 0, 1, 2)
    plan.set_topology(neigh)
    got = plan.index_map()
    ref = global_definition_map(dims, g, nb, bc, bc, coords)
    assert np.array_equal(got, ref)


def test_mixed_lo_hi_boundaries_and_permutation():
    dims, g, nb = (4, 5, 4), 3, (2, 2, 2)
    lo = [fxo.TOPO_OUTFLOW, fxo.TOPO_PERIODIC, fxo.TOPO_OUTFLOW]
    hi = [fxo.TOPO_OUTFLOW, fxo.TOPO_PERIODIC, fxo.TOPO_OUTFLOW]
    neigh, coords = fxo.topology_cartesian(nb, lo, hi, fxo.ORDER_LEX)
    plan = fxo.OraclePlan(dims, g, 8, 1.4, 0, 1, 2)
    plan.set_topology(neigh)
    ref = global_definition_map(dims, g, nb, lo, hi, coords)
    assert np.array_equal(plan.index_map(), ref)
    # permute block ids: new id p[b]; table permuted accordingly [A19]
    rng = np.random.default_rng(5)
    perm = rng.permutation(8)  # new block q holds old block perm[q]
    inv = np.argsort(perm)
    neigh_p = neigh[perm].copy()
    neigh_p[neigh_p >= 0] = inv[neigh_p[neigh_p >= 0]]
    plan_p = fxo.OraclePlan(dims, g, 8, 1.4, 0, 1, 2)
    plan_p.set_topology(neigh_p)
    ref_p = global_definition_map(dims, g, nb, lo, hi, coords[perm])
    assert np.array_equal(plan_p.index_map(), ref_p)


def test_fill_copies_data_by_the_map_and_is_idempotent():
    dims, g, nb = (4, 4, 4), 3, (2, 2, 1)
    bc = bcs("pop")
    neigh, coords = fxo.topology_cartesian(nb, bc, bc, fxo.ORDER_LEX)
    plan = fxo.OraclePlan(dims, g, 4, 1.4, 0, 1, 2)
    plan.set_topology(neigh)
    rng = np.random.default_rng(7)
    U = rng.normal(size=plan.shape)
    Ui = plan.interior(U).copy()
    V = np.full(plan.shape, np.nan)
    plan.interior(V)[...] = Ui
    plan.fill_guardcells(V)
    src = plan.index_map()
    for v in range(5):
        flat = V[v].reshape(-1)
        assert np.array_equal(flat[src.reshape(-1)].reshape(V[v].shape), V[v])  # every zone equals its source
    assert np.array_equal(plan.interior(V), Ui)  # interior untouched
    W = V.copy()
    plan.fill_guardcells(W)
    assert np.array_equal(W, V)


def test_index_map_block_range_and_errors():
    dims, g, nb = (4, 4, 1), 2, (3, 2, 1)
    bc = bcs("pp-")
    neigh, _ = fxo.topology_cartesian(nb, bc, bc, fxo.ORDER_LEX)
    plan = fxo.OraclePlan(dims, g, 6, 1.4, 0, 1, 2)
    U = np.zeros(plan.shape)
    with pytest.raises(RuntimeError):
        plan.fill_guardcells(U)  # topology not set
    plan.set_topology(neigh)
    full = plan.index_map()
    assert np.array_equal(plan.index_map(2, 3), full[2:5])
    bad = neigh.copy()
    bad[0, 0] = -2  # BC_NONE in an active dimension = a coarse/fine relation: unsupported
    with pytest.raises(ValueError):
        plan.set_topology(bad)


def test_reflecting_wall_images_and_momentum_signs():
    """[B9] A reflecting wall: guard zone -1-m holds interior zone m with the momentum normal to the wall negated;
    an edge / corner guard zone behind two or three walls has each of those components negated; density, energy and
    the tangential momenta are copied.  Checked against the mirrored global field built in numpy."""
    dims, g, nb = (4, 5, 3), 3, (2, 1, 2)
    lo = [fxo.TOPO_REFLECT, fxo.TOPO_REFLECT, fxo.TOPO_OUTFLOW]
    hi = [fxo.TOPO_OUTFLOW, fxo.TOPO_REFLECT, fxo.TOPO_REFLECT]
    neigh, coords = fxo.topology_cartesian(nb, lo, hi, fxo.ORDER_LEX)
    assert neigh[0, 0] == fxo.BC_REFLECT and neigh[0, 2] == fxo.BC_REFLECT and neigh[0, 3] == fxo.BC_REFLECT
    plan = fxo.OraclePlan(dims, g, 4, 1.4, 0, 1, 2)
    plan.set_topology(neigh)
    rng = np.random.default_rng(3)
    N = [dims[d] * nb[d] for d in range(3)]
    G = rng.normal(size=(5, N[2], N[1], N[0]))  # global field
    U = np.full(plan.shape, np.nan)
    Ui = plan.interior(U)
    for b, (bx, by, bz) in enumerate(coords):
        Ui[:, b] = G[:, bz * dims[2]:(bz + 1) * dims[2], by * dims[1]:(by + 1) * dims[1], bx * dims[0]:(bx + 1) * dims[0]]
    plan.fill_guardcells(U)

    def image(d, G_):  # global index of dimension d (0 = x) -> (source index, sign flip)
        n = N[d]
        if G_ < 0:
            return (-1 - G_, True) if lo[d] == fxo.TOPO_REFLECT else (0, False)
        if G_ >= n:
            return (2 * n - 1 - G_, True) if hi[d] == fxo.TOPO_REFLECT else (n - 1, False)
        return G_, False

    for b, (bx, by, bz) in enumerate(coords):
        for k, j, i in itertools.product(range(dims[2] + 2 * g), range(dims[1] + 2 * g), range(dims[0] + 2 * g)):
            (sx, fx_), (sy, fy_), (sz, fz_) = (image(0, bx * dims[0] + i - g), image(1, by * dims[1] + j - g),
                                               image(2, bz * dims[2] + k - g))
            ref = G[:, sz, sy, sx].copy()
            for comp, f in ((1, fx_), (2, fy_), (3, fz_)):
                if f:
                    ref[comp] = -ref[comp]
            assert np.array_equal(U[:, b, k, j, i], ref), (b, k, j, i)
