"""The two-level workload generator of bench.py --amr (paper_2208_11630_b200/inputs.py): its tables against the test helper
written separately from the same definition (tests/helpers.two_level_grid), and the coarse field's recipe."""
import numpy as np
import pytest

from paper_2208_11630_b200 import inputs
from tests.helpers import two_level_grid


@pytest.mark.parametrize("nbc,lo,hi", [((4, 4, 3), (1, 1, 0), (3, 2, 2)), ((3, 3, 3), (1, 1, 1), (2, 2, 2)), ((4, 2, 2), (0, 0, 0), (2, 2, 1))])
def test_two_level_tiling_tables(nbc, lo, hi):
    g = inputs.two_level_tiling(nbc, lo, hi, order=inputs.ORDER_LEX)
    ref = {(x, y, z) for x in range(lo[0], hi[0]) for y in range(lo[1], hi[1]) for z in range(lo[2], hi[2])}
    h = two_level_grid(nbc, ref, (16, 16, 16))
    assert np.array_equal(g["neigh"], h["neigh"]) and np.array_equal(g["jump"], h["jump"]) and np.array_equal(g["level"], h["level"])
    assert np.array_equal(g["fine"], (2 * h["cell"] + h["child"]))
    # Morton order: the same grid, blocks permuted -- every relation maps back
    m = inputs.two_level_tiling(nbc, lo, hi, order=inputs.ORDER_MORTON)
    key = {tuple(f) + (int(l),): i for i, (f, l) in enumerate(zip(m["fine"], m["level"]))}
    perm = np.array([key[tuple(f) + (int(l),)] for f, l in zip(g["fine"], g["level"])])
    for b in range(len(perm)):
        for f in range(6):
            v, w = g["neigh"][b, f], m["neigh"][perm[b], f]
            assert (w == perm[v]) if v >= 0 else (w == v)
            if v == inputs.NEIGH_FINER:
                assert np.array_equal(m["jump"][perm[b], f], perm[g["jump"][b, f]])
            if v == inputs.NEIGH_COARSER:
                assert m["jump"][perm[b], f, 0] == perm[g["jump"][b, f, 0]] and m["jump"][perm[b], f, 1] == g["jump"][b, f, 1]


def test_two_level_interiors_are_the_fine_field_and_its_means():
    nbc, lo, hi = (3, 3, 3), (1, 1, 1), (2, 2, 2)
    g = inputs.two_level_tiling(nbc, lo, hi, order=inputs.ORDER_LEX)
    fine = inputs.config(5, nb=(6, 6, 6))
    n = len(g["level"])
    I = inputs.two_level_interiors(fine, g, 0, n).numpy()
    b = int(np.nonzero(g["level"] == 1)[0][3])
    assert np.array_equal(I[:, b], inputs.block_interiors(fine, g["fine"][b:b + 1]).numpy()[:, 0])
    c = int(np.nonzero(g["level"] == 0)[0][5])
    kids = np.zeros((5, 32, 32, 32))
    for cz in range(2):
        for cy in range(2):
            for cx in range(2):
                k = inputs.block_interiors(fine, g["fine"][c:c + 1] + np.array([[cx, cy, cz]], np.int32)).numpy()[:, 0]
                kids[:, 16 * cz:16 * cz + 16, 16 * cy:16 * cy + 16, 16 * cx:16 * cx + 16] = k
    want = kids.reshape(5, 16, 2, 16, 2, 16, 2).mean(axis=(2, 4, 6))
    assert np.allclose(I[:, c], want, rtol=1e-14, atol=0)
    # chunked generation gives the same bytes
    assert np.array_equal(inputs.two_level_interiors(fine, g, 7, 19).numpy(), I[:, 7:19])
