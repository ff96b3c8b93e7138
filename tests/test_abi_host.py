"""CPU-side checks of the C ABI: the library loads, exports every symbol include/fx_hydro.h declares, and its
host logic (argument checks, layout, topology helper) agrees with the oracle's independent implementation."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from oracle import fxoracle as fxo
from paper_2208_11630_b200 import binding as fx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "fx_hydro.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(fx_[a-z0-9_]+)\s*\(", text)))


def test_library_exports_every_declared_symbol():
    L = fx.lib()
    syms = declared_symbols()
    assert len(syms) >= 18
    for s in syms:
        assert hasattr(L, s), s
    assert sorted(fx.EXPORTS) == syms


def test_enum_values_match_between_header_oracle_and_binding():
    text = open(os.path.join(ROOT, "include", "fx_hydro.h")).read()
    def val(name):
        m = re.search(r"\b%s\s*=\s*(-?\d+)" % name, text) or re.search(r"#define\s+%s\s+\(?(-?\d+)" % name, text)
        return int(m.group(1))
    for name in ("RECON_PLM_MINMOD", "RECON_WENO5", "RIEMANN_HLLE", "RIEMANN_HLLC", "BC_OUTFLOW", "BC_NONE",
                 "TOPO_PERIODIC", "TOPO_OUTFLOW", "TOPO_NONE", "ORDER_LEX", "ORDER_MORTON", "OPT_RHO_FLOOR",
                 "OPT_P_FLOOR", "OPT_WENO_EPS", "OPT_WAVESPEED"):
        assert val("FX_" + name) == getattr(fx, name) == getattr(fxo, name), name


def create(dims, g, nb, gamma=1.4, recon=0, riemann=1, rk=2, nvars=5):
    h = C.c_void_p()
    rc = fx.lib().fx_hydro_plan_create(C.byref(h), (C.c_int * 3)(*dims), g, nvars, nb, gamma, recon, riemann, rk)
    return rc, h


def test_plan_create_argument_checks():
    assert create((16, 16, 16), 4, 8)[0] == fx.OK
    assert create((16, 16, 16), 1, 8)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 2, 8, recon=1)[0] == fx.ERR_INVALID_ARG  # WENO5 needs 3
    assert create((2, 1, 1), 3, 8)[0] == fx.ERR_INVALID_ARG              # nguard > block dim
    assert create((16, 0, 1), 4, 8)[0] == fx.ERR_INVALID_ARG
    assert create((1, 1, 1), 2, 8)[0] == fx.ERR_INVALID_ARG              # no active dim
    assert create((16, 16, 16), 4, 8, gamma=1.0)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, 8, rk=4)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, 8, recon=2)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, 8, riemann=7)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, -1)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, 8, nvars=4)[0] == fx.ERR_INVALID_ARG
    assert create((16, 16, 16), 4, 8, nvars=33)[0] == fx.ERR_UNSUPPORTED   # more than 27 passive scalars [B11]
    assert b"nvars" in fx.lib().fx_last_error()
    rc, h = create((16, 16, 16), 4, 8, nvars=9)
    assert rc == 0 and fx.lib().fx_hydro_plan_path(h) == 0                  # scalars ride on the generic path
    L = fx.Layout()
    assert fx.lib().fx_hydro_plan_layout(h, C.byref(L)) == 0 and L.bytes_per_state == 9 * 8 * 24 ** 3 * 8
    fx.lib().fx_hydro_plan_destroy(h)


@pytest.mark.parametrize("dims,g,nb", [((16, 16, 16), 4, 32768), ((256, 1, 1), 4, 1), ((16, 16, 1), 4, 64), ((8, 8, 8), 3, 5)])
def test_layout_matches_oracle_and_closed_form(dims, g, nb):
    rc, h = create(dims, g, nb)
    assert rc == 0
    L = fx.Layout()
    assert fx.lib().fx_hydro_plan_layout(h, C.byref(L)) == 0
    o = fxo.OraclePlan(dims, g, nb, 1.4, 0, 1, 2)
    assert tuple(L.np) == o.np and tuple(L.gd) == o.gd
    assert (L.S_j, L.S_k, L.S_b, L.S_v, L.bytes_per_state) == (o.S_j, o.S_k, o.S_b, o.S_v, o.bytes_per_state)
    npd = [d + 2 * g if d > 1 else d for d in dims]
    assert L.S_b == npd[0] * npd[1] * npd[2] and L.bytes_per_state == 5 * 8 * nb * L.S_b
    # workspace = 256-byte scratch + 256-byte pad + (rk - 1) state copies (256-byte aligned) + z-segment table (12 ints per
    # block; 8 x 8 x nz blocks: room for one 76-int bundle segment per four blocks if that is more)
    seg_ints = nb * 12
    if dims[0] == 8 and dims[1] == 8:
        seg_ints = max(seg_ints, (nb // 4 + 1) * 76)
    seg = ((seg_ints * 4 + 255) // 256) * 256
    ws = fx.lib().fx_hydro_plan_workspace_bytes(h)
    assert ws == 512 + ((L.bytes_per_state + 255) // 256) * 256 + seg
    rc3, h3 = create(dims, g, nb, rk=3)
    assert fx.lib().fx_hydro_plan_workspace_bytes(h3) == 512 + 2 * (((L.bytes_per_state + 255) // 256) * 256) + seg


def test_config5_needs_64bit_indexing():
    rc, h = create((16, 16, 16), 4, 32768)
    L = fx.Layout()
    fx.lib().fx_hydro_plan_layout(h, C.byref(L))
    assert 5 * L.S_v > 2 ** 31 and L.bytes_per_state == 18119393280


@pytest.mark.parametrize("nb,lo,hi,order", [((4, 3, 2), (0, 1, 0), (0, 1, 0), 0), ((4, 4, 4), (0, 0, 0), (0, 0, 0), 1),
                                            ((5, 1, 1), (1, 2, 2), (0, 2, 2), 0), ((3, 5, 1), (0, 1, 2), (1, 0, 2), 1),
                                            ((1, 1, 1), (0, 0, 0), (0, 0, 0), 1)])
def test_topology_helper_matches_oracle(nb, lo, hi, order):
    n1, c1 = fx.fx_topology_cartesian(nb, lo, hi, order)
    n2, c2 = fxo.topology_cartesian(nb, lo, hi, order)
    assert np.array_equal(n1, n2) and np.array_equal(c1, c2)


def test_options_and_state_errors_without_gpu():
    rc, h = create((16, 16, 16), 4, 8)
    L = fx.lib()
    assert L.fx_hydro_plan_set_option(h, fx.OPT_WAVESPEED, 1.0) == 0
    assert L.fx_hydro_plan_set_option(h, fx.OPT_WAVESPEED, 2.0) == fx.ERR_INVALID_ARG
    assert L.fx_hydro_plan_set_option(h, 99, 0.0) == fx.ERR_INVALID_ARG
    assert L.fx_hydro_plan_set_option(h, fx.OPT_WENO_EPS, 0.0) == fx.ERR_INVALID_ARG
    # operations before topology / workspace are refused before any CUDA call is made
    assert L.fx_fill_guardcells(h, None, None) == fx.ERR_STATE
    assert L.fx_hydro_advance(h, None, None, 0.1, None) == fx.ERR_STATE
    assert L.fx_hydro_compute_dt(h, None, None, 0.3, None, None) == fx.ERR_STATE
    assert L.fx_hydro_plan_set_workspace(h, C.c_void_p(8), 1 << 30) == fx.ERR_WORKSPACE  # misaligned
    assert L.fx_hydro_plan_set_workspace(h, C.c_void_p(256), 16) == fx.ERR_WORKSPACE     # too small


def test_shard_partition_lists_agree_between_ranks():
    """fx_shard_* (host index logic): contiguous runs that cover the order; what rank p sends to q is, item for item and in
    the same order, what q expects from p (global block id, side); ghosts are exactly the foreign neighbours of the owned
    blocks; a ghost row names no neighbour; on an irregular table too (one-sided links, outflow, walls)."""
    import numpy as np
    from paper_2208_11630_b200 import binding as fx
    per, out = fx.TOPO_PERIODIC, fx.TOPO_OUTFLOW
    neigh, coords = fx.fx_topology_cartesian((4, 3, 5), (per, out, per), (per, fx.TOPO_REFLECT, per), fx.ORDER_MORTON)
    neigh = np.array(neigh, np.int32)
    neigh[7, 1] = fx.BC_OUTFLOW  # a one-sided cut link
    N = neigh.shape[0]
    for world in (1, 2, 3, 7):
        shards = [fx.Shard(neigh, world, r) for r in range(world)]
        assert [s.owned_begin for s in shards] == [N * r // world for r in range(world)]
        assert sum(s.n_owned for s in shards) == N
        for q, s in enumerate(shards):
            own = set(range(s.owned_begin, s.owned_begin + s.n_owned))
            foreign = {int(g) for b in own for g in neigh[b] if g >= 0 and g not in own}
            assert set(s.global_id[s.n_owned:].tolist()) == foreign and list(s.global_id[:s.n_owned]) == sorted(own)
            assert (s.neigh_local[s.n_owned:] == fx.BC_OUTFLOW).all()
            # local table = global table through the numbering
            back = np.where(s.neigh_local[:s.n_owned] >= 0, s.global_id[np.maximum(s.neigh_local[:s.n_owned], 0)], s.neigh_local[:s.n_owned])
            assert np.array_equal(back, neigh[s.owned_begin:s.owned_begin + s.n_owned])
            ro = np.concatenate([[0], np.cumsum(s.recv_counts)])
            for p, t in enumerate(shards):
                so = np.concatenate([[0], np.cumsum(t.send_counts)])
                recv = [(int(s.global_id[b]), int(sd)) for b, sd in s.recv_items[ro[p]:ro[p + 1]]]
                send = [(int(t.global_id[b]), int(sd)) for b, sd in t.send_items[so[q]:so[q + 1]]]
                assert recv == send and recv == sorted(set(recv))
                assert all(b < t.n_owned for b, _ in t.send_items[so[q]:so[q + 1]])
            assert all(b >= s.n_owned for b, _ in s.recv_items)
