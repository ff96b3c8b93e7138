"""Thin ctypes binding of libfxhydro.so (include/fx_hydro.h): argument marshalling only.

Every step of the path runs inside the CUDA library; PyTorch supplies device memory and streams.  There is
no CPU fallback: a missing library or a failing call raises.  Names mirror the C ABI.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libfxhydro.so")

OK, ERR_INVALID_ARG, ERR_STATE, ERR_UNSUPPORTED, ERR_WORKSPACE, ERR_CUDA = 0, -1, -2, -3, -4, -5
RECON_PLM_MINMOD, RECON_WENO5 = 0, 1
RIEMANN_HLLE, RIEMANN_HLLC = 0, 1
BC_OUTFLOW, BC_NONE, BC_REFLECT = -1, -2, -3
PART_INNER, PART_BOUNDARY = 1, 2
NEIGH_COARSER, NEIGH_FINER = -4, -5
TOPO_PERIODIC, TOPO_OUTFLOW, TOPO_NONE, TOPO_REFLECT = 0, 1, 2, 3
ORDER_LEX, ORDER_MORTON = 0, 1
OPT_RHO_FLOOR, OPT_P_FLOOR, OPT_WENO_EPS, OPT_WAVESPEED, OPT_PATH, OPT_ZCHAIN = 0, 1, 2, 3, 4, 5
OPT_GRAVITY_X, OPT_GRAVITY_Y, OPT_GRAVITY_Z, OPT_GUARD_X, OPT_OWNED_BLOCKS = 6, 7, 8, 9, 10
STATUS_NONFINITE, STATUS_RHO_FLOOR, STATUS_P_FLOOR, STATUS_WENO_FALLBACK = 1, 2, 4, 8

EXPORTS = [
    "fx_last_error", "fx_hydro_plan_create", "fx_hydro_plan_destroy", "fx_hydro_plan_layout",
    "fx_hydro_plan_set_option", "fx_hydro_plan_workspace_bytes", "fx_hydro_plan_set_workspace",
    "fx_hydro_plan_set_topology", "fx_hydro_plan_set_refinement", "fx_topology_cartesian", "fx_fill_guardcells", "fx_guardcell_index_map",
    "fx_hydro_compute_dt", "fx_hydro_compute_dt_static", "fx_hydro_advance", "fx_hydro_advance_host", "fx_hydro_advance_host_interior", "fx_hydro_advance_devdt", "fx_hydro_advance_ca", "fx_hydro_step",
    "fx_hydro_status", "fx_hydro_status_reset", "fx_debug_compute_fluxes", "fx_hydro_plan_path",
    "fx_hydro_plan_set_timing", "fx_hydro_plan_get_timing",
    "fx_shard_create", "fx_shard_destroy", "fx_shard_sizes", "fx_shard_tables", "fx_shard_items", "fx_halo_item_elems",
    "fx_halo_pack", "fx_halo_unpack", "fx_hydro_advance_stage", "fx_hydro_stage_arrays",
    "fx_hydro_advance_stage_part", "fx_hydro_plan_stage_parts",
]


class FxError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"libfxhydro error {code}: {msg}")
        self.code = code


class Layout(C.Structure):
    _fields_ = [("np", C.c_int32 * 3), ("gd", C.c_int32 * 3), ("S_j", C.c_int64), ("S_k", C.c_int64),
                ("S_b", C.c_int64), ("S_v", C.c_int64), ("bytes_per_state", C.c_int64)]


_lib = None


def lib():
    """Load libfxhydro.so; raises if it has not been built (no fallback)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise ImportError(f"{LIB_PATH} is missing: run `python -m paper_2208_11630_b200.build` "
                              "(the CUDA library is the only implementation; there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        vp, i3 = C.c_void_p, C.POINTER(C.c_int)
        L.fx_last_error.restype = C.c_char_p
        L.fx_hydro_plan_create.argtypes = [C.POINTER(vp), i3, C.c_int, C.c_int, C.c_int64, C.c_double, C.c_int,
                                           C.c_int, C.c_int]
        L.fx_hydro_plan_destroy.argtypes = [vp]
        L.fx_hydro_plan_layout.argtypes = [vp, C.POINTER(Layout)]
        L.fx_hydro_plan_set_option.argtypes = [vp, C.c_int, C.c_double]
        L.fx_hydro_plan_workspace_bytes.argtypes = [vp]
        L.fx_hydro_plan_workspace_bytes.restype = C.c_size_t
        L.fx_hydro_plan_set_workspace.argtypes = [vp, vp, C.c_size_t]
        L.fx_hydro_plan_set_topology.argtypes = [vp, vp]
        L.fx_hydro_plan_set_refinement.argtypes = [vp, vp]
        L.fx_topology_cartesian.argtypes = [i3, i3, i3, C.c_int, vp, vp]
        L.fx_fill_guardcells.argtypes = [vp, vp, vp]
        L.fx_guardcell_index_map.argtypes = [vp, C.c_int64, C.c_int64, vp, vp]
        L.fx_hydro_compute_dt.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.fx_hydro_compute_dt_static.argtypes = [vp, vp, vp, C.c_double, vp, vp, vp]
        L.fx_hydro_advance.argtypes = [vp, vp, vp, C.c_double, vp]
        L.fx_hydro_advance_devdt.argtypes = [vp, vp, vp, vp, vp]
        L.fx_hydro_advance_ca.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.fx_hydro_step.argtypes = [vp, vp, vp, C.c_double, vp, vp]
        L.fx_hydro_advance_host.argtypes = [vp, vp, vp, C.c_double, C.c_int, vp, vp, vp, vp]
        L.fx_hydro_advance_host_interior.argtypes = [vp, vp, vp, C.c_double, C.c_int, vp, vp, vp, vp, vp]
        L.fx_hydro_status.argtypes = [vp, C.POINTER(C.c_uint32), C.POINTER(C.c_ulonglong), vp]
        L.fx_hydro_status_reset.argtypes = [vp, vp]
        L.fx_debug_compute_fluxes.argtypes = [vp, vp, C.c_int, vp, vp]
        L.fx_hydro_plan_path.argtypes = [vp]
        L.fx_hydro_plan_set_timing.argtypes = [vp, C.c_int]
        L.fx_hydro_plan_get_timing.argtypes = [vp, C.POINTER(C.c_double), C.POINTER(C.c_longlong)]
        p64 = C.POINTER(C.c_int64)
        L.fx_shard_create.argtypes = [C.POINTER(vp), C.c_int64, vp, C.c_int, C.c_int]
        L.fx_shard_destroy.argtypes = [vp]
        L.fx_shard_sizes.argtypes = [vp, p64, p64, p64, p64, p64]
        L.fx_shard_tables.argtypes = [vp, vp, vp]
        L.fx_shard_items.argtypes = [vp, vp, vp, vp, vp]
        L.fx_halo_item_elems.argtypes = [vp, C.c_int]
        L.fx_halo_item_elems.restype = C.c_int64
        L.fx_halo_pack.argtypes = [vp, vp, vp, vp, C.c_int64, vp, vp]
        L.fx_halo_unpack.argtypes = [vp, vp, vp, vp, C.c_int64, vp, vp]
        L.fx_hydro_advance_stage.argtypes = [vp, vp, vp, C.c_double, vp, C.c_int, C.c_double, vp, vp]
        L.fx_hydro_stage_arrays.argtypes = [vp, vp, C.c_int, C.POINTER(vp), C.POINTER(vp)]
        L.fx_hydro_advance_stage_part.argtypes = [vp, vp, vp, C.c_double, vp, C.c_int, C.c_int, C.c_double, vp, vp]
        L.fx_hydro_plan_stage_parts.argtypes = [vp, C.POINTER(C.c_int64), C.POINTER(C.c_int64)]
        _lib = L
    return _lib


def _check(rc):
    if rc != 0:
        raise FxError(rc, lib().fx_last_error().decode())


def _stream(stream=None):
    s = torch.cuda.current_stream() if stream is None else stream
    return C.c_void_p(s.cuda_stream)


STATIC_DT_MAX_BLOCKS = 65536  # FX_STATIC_DT_MAX_BLOCKS: owned blocks fx_hydro_compute_dt_static's scratch array has room for


def _dev(t: torch.Tensor, dtype):
    assert t.is_cuda and t.dtype == dtype and t.is_contiguous(), (t.device, t.dtype, t.is_contiguous())
    return C.c_void_p(t.data_ptr())


def fx_topology_cartesian(nb, bc_lo, bc_hi, order=ORDER_LEX):
    """Host helper: (neigh int32 [nblocks,6], coords int32 [nblocks,3]) numpy arrays."""
    n = int(nb[0]) * int(nb[1]) * int(nb[2])
    neigh = np.empty((max(n, 0), 6), np.int32)
    coords = np.empty((max(n, 0), 3), np.int32)
    i3 = C.c_int * 3
    _check(lib().fx_topology_cartesian(i3(*nb), i3(*bc_lo), i3(*bc_hi), order, C.c_void_p(neigh.ctypes.data),
                                       C.c_void_p(coords.ctypes.data)))
    return neigh, coords


class Shard:
    """fx_shard: rank `rank`'s part of a block batch cut into `nranks` contiguous runs (host index logic only; no GPU).
    Attributes: owned_begin, n_owned, n_ghost, neigh_local int32 [n_local, 6], global_id int64 [n_local],
    send_items / recv_items int32 [n, 2] (local block, side), send_counts / recv_counts int64 [nranks] (items per peer)."""

    def __init__(self, neigh_global, nranks, rank):
        neigh_global = np.ascontiguousarray(neigh_global, np.int32)
        self._h = C.c_void_p()
        _check(lib().fx_shard_create(C.byref(self._h), neigh_global.shape[0], C.c_void_p(neigh_global.ctypes.data), nranks, rank))
        v = [C.c_int64() for _ in range(5)]
        _check(lib().fx_shard_sizes(self._h, *[C.byref(x) for x in v]))
        self.owned_begin, self.n_owned, self.n_ghost, n_send, n_recv = (int(x.value) for x in v)
        self.n_local, self.nranks, self.rank = self.n_owned + self.n_ghost, nranks, rank
        self.neigh_local = np.empty((self.n_local, 6), np.int32)
        self.global_id = np.empty(self.n_local, np.int64)
        _check(lib().fx_shard_tables(self._h, C.c_void_p(self.neigh_local.ctypes.data), C.c_void_p(self.global_id.ctypes.data)))
        self.send_items, self.recv_items = np.empty((n_send, 2), np.int32), np.empty((n_recv, 2), np.int32)
        self.send_counts, self.recv_counts = np.empty(nranks, np.int64), np.empty(nranks, np.int64)
        _check(lib().fx_shard_items(self._h, C.c_void_p(self.send_items.ctypes.data), C.c_void_p(self.send_counts.ctypes.data),
                                    C.c_void_p(self.recv_items.ctypes.data), C.c_void_p(self.recv_counts.ctypes.data)))

    def __del__(self):
        try:
            if getattr(self, "_h", None) and self._h.value:
                lib().fx_shard_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:  # interpreter shutdown
            pass


def _ptr(x, dtype=torch.float64):
    """A device tensor or a raw device address (the stage copies live inside the workspace)."""
    return C.c_void_p(int(x)) if isinstance(x, int) else _dev(x, dtype)


class HydroPlan:
    """fx_hydro_plan with its caller-owned device buffers (workspace, neighbour table) held as torch tensors."""

    def __init__(self, block_dims, nguard, nblocks, gamma, recon, riemann, rk_order, nvars=5, device="cuda"):
        self._h = C.c_void_p()
        _check(lib().fx_hydro_plan_create(C.byref(self._h), (C.c_int * 3)(*block_dims), nguard, nvars, nblocks, gamma,
                                          recon, riemann, rk_order))
        self.block_dims = tuple(int(d) for d in block_dims)
        self.nblocks, self.nvars, self.gamma, self.rk_order = int(nblocks), nvars, gamma, rk_order
        self._read_layout()
        self.device = torch.device(device)
        self._ws = None
        self._neigh = None
        self._dt = None

    def __del__(self):
        if getattr(self, "_h", None) is not None and self._h.value and _lib is not None:
            try:  # at interpreter shutdown module globals may already be gone
                _lib.fx_hydro_plan_destroy(self._h)
            except Exception:
                pass
            self._h = C.c_void_p()

    def _read_layout(self):
        L = Layout()
        _check(lib().fx_hydro_plan_layout(self._h, C.byref(L)))
        self.np, self.gd = tuple(L.np), tuple(L.gd)
        self.S_j, self.S_k, self.S_b, self.S_v = L.S_j, L.S_k, L.S_b, L.S_v
        self.bytes_per_state = L.bytes_per_state

    def alloc_state(self, fill=None, device=None, pin_memory=False):
        """A state array `shape` placed so that its interior rows start on a 128-byte boundary where the row pitch allows
        it (include/fx_hydro.h, "Layout and DRAM lines"): any placement is correct, this one reads no guard bytes."""
        n = int(np.prod(self.shape))
        off = ((128 - (8 * self.gd[0]) % 128) % 128) // 8
        dev = self.device if device is None else torch.device(device)
        buf = torch.empty(n + 16, dtype=torch.float64, device=dev, pin_memory=pin_memory)
        assert buf.data_ptr() % 128 == 0
        U = buf[off:off + n].view(self.shape)
        if fill is not None:
            U.fill_(fill)
        return U

    def embed(self, interior, guard_value=float("nan")):
        """Device state array (alloc_state placement) holding `interior` [5][nblocks][nz][ny][nx]; guard zones get
        guard_value (NaN: the advance must not depend on them)."""
        U = self.alloc_state(fill=guard_value)
        self.interior(U).copy_(torch.as_tensor(interior).to(self.device))
        return U

    @property
    def shape(self):
        return (self.nvars, self.nblocks, self.np[2], self.np[1], self.np[0])

    @property
    def path(self):
        return lib().fx_hydro_plan_path(self._h)

    def fx_hydro_plan_set_option(self, key, value):
        _check(lib().fx_hydro_plan_set_option(self._h, key, float(value)))
        if key == OPT_GUARD_X:
            self._read_layout()  # the option changes np[0] and the strides

    def fx_hydro_plan_workspace_bytes(self):
        return int(lib().fx_hydro_plan_workspace_bytes(self._h))

    def fx_hydro_plan_set_workspace(self, ws: torch.Tensor | None = None):
        if ws is None:
            ws = torch.empty(self.fx_hydro_plan_workspace_bytes(), dtype=torch.uint8, device=self.device)
        assert ws.is_cuda and ws.dtype == torch.uint8
        _check(lib().fx_hydro_plan_set_workspace(self._h, C.c_void_p(ws.data_ptr()), ws.numel()))
        self._ws = ws
        self._dt = torch.empty(1, dtype=torch.float64, device=self.device)

    def fx_hydro_plan_set_refinement(self, jump):
        """Refinement-jump table int32 [nblocks, 6, 4] (numpy or tensor) [B12]; before workspace and topology."""
        t = torch.as_tensor(np.ascontiguousarray(jump, np.int32) if not isinstance(jump, torch.Tensor) else jump).to(self.device).contiguous()
        _check(lib().fx_hydro_plan_set_refinement(self._h, _dev(t, torch.int32)))
        self._jump = t  # caller-owned device memory: keep it alive

    def fx_hydro_plan_set_topology(self, neigh):
        if not isinstance(neigh, torch.Tensor):
            neigh = torch.as_tensor(np.ascontiguousarray(neigh, np.int32))
        neigh = neigh.to(self.device, torch.int32).contiguous().reshape(self.nblocks, 6)
        _check(lib().fx_hydro_plan_set_topology(self._h, C.c_void_p(neigh.data_ptr())))
        self._neigh = neigh  # caller-owned table must outlive the plan's use of it

    def fx_fill_guardcells(self, U, stream=None):
        _check(lib().fx_fill_guardcells(self._h, _dev(U, torch.float64), _stream(stream)))

    def fx_guardcell_index_map(self, block_begin=0, block_count=None, stream=None):
        if block_count is None:
            block_count = self.nblocks - block_begin
        src = torch.empty((block_count, self.np[2], self.np[1], self.np[0]), dtype=torch.int64, device=self.device)
        _check(lib().fx_guardcell_index_map(self._h, block_begin, block_count, C.c_void_p(src.data_ptr()), _stream(stream)))
        return src

    def fx_hydro_compute_dt(self, U, dx, cfl, dt_out=None, stream=None):
        """Enqueues the reduction; returns the 1-element device tensor holding dt (no sync)."""
        dt_out = self._dt if dt_out is None else dt_out
        _check(lib().fx_hydro_compute_dt(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), float(cfl),
                                         _dev(dt_out, torch.float64), _stream(stream)))
        return dt_out

    def fx_hydro_advance_ca(self, U, dx, dt, stream=None):
        """The communication-avoiding step: one guard fill, stages on a shrinking extension of the interior.  dt: a float,
        or a 1-element device tensor read on the device."""
        if isinstance(dt, torch.Tensor):
            _check(lib().fx_hydro_advance_ca(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), 0.0,
                                             _dev(dt, torch.float64), _stream(stream)))
        else:
            _check(lib().fx_hydro_advance_ca(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), float(dt), None,
                                             _stream(stream)))

    def fx_hydro_compute_dt_static(self, U, dx, cfl, dt_out, flags_out=None, stream=None):
        """The reduction with its scratch in the library's static device array (no workspace, no allocation: the caller
        passes dt_out, a 1-element float64 device tensor, and optionally flags_out, a 1-element int32 device tensor)."""
        _check(lib().fx_hydro_compute_dt_static(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), float(cfl),
                                                _dev(dt_out, torch.float64),
                                                None if flags_out is None else _dev(flags_out, torch.int32), _stream(stream)))
        return dt_out

    def fx_hydro_advance(self, U, dx, dt, stream=None):
        if isinstance(dt, torch.Tensor):
            _check(lib().fx_hydro_advance_devdt(self._h, _dev(U, torch.float64), _dev(dx, torch.float64),
                                                _dev(dt, torch.float64), _stream(stream)))
        else:
            _check(lib().fx_hydro_advance(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), float(dt),
                                          _stream(stream)))

    def fx_hydro_step(self, U, dx, cfl, dt, stream=None):
        """Advance by the device-resident dt (a 1-element float64 CUDA tensor) and overwrite it with the next step's dt."""
        _check(lib().fx_hydro_step(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), float(cfl),
                                   _dev(dt, torch.float64), _stream(stream)))

    def fx_hydro_stage_arrays(self, U, stage):
        """(address of the array stage `stage` reads, address of the one it writes): U or a stage copy in the workspace."""
        a, b = C.c_void_p(), C.c_void_p()
        _check(lib().fx_hydro_stage_arrays(self._h, _dev(U, torch.float64), stage, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def fx_hydro_advance_stage(self, U, dx, dt, stage, cfl_next=0.0, dt_next=None, stream=None):
        """One RK stage; dt a float or a device scalar; dt_next (last stage): device scalar receiving the next time step."""
        on_dev = isinstance(dt, torch.Tensor)
        _check(lib().fx_hydro_advance_stage(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), 0.0 if on_dev else float(dt),
                                            _dev(dt, torch.float64) if on_dev else None, stage, float(cfl_next),
                                            _dev(dt_next, torch.float64) if dt_next is not None else None, _stream(stream)))

    def fx_hydro_advance_stage_part(self, U, dx, dt, stage, part, cfl_next=0.0, dt_next=None, stream=None):
        """One part (PART_INNER: the owned blocks that read no ghost zone; PART_BOUNDARY: the others) of one RK stage."""
        on_dev = isinstance(dt, torch.Tensor)
        _check(lib().fx_hydro_advance_stage_part(self._h, _dev(U, torch.float64), _dev(dx, torch.float64), 0.0 if on_dev else float(dt),
                                                 _dev(dt, torch.float64) if on_dev else None, stage, part, float(cfl_next),
                                                 _dev(dt_next, torch.float64) if dt_next is not None else None, _stream(stream)))

    def fx_hydro_plan_stage_parts(self):
        """(owned blocks advanced by PART_INNER, by PART_BOUNDARY)."""
        a, b = C.c_int64(0), C.c_int64(0)
        _check(lib().fx_hydro_plan_stage_parts(self._h, C.byref(a), C.byref(b)))
        return int(a.value), int(b.value)

    def fx_halo_item_elems(self, side):
        return int(lib().fx_halo_item_elems(self._h, side))

    def fx_halo_pack(self, U, items, offsets, buf, stream=None):
        _check(lib().fx_halo_pack(self._h, _ptr(U), _dev(items, torch.int32), _dev(offsets, torch.int64), items.shape[0],
                                  _dev(buf, torch.float64), _stream(stream)))

    def fx_halo_unpack(self, U, items, offsets, buf, stream=None):
        _check(lib().fx_halo_unpack(self._h, _ptr(U), _dev(items, torch.int32), _dev(offsets, torch.int64), items.shape[0],
                                    _dev(buf, torch.float64), _stream(stream)))

    @property
    def interior_shape(self):
        n = self.block_dims
        return (self.nvars, self.nblocks, n[2], n[1], n[0])

    def fx_hydro_advance_host_interior(self, Uint_host, dx_host, cfl, nsteps, U_stage, packed_stage, dx_stage, stream=None):
        """Uint_host: CPU (preferably pinned) float64 tensor of interior zones [5][nblocks][nz][ny][nx], updated in place;
        U_stage: device padded state; packed_stage: device tensor of Uint_host's size.  Returns the last dt."""
        assert not Uint_host.is_cuda and Uint_host.dtype == torch.float64 and Uint_host.is_contiguous()
        assert tuple(Uint_host.shape) == self.interior_shape and packed_stage.numel() == Uint_host.numel()
        assert not dx_host.is_cuda and dx_host.dtype == torch.float64 and dx_host.is_contiguous()
        dt_last = C.c_double(float("nan"))
        _check(lib().fx_hydro_advance_host_interior(self._h, C.c_void_p(Uint_host.data_ptr()), C.c_void_p(dx_host.data_ptr()),
                                                    float(cfl), int(nsteps), _dev(U_stage, torch.float64),
                                                    _dev(packed_stage, torch.float64), _dev(dx_stage, torch.float64),
                                                    C.cast(C.byref(dt_last), C.c_void_p), _stream(stream)))
        return float(dt_last.value)

    def fx_hydro_advance_host(self, U_host, dx_host, cfl, nsteps, U_stage, dx_stage, stream=None):
        """U_host / dx_host: CPU (preferably pinned) float64 tensors, updated in place.  Returns the last dt."""
        assert not U_host.is_cuda and U_host.dtype == torch.float64 and U_host.is_contiguous()
        assert not dx_host.is_cuda and dx_host.dtype == torch.float64 and dx_host.is_contiguous()
        dt_last = C.c_double(float("nan"))
        _check(lib().fx_hydro_advance_host(self._h, C.c_void_p(U_host.data_ptr()), C.c_void_p(dx_host.data_ptr()),
                                           float(cfl), int(nsteps), _dev(U_stage, torch.float64),
                                           _dev(dx_stage, torch.float64), C.cast(C.byref(dt_last), C.c_void_p),
                                           _stream(stream)))
        return float(dt_last.value)

    def fx_hydro_status(self, stream=None):
        f = C.c_uint32()
        cnt = (C.c_ulonglong * 4)()
        _check(lib().fx_hydro_status(self._h, C.byref(f), cnt, _stream(stream)))
        return int(f.value), [int(x) for x in cnt]

    def fx_hydro_status_reset(self, stream=None):
        _check(lib().fx_hydro_status_reset(self._h, _stream(stream)))

    def fx_hydro_plan_set_timing(self, enable=True):
        _check(lib().fx_hydro_plan_set_timing(self._h, int(bool(enable))))

    def fx_hydro_plan_get_timing(self):
        """(sum of stage-kernel milliseconds, number of launches) since the last read."""
        ms, n = C.c_double(), C.c_longlong()
        _check(lib().fx_hydro_plan_get_timing(self._h, C.byref(ms), C.byref(n)))
        return float(ms.value), int(n.value)

    def flux_shape(self, direction):
        e = list(self.block_dims)
        e[direction] += 1
        return (self.nvars, self.nblocks, e[2], e[1], e[0])

    def fx_debug_compute_fluxes(self, U, direction, stream=None):
        F = torch.empty(self.flux_shape(direction), dtype=torch.float64, device=self.device)
        _check(lib().fx_debug_compute_fluxes(self._h, _dev(U, torch.float64), direction, _dev(F, torch.float64),
                                             _stream(stream)))
        return F

    def interior(self, U):
        g, n = self.gd, self.block_dims
        return U[:, :, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]]
