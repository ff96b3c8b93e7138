"""ctypes wrapper of the CPU oracle (oracle/fxoracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the
cpu_baseline / --impl reference legs of bench.py; never by the product package.
It imports nothing from paper_2208_11630_b200.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "fxoracle.c")
_LIB = os.path.join(_HERE, "libfxoracle.so")

RECON_PLM_MINMOD, RECON_WENO5 = 0, 1
RIEMANN_HLLE, RIEMANN_HLLC = 0, 1
BC_OUTFLOW, BC_NONE, BC_REFLECT = -1, -2, -3
NEIGH_COARSER, NEIGH_FINER = -4, -5
OPT_GRAVITY_X, OPT_GRAVITY_Y, OPT_GRAVITY_Z = 6, 7, 8
TOPO_PERIODIC, TOPO_OUTFLOW, TOPO_NONE, TOPO_REFLECT = 0, 1, 2, 3
ORDER_LEX, ORDER_MORTON = 0, 1
OPT_RHO_FLOOR, OPT_P_FLOOR, OPT_WENO_EPS, OPT_WAVESPEED = 0, 1, 2, 3
STATUS_NONFINITE, STATUS_RHO_FLOOR, STATUS_P_FLOOR, STATUS_WENO_FALLBACK = 1, 2, 4, 8


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (no FMA contraction, no fast-math)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(
            ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-std=c99", "-Wall", "-Wno-maybe-uninitialized", "-shared", "-fPIC",
             "-o", _LIB, _SRC, "-lm"])
    return _LIB


class _Layout(C.Structure):
    _fields_ = [("np", C.c_int32 * 3), ("gd", C.c_int32 * 3), ("S_j", C.c_int64), ("S_k", C.c_int64),
                ("S_b", C.c_int64), ("S_v", C.c_int64), ("bytes_per_state", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        dp, ip = C.POINTER(C.c_double), C.POINTER(C.c_int32)
        L.fxo_plan_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(C.c_int), C.c_int, C.c_int, C.c_int64,
                                      C.c_double, C.c_int, C.c_int, C.c_int]
        L.fxo_plan_destroy.argtypes = [C.c_void_p]
        L.fxo_plan_destroy.restype = None
        L.fxo_plan_layout.argtypes = [C.c_void_p, C.POINTER(_Layout)]
        L.fxo_plan_set_option.argtypes = [C.c_void_p, C.c_int, C.c_double]
        L.fxo_plan_set_topology.argtypes = [C.c_void_p, ip]
        L.fxo_plan_set_refinement.argtypes = [C.c_void_p, ip]
        L.fxo_status.argtypes = [C.c_void_p, C.POINTER(C.c_uint32), C.POINTER(C.c_ulonglong)]
        L.fxo_status_reset.argtypes = [C.c_void_p]
        L.fxo_status_reset.restype = None
        L.fxo_topology_cartesian.argtypes = [C.POINTER(C.c_int), C.POINTER(C.c_int), C.POINTER(C.c_int), C.c_int, ip, ip]
        L.fxo_guardcell_index_map.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.POINTER(C.c_int64)]
        L.fxo_fill_guardcells.argtypes = [C.c_void_p, dp]
        L.fxo_cons2prim.argtypes = [C.c_void_p, dp, dp]
        L.fxo_cons2prim.restype = None
        L.fxo_minmod.argtypes = [C.c_double, C.c_double]
        L.fxo_minmod.restype = C.c_double
        L.fxo_weno5.argtypes = [C.c_double] * 6
        L.fxo_weno5.restype = C.c_double
        L.fxo_face_states.argtypes = [C.c_void_p, dp, C.c_int64, C.c_int64, C.c_int64, dp, dp, C.POINTER(C.c_uint32)]
        L.fxo_face_states.restype = None
        L.fxo_riemann_flux.argtypes = [C.c_void_p, dp, dp, dp]
        L.fxo_riemann_flux.restype = None
        L.fxo_cons2prim_nv.argtypes = [C.c_void_p, dp, dp]
        L.fxo_cons2prim_nv.restype = None
        L.fxo_riemann_flux_nv.argtypes = [C.c_void_p, dp, dp, dp]
        L.fxo_riemann_flux_nv.restype = None
        L.fxo_euler_step.argtypes = [C.c_void_p, dp, dp, C.c_double]
        L.fxo_hydro_advance.argtypes = [C.c_void_p, dp, dp, C.c_double]
        L.fxo_hydro_advance_ca.argtypes = [C.c_void_p, dp, dp, C.c_double]
        L.fxo_debug_compute_fluxes.argtypes = [C.c_void_p, dp, C.c_int, dp]
        L.fxo_hydro_compute_dt.argtypes = [C.c_void_p, dp, dp, C.c_double, dp]
        _lib = L
    return _lib


def _dptr(a: np.ndarray):
    assert a.dtype == np.float64 and a.flags["C_CONTIGUOUS"]
    return a.ctypes.data_as(C.POINTER(C.c_double))


def _check(rc: int, what: str):
    if rc != 0:
        raise RuntimeError(f"oracle {what} failed with code {rc}")


def minmod(a: float, b: float) -> float:
    return lib().fxo_minmod(a, b)


def weno5(a, b, c, d, e, eps=1e-6) -> float:
    return lib().fxo_weno5(a, b, c, d, e, eps)


def topology_cartesian(nb, bc_lo, bc_hi, order=ORDER_LEX):
    """neigh [nblocks,6] int32 and block coordinates [nblocks,3] int32 of a regular tiling."""
    n = int(nb[0]) * int(nb[1]) * int(nb[2])
    neigh = np.empty((n, 6), np.int32)
    coords = np.empty((n, 3), np.int32)
    i3 = C.c_int * 3
    _check(lib().fxo_topology_cartesian(i3(*nb), i3(*bc_lo), i3(*bc_hi), order,
                                        neigh.ctypes.data_as(C.POINTER(C.c_int32)),
                                        coords.ctypes.data_as(C.POINTER(C.c_int32))), "topology_cartesian")
    return neigh, coords


class OraclePlan:
    def __init__(self, dims, nguard, nblocks, gamma, recon, riemann, rk_order, nvars=5):
        self._h = C.c_void_p()
        rc = lib().fxo_plan_create(C.byref(self._h), (C.c_int * 3)(*dims), nguard, nvars, nblocks, gamma, recon,
                                   riemann, rk_order)
        if rc != 0:
            self._h = C.c_void_p()
            raise ValueError(f"fxo_plan_create failed with code {rc}")
        L = _Layout()
        _check(lib().fxo_plan_layout(self._h, C.byref(L)), "plan_layout")
        self.dims = tuple(int(d) for d in dims)
        self.nblocks = int(nblocks)
        self.nvars = nvars
        self.gamma = gamma
        self.np = tuple(L.np)
        self.gd = tuple(L.gd)
        self.S_j, self.S_k, self.S_b, self.S_v = L.S_j, L.S_k, L.S_b, L.S_v
        self.bytes_per_state = L.bytes_per_state
        self._neigh = None

    def __del__(self):
        try:
            if getattr(self, "_h", None) and self._h.value:
                lib().fxo_plan_destroy(self._h)
                self._h = C.c_void_p()
        except Exception:  # interpreter shutdown
            pass

    @property
    def shape(self):
        """Shape of a state array U[v][b][k][j][i]."""
        return (self.nvars, self.nblocks, self.np[2], self.np[1], self.np[0])

    def set_option(self, key, value):
        rc = lib().fxo_plan_set_option(self._h, key, float(value))
        if rc != 0:
            raise ValueError(f"fxo_plan_set_option failed with code {rc}")

    def set_refinement(self, jump):
        """Refinement-jump table int32 [nblocks, 6, 4] [B12]; before set_topology."""
        jump = np.ascontiguousarray(jump, np.int32).reshape(self.nblocks, 6, 4)
        rc = lib().fxo_plan_set_refinement(self._h, jump.ctypes.data_as(C.POINTER(C.c_int32)))
        if rc != 0:
            raise ValueError(f"fxo_plan_set_refinement failed with code {rc}")
        self._jump = jump  # keep alive: the plan borrows it

    def set_topology(self, neigh):
        neigh = np.ascontiguousarray(neigh, np.int32).reshape(self.nblocks, 6)
        rc = lib().fxo_plan_set_topology(self._h, neigh.ctypes.data_as(C.POINTER(C.c_int32)))
        if rc != 0:
            raise ValueError(f"fxo_plan_set_topology failed with code {rc}")
        self._neigh = neigh  # keep alive: the plan borrows it

    def status(self):
        f = C.c_uint32()
        cnt = (C.c_ulonglong * 4)()
        _check(lib().fxo_status(self._h, C.byref(f), cnt), "status")
        return int(f.value), [int(x) for x in cnt]

    def status_reset(self):
        lib().fxo_status_reset(self._h)

    def index_map(self, block_begin=0, block_count=None):
        if block_count is None:
            block_count = self.nblocks - block_begin
        src = np.empty((block_count, self.np[2], self.np[1], self.np[0]), np.int64)
        _check(lib().fxo_guardcell_index_map(self._h, block_begin, block_count,
                                             src.ctypes.data_as(C.POINTER(C.c_int64))), "index_map")
        return src

    def fill_guardcells(self, U):
        _check(lib().fxo_fill_guardcells(self._h, _dptr(U)), "fill_guardcells")

    def cons2prim(self, U5):
        U5 = np.ascontiguousarray(U5, np.float64)
        W = np.empty(5)
        lib().fxo_cons2prim(self._h, _dptr(U5), _dptr(W))
        return W

    def cons2prim_nv(self, U):
        """All nvars entries (hydro variables + passive scalars, reading B11)."""
        U = np.ascontiguousarray(U, np.float64)
        assert U.shape == (self.nvars,)
        W = np.empty(self.nvars)
        lib().fxo_cons2prim_nv(self._h, _dptr(U), _dptr(W))
        return W

    def face_states(self, W, cL):
        """Face states [O3, A6] between cells cL and cL + 1 of a line of primitives W[nvars][ncells]; returns
        (WL, WR, status bits raised)."""
        W = np.ascontiguousarray(W, np.float64)
        assert W.ndim == 2 and W.shape[0] == self.nvars
        WL, WR = np.empty(self.nvars), np.empty(self.nvars)
        hit = C.c_uint32()
        lib().fxo_face_states(self._h, _dptr(W), W.shape[1], int(cL), 1, _dptr(WL), _dptr(WR), C.byref(hit))
        return WL, WR, int(hit.value)

    def riemann_flux_nv(self, WL, WR):
        """Face-frame states (rho, un, ut1, ut2, p, X_1..) of nvars entries -> flux of nvars entries (B11)."""
        WL = np.ascontiguousarray(WL, np.float64)
        WR = np.ascontiguousarray(WR, np.float64)
        assert WL.shape == (self.nvars,) and WR.shape == (self.nvars,)
        F = np.empty(self.nvars)
        lib().fxo_riemann_flux_nv(self._h, _dptr(WL), _dptr(WR), _dptr(F))
        return F

    def riemann_flux(self, WL, WR):
        WL = np.ascontiguousarray(WL, np.float64)
        WR = np.ascontiguousarray(WR, np.float64)
        F = np.empty(5)
        lib().fxo_riemann_flux(self._h, _dptr(WL), _dptr(WR), _dptr(F))
        return F

    def euler_step(self, U, dx, dt):
        dx = np.ascontiguousarray(dx, np.float64)
        _check(lib().fxo_euler_step(self._h, _dptr(U), _dptr(dx), float(dt)), "euler_step")

    def advance(self, U, dx, dt):
        dx = np.ascontiguousarray(dx, np.float64)
        rc = lib().fxo_hydro_advance(self._h, _dptr(U), _dptr(dx), float(dt))
        if rc != 0:
            raise ValueError(f"fxo_hydro_advance failed with code {rc}")

    def advance_ca(self, U, dx, dt):
        """The communication-avoiding step [B17]: one guard fill, stages on a shrinking extension of the interior."""
        dx = np.ascontiguousarray(dx, np.float64)
        rc = lib().fxo_hydro_advance_ca(self._h, _dptr(U), _dptr(dx), float(dt))
        if rc != 0:
            raise ValueError(f"fxo_hydro_advance_ca failed with code {rc}")

    def compute_dt(self, U, dx, cfl):
        dx = np.ascontiguousarray(dx, np.float64)
        out = C.c_double()
        _check(lib().fxo_hydro_compute_dt(self._h, _dptr(U), _dptr(dx), float(cfl), C.byref(out)), "compute_dt")
        return float(out.value)

    def flux_shape(self, direction):
        e = [self.dims[0], self.dims[1], self.dims[2]]
        e[direction] += 1
        return (self.nvars, self.nblocks, e[2], e[1], e[0])

    def debug_compute_fluxes(self, U, direction):
        F = np.empty(self.flux_shape(direction))
        _check(lib().fxo_debug_compute_fluxes(self._h, _dptr(U), direction, _dptr(F)), "debug_compute_fluxes")
        return F

    def interior(self, U):
        g = self.gd
        n = self.dims
        return U[:, :, g[2]:g[2] + n[2], g[1]:g[1] + n[1], g[0]:g[0] + n[0]]
