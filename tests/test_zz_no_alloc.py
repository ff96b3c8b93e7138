"""fx_hydro_compute_dt_static: the CFL reduction with its scratch in the library's static device array (for callers that may
not allocate: no workspace, no cudaMalloc inside the call).  Checked against fx_hydro_compute_dt, the existing path with its
reduction words in the caller's workspace, on two calls in a row; plus the size limit, the status bits and that the header is
cleared between calls.  Collected last on purpose (file name): the suite runs with pytest -x."""
import numpy as np
import pytest
import torch

from paper_2208_11630_b200 import inputs
from tests.helpers import gpu_plan_for

pytestmark = pytest.mark.gpu

DT_TOL = 1e-14  # the relative tolerance the dt comparisons of the other GPU tests use


def _bare_plan(fx, cfg, nblocks=None):
    """A plan with neither topology nor workspace: all the static entry point needs."""
    return fx.HydroPlan(cfg.block_dims, cfg.nguard, cfg.nblocks if nblocks is None else nblocks, cfg.gamma, cfg.recon,
                        cfg.riemann, cfg.rk_order)


@pytest.mark.parametrize("number,nb", [(5, (3, 3, 3)), (4, (2, 2, 2)), (2, (4, 4, 1))])
def test_static_dt_equals_workspace_dt_on_two_calls_in_a_row(number, nb):
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(number, nb=nb)
    plan, neigh, coords = gpu_plan_for(cfg)            # existing path: topology + workspace
    bare = _bare_plan(fx, cfg)                          # the new entry point's plan
    U = plan.embed(inputs.block_interiors(cfg, coords))
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dt_s = torch.full((1,), float("nan"), dtype=torch.float64, device="cuda")
    flags = torch.full((1,), -1, dtype=torch.int32, device="cuda")
    seen = []
    for call in range(2):                               # second call: a different state, the array holds the first call's partials
        want = float(plan.fx_hydro_compute_dt(U, dx, cfg.cfl).item())
        bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s, flags)
        got = float(dt_s.item())
        assert np.isfinite(want) and want > 0
        assert abs(got - want) <= DT_TOL * want, (call, got, want)
        assert int(flags.item()) == 0
        seen.append(got)
        plan.fx_hydro_advance(U, dx, want)              # move the state on
        flags.fill_(-1)
        dt_s.fill_(float("nan"))
    assert seen[0] != seen[1]                           # the two calls did see different states
    # and the same state twice in a row gives the same bits
    bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s)
    a = float(dt_s.item())
    bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s)
    assert float(dt_s.item()) == a
    assert abs(a - float(plan.fx_hydro_compute_dt(U, dx, cfg.cfl).item())) <= DT_TOL * a


def test_static_dt_allocates_no_device_memory():
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 2))
    plan, neigh, coords = gpu_plan_for(cfg)
    bare = _bare_plan(fx, cfg)
    U = plan.embed(inputs.block_interiors(cfg, coords))
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dt_s = torch.empty(1, dtype=torch.float64, device="cuda")
    bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s)   # set-up (address look-up) happens here at the latest
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 == free0


def test_static_dt_status_bits_and_header_clearing():
    """A NaN zone raises FX_STATUS_NONFINITE in flags_out; the next call on clean data reports 0 (the header does not keep
    the last call's bits) and the right dt."""
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 2))
    plan, neigh, coords = gpu_plan_for(cfg)
    bare = _bare_plan(fx, cfg)
    U = plan.embed(inputs.block_interiors(cfg, coords))
    dx = torch.from_numpy(inputs.dx_array(cfg)).cuda()
    dt_s = torch.empty(1, dtype=torch.float64, device="cuda")
    flags = torch.zeros(1, dtype=torch.int32, device="cuda")
    Ubad = U.clone()
    plan.interior(Ubad)[4, 3, 5, 6, 7] = float("nan")
    bare.fx_hydro_compute_dt_static(Ubad, dx, cfg.cfl, dt_s, flags)
    assert int(flags.item()) & fx.STATUS_NONFINITE
    bare.fx_hydro_compute_dt_static(U, dx, cfg.cfl, dt_s, flags)
    assert int(flags.item()) == 0
    want = float(plan.fx_hydro_compute_dt(U, dx, cfg.cfl).item())
    assert abs(float(dt_s.item()) - want) <= DT_TOL * want


def test_static_dt_size_limit_empty_batch_and_null_arguments():
    from paper_2208_11630_b200 import binding as fx
    cfg = inputs.config(5, nb=(2, 2, 2))
    dt_s = torch.full((1,), 1.0, dtype=torch.float64, device="cuda")
    dummy = torch.zeros(8, dtype=torch.float64, device="cuda")
    # one block more than the array has room for: refused with a message, nothing launched (the dummies are never read)
    big = _bare_plan(fx, cfg, nblocks=fx.STATIC_DT_MAX_BLOCKS + 1)
    with pytest.raises(fx.FxError, match="exceed the static scratch"):
        big.fx_hydro_compute_dt_static(dummy, dummy, cfg.cfl, dt_s)
    torch.cuda.synchronize()
    assert float(dt_s.item()) == 1.0
    # an empty batch: +inf, as fx_hydro_compute_dt
    empty = _bare_plan(fx, cfg, nblocks=0)
    empty.fx_hydro_compute_dt_static(dummy, dummy, cfg.cfl, dt_s)
    assert float(dt_s.item()) == float("inf")
    # null output
    import ctypes as C
    rc = fx.lib().fx_hydro_compute_dt_static(big._h, C.c_void_p(dummy.data_ptr()), C.c_void_p(dummy.data_ptr()), 0.3, None, None, None)
    assert rc == fx.ERR_INVALID_ARG
