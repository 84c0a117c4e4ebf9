"""rt_cfl_dt_uniform_noalloc (include/rt.h): the entry point that allocates nothing, against the existing path
(rt_cfl_dt_async through a grid handle) on the same seeded states, two calls in a row.  Collected last on purpose (the
suite runs with pytest -x).  Tolerance: 1e-14 relative, the one test_cfl_dt_matches_oracle uses for this quantity."""
import numpy as np
import pytest
import torch

import rt_workloads as W

pytestmark = pytest.mark.gpu

TOL_DT = 1e-14


@pytest.fixture(scope="module")
def rt():
    assert torch.cuda.is_available(), "the -m gpu tests need a CUDA device"
    from paper_2606_26268_b200 import rt as _rt
    _rt.lib()
    return _rt


def _uniform_grid(rt, n, box):
    xf = [np.linspace(0.0, box[d], n[d] + 1) for d in range(3)]
    g = rt.Grid(rt.CARTESIAN, n, xf[0], xf[1], xf[2], (rt.BC_PERIODIC,) * 6)
    dx = [box[d] / n[d] for d in range(3)]
    return g, dx


@pytest.mark.parametrize("n,box", [((141, 37, 35), (1.0, 0.7, 2.0)), ((64, 48, 1), (1.0, 1.0, 1.0)), ((300, 1, 1), (3.0, 1.0, 1.0)),
                                   ((32, 256, 256), (1.0, 1.0, 1.0))])
def test_noalloc_cfl_matches_handle_path_twice(rt, n, box):
    g, dx = _uniform_grid(rt, n, box)
    chat = 3.0
    g.set_params(rt.make_params(chat=chat))
    rng = np.random.default_rng(260626268 + n[0])
    dt_ref = torch.zeros(1, dtype=torch.float64, device="cuda")
    dt_new = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    # two calls in a row on different states and cfl numbers: the second must not see anything of the first in the
    # shared static scratch (the second state is much dimmer in f, so its rate maximum is SMALLER than what the first
    # call left in the row slots)
    for call, (fmax, cfl) in enumerate(((1.0, 0.4), (0.05, 0.8))):
        U = [g.to_device(a) for a in W.random_state(rng, n, fmax=fmax)]
        g.cfl_dt_async(U, cfl, dt_ref)
        rt.cfl_dt_uniform_noalloc(n, dx, chat, cfl, U, dt_new)
        torch.cuda.synchronize()
        ref, got = dt_ref.item(), dt_new.item()
        assert ref > 0.0 and np.isfinite(ref)
        assert abs(got - ref) <= TOL_DT * ref, (call, got, ref)


def test_noalloc_cfl_rejects_what_does_not_fit(rt):
    n = (8, 257, 256)   # 65 792 rows > RT_NOALLOC_MAX_ROWS
    assert n[1] * n[2] > rt.NOALLOC_MAX_ROWS
    U = [torch.ones((n[2] + 4, n[1] + 4, n[0] + 4), dtype=torch.float64, device="cuda") for _ in range(4)]
    dt = torch.full((1,), -1.0, dtype=torch.float64, device="cuda")
    with pytest.raises(rt.RtError) as ei:
        rt.cfl_dt_uniform_noalloc(n, (1.0, 1.0, 1.0), 1.0, 0.4, U, dt)
    assert ei.value.status == rt.ERR_INVALID_ARG and "RT_NOALLOC_MAX_ROWS" in str(ei.value)
    for bad_dx in ((0.0, 1.0, 1.0), (1.0, float("nan"), 1.0)):
        with pytest.raises(rt.RtError):
            rt.cfl_dt_uniform_noalloc((8, 8, 8), bad_dx, 1.0, 0.4, [u[:12, :12, :12].contiguous() for u in U], dt)
    torch.cuda.synchronize()
    assert dt.item() == -1.0, "a rejected call must not enqueue work"
