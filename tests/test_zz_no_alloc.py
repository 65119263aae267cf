"""dd4dvar_forecast_static: the forecast entry point for callers that cannot allocate device memory.

Who needs it: a user whose process has no device allocator left to call when the forecast is wanted.  The
device may belong to another framework's memory pool that gives nothing to plug-ins, it may simply be full (a
fail-over path must still produce the background trajectory), or the caller sits in a latency-bound loop and may
not stall the device with cudaMalloc / cudaFree.  Every other entry point of the library works out of a workspace
the caller allocates; this one works out of a 16 MiB array compiled into the library, so it needs no handle and no
workspace, at the price of a grid-size limit (about 349 000 cells) and of calls that must not overlap on one GPU.

The tests compare it with the handle-based dd4dvar_forecast (same step code, workspace memory) on two calls in a
row that leave different contents behind in the shared array, on a grid small enough to keep every level in the
array and on one where the levels wrap around inside it, and check that a grid beyond the limit is refused with a
message instead of being run.  (This file sorts last on purpose: `pytest -x` stops at the first failure, and a failure
here should not hide the parity tests.)"""
import ctypes as C

import numpy as np
import pytest

from paper_2205_06649_b200 import synth

from helpers import small_workload

TOL = 1e-12         # the tolerance of the trajectory comparisons in test_gpu_parity.py


def _x0(w, seed):
    """A model state with some structure: the workload's analytic truth plus seeded noise of 1 % of each field's RMS."""
    x = synth.truth_initial(w)
    return x + 0.01 * synth.field_rms(x)[:, None, None] * synth.random_fields(x.shape, seed)


def _max_rel(a, b):
    return float(np.max(np.abs(a - b)) / np.max(np.abs(b)))


def test_static_forecast_refuses_grids_beyond_its_scratch_without_touching_the_device():
    """The size check comes before any CUDA call: it can be exercised here without a GPU (pointers never dereferenced)."""
    from paper_2205_06649_b200 import binding
    lib = binding.load_library()
    g = binding.Grid(1440, 720, 6.371e6, 7.292e-5, 9.806, 0.64, 0.02)
    w = binding.Window(75.0, 4)
    lv = (C.c_int * 1)(4)
    err = C.create_string_buffer(512)
    rc = lib.dd4dvar_forecast_static(C.byref(g), C.byref(w), C.c_void_p(0x1000), 1, lv, C.c_void_p(0x2000), None, err, len(err))
    assert rc == -6
    text = err.value.decode()
    assert "1440 x 720" in text and str(binding.STATIC_SCRATCH_BYTES) in text
    # bad arguments are told apart from "too large"
    assert lib.dd4dvar_forecast_static(C.byref(g), C.byref(w), None, 1, lv, C.c_void_p(0x2000), None, err, len(err)) == -1
    lv[0] = 5
    assert lib.dd4dvar_forecast_static(C.byref(g), C.byref(w), C.c_void_p(0x1000), 1, lv, C.c_void_p(0x2000), None, None, 0) == -1


@pytest.mark.gpu
@pytest.mark.parametrize("shape", ["all_levels_resident", "levels_wrap_inside_the_array"])
def test_static_forecast_matches_the_workspace_forecast_on_two_calls_in_a_row(shape):
    import torch
    from paper_2205_06649_b200.binding import DD4DVar, forecast_static, STATIC_SCRATCH_BYTES
    if shape == "all_levels_resident":
        w = small_workload(nlon=36, nlat=18, dt=600.0, nsteps=16)
        levels = [0, 1, 7, 7, 16]
    else:
        # 360 x 180: one level is 1.56 MB, the array holds 10 of them, the window has 25
        w = small_workload(nlon=360, nlat=180, dt=300.0, nsteps=24, nbumps=10, cfg=1)
        levels = [0, 3, 9, 10, 19, 24]
        assert (STATIC_SCRATCH_BYTES // 8) // (3 * 360 * 180) < w.nsteps + 1
    dev = torch.device("cuda:0")
    g = DD4DVar.from_workload(w, device="cuda:0")          # the existing path: handle + caller-allocated workspace
    try:
        out = torch.empty((len(levels), 3, w.nlat, w.nlon), dtype=torch.float64, device=dev)
        # two calls in a row with different inputs: the second runs on top of what the first left in the array
        for seed in (11, 12):
            x0 = _x0(w, seed)
            want = g.forecast(x0, levels)
            out.fill_(float("nan"))
            got = forecast_static(torch.as_tensor(x0, device=dev), levels, out, w.dt, w.nsteps).cpu().numpy()
            assert np.isfinite(got).all()
            assert _max_rel(got, want) <= TOL, (shape, seed, _max_rel(got, want))
            assert np.array_equal(got[0], x0)               # level 0 is the input itself
        # and once more with the first input: same answer as before, whatever the array held in between
        x0 = _x0(w, 11)
        again = forecast_static(torch.as_tensor(x0, device=dev), levels, out, w.dt, w.nsteps).cpu().numpy()
        assert _max_rel(again, g.forecast(x0, levels)) <= TOL
    finally:
        g.close()


@pytest.mark.gpu
def test_static_forecast_refuses_the_quarter_degree_grid_on_the_device():
    import torch
    from paper_2205_06649_b200.binding import DD4DVarError, forecast_static
    dev = torch.device("cuda:0")
    x0 = torch.zeros((3, 720, 1440), dtype=torch.float64, device=dev)
    out = torch.full((1, 3, 720, 1440), 7.0, dtype=torch.float64, device=dev)
    with pytest.raises(DD4DVarError) as ei:
        forecast_static(x0, [2], out, 75.0, 4)
    assert ei.value.code == -6 and "1440 x 720" in str(ei.value)
    assert float(out.min()) == 7.0 and float(out.max()) == 7.0      # nothing was launched
