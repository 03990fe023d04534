"""`swept_run_static`: the swept rule for callers that cannot allocate device memory.

Some programs cannot let a library call cudaMalloc: the GPU's memory is wholly in the hands of their own pool (a framework's
caching allocator, a solver's arena, a fixed budget per tenant), or they call from a loop in which the device-wide stall of an
allocation is not acceptable.  For them the library has one entry point without a handle, whose odd-tier edge row is a fixed
array inside the library image (SWEPT_STATIC_SCRATCH_BYTES) instead of the workspace a handle allocates.

What is checked here, on a GPU: the entry point gives the same bits as the handle path (`Solver.swept_run` on the same
kernels, and the classic path) -- bit-exact, the tolerance every swept-vs-classic test of this suite uses -- on TWO calls in a
row that share the array (the second must not be disturbed by what the first left behind), that device memory in use does
not grow across a call, and, without a GPU, that a field beyond the array's size is refused with a clear message.

This file sorts last on purpose: `pytest -x` stops at the first failure, so a failure here hides no other test.
"""
import ctypes

import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl


def _handle_path(w, dtype, nsteps, W):
    """The existing path on the same kernels: a Solver with the register-resident tile kernels, one launch per half-cycle."""
    import torch
    with sw.Solver(w.problem, w.nx, w.dx, w.dt, dtype=sw.F64 if dtype == np.float64 else sw.F32, alpha=w.alpha, gamma=w.gamma) as s:
        s.set_option(sw.OPT_KERNEL, sw.KERNEL_WAVE)
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_OFF)
        u = torch.from_numpy(w.initial(dtype)).cuda()
        s.swept_run(u, nsteps, W)
        c = torch.from_numpy(w.initial(dtype)).cuda()
        s.naive_run(c, nsteps)
        torch.cuda.synchronize()
        return u.cpu().numpy(), c.cpu().numpy()


def _static_path(w, dtype, nsteps, W):
    import torch
    u = torch.from_numpy(w.initial(dtype)).cuda()
    sw.swept_run_static(w.problem, u, nsteps, w.dx, w.dt, tile_width=W, alpha=w.alpha, gamma=w.gamma)
    torch.cuda.synchronize()
    return u.cpu().numpy()


# (workload, dtype, tile width, timesteps): three half-cycles plus a remainder that needs narrower tiles and classic steps;
# consecutive cases differ in problem, size and dtype, so each call finds the previous one's edges in the shared array
CASES = [
    (lambda: wl.heat_noise(1 << 16), np.float64, 256, 3 * 128 + 37),
    (lambda: wl.euler_noise(1 << 12), np.float32, 128, 3 * 16 + 5),
    (lambda: wl.ks_noise(1 << 14), np.float64, 256, 2 * 32 + 9),
    (lambda: wl.heat_noise(1 << 12), np.float32, 0, 200),          # tile_width 0: the default width
]


@pytest.mark.gpu
def test_static_scratch_entry_point_equals_the_handle_path_on_consecutive_calls():
    import torch
    for make, dtype, W, nsteps in CASES:
        w = make()
        want_swept, want_classic = _handle_path(w, dtype, nsteps, W if W else 256)
        # two calls in a row on the same input, sharing the static array
        first = _static_path(w, dtype, nsteps, W)
        second = _static_path(w, dtype, nsteps, W)
        assert np.array_equal(first, want_swept), (w.name, "first call differs from Solver.swept_run")
        assert np.array_equal(second, want_swept), (w.name, "second call differs from Solver.swept_run")
        assert np.array_equal(first, want_classic), (w.name, "differs from the classic path")
        assert np.isfinite(first).all()
    # back-to-back on one stream without a host synchronisation in between: stream order is all the ordering the array needs
    w = wl.heat_noise(1 << 16)
    a = torch.from_numpy(w.initial(np.float64)).cuda()
    b = torch.from_numpy(w.initial(np.float64)).cuda()
    sw.swept_run_static(w.problem, a, 300, w.dx, w.dt, tile_width=128)
    sw.swept_run_static(w.problem, b, 300, w.dx, w.dt, tile_width=512)
    torch.cuda.synchronize()
    assert torch.equal(a, b)            # the result does not depend on the tile width
    assert np.array_equal(a.cpu().numpy(), _handle_path(w, np.float64, 300, 128)[1])


@pytest.mark.gpu
def test_static_scratch_entry_point_leaves_device_memory_alone():
    """After the one-off set-up, a call must not change the amount of device memory in use (it makes no allocation)."""
    import torch
    w = wl.heat_noise(1 << 18)
    u = torch.from_numpy(w.initial(np.float64)).cuda()
    sw.swept_run_static(w.problem, u, 64, w.dx, w.dt)          # set-up for (device, heat, f64) happens here at the latest
    torch.cuda.synchronize()
    free0, _ = torch.cuda.mem_get_info()
    sw.swept_run_static(w.problem, u, 1000, w.dx, w.dt)
    torch.cuda.synchronize()
    free1, _ = torch.cuda.mem_get_info()
    assert free1 >= free0, f"device memory in use grew by {free0 - free1} bytes across swept_run_static"


def test_static_scratch_entry_point_refuses_fields_beyond_the_array():
    """No GPU needed: the size check comes before the first CUDA call."""
    L = sw.lib()
    for problem, dtype, nx_ok, in ((sw.HEAT, sw.F64, 1 << 20), (sw.HEAT, sw.F32, 1 << 21), (sw.EULER, sw.F64, 1 << 18), (sw.EULER, sw.F32, 1 << 19)):
        p = sw._Params(dtype, 1.0, 1.4, 0, sw.BC_PERIODIC)
        rc = L.swept_run_static(problem, 2 * nx_ok, 1.0 / nx_ok, 1e-9, ctypes.byref(p), ctypes.c_void_p(256), 1, 0, None)
        assert rc == sw.EINVAL
        msg = L.swept_last_error().decode()
        assert "SWEPT_STATIC_SCRATCH_BYTES" in msg and str(sw.STATIC_SCRATCH_BYTES) in msg, msg
    # other argument errors, also without a device
    p = sw._Params(sw.F64, 1.0, 1.4, 0, sw.BC_INSULATED)
    assert L.swept_run_static(sw.HEAT, 1024, 1e-3, 1e-7, ctypes.byref(p), ctypes.c_void_p(256), 1, 0, None) == sw.EINVAL
    assert b"periodic" in L.swept_last_error()
    assert L.swept_run_static(sw.HEAT, 1000, 1e-3, 1e-7, None, ctypes.c_void_p(256), 1, 0, None) == sw.EINVAL
    assert L.swept_run_static(sw.HEAT, 1024, 1e-3, 1e-7, None, None, 1, 0, None) == sw.EINVAL
    assert L.swept_run_static(sw.HEAT, 1024, 1e-3, 1e-7, None, ctypes.c_void_p(256), -1, 0, None) == sw.EINVAL
    assert L.swept_run_static(sw.HEAT, 1024, 1e-3, 1e-7, None, ctypes.c_void_p(256), 1, 48, None) == sw.EINVAL
    assert b"tile_width" in L.swept_last_error()
