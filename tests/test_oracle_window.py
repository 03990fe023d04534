"""-m "not gpu": the finite domain of dependence the full-size GPU tests rely on (tests/test_gpu_fullsize.py).  The oracle
run on a periodic WINDOW cut out of the field reproduces the full-field oracle bit for bit at every point whose cone of
dependence (h*S points per timestep, "domain of dependence") lies inside the window -- and not beyond."""
import numpy as np
import pytest

import oracle
import workloads as wl


@pytest.mark.parametrize("problem", [wl.HEAT, wl.KS, wl.EULER], ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("dtype", [np.float64, np.float32], ids=["f64", "f32"])
def test_window_reproduces_the_full_field_inside_the_cone(problem, dtype):
    nx, nsteps, M, centre = 4096, 60, 1024, 5
    w = wl.make(problem, nx, "noise")
    u0 = w.initial(dtype)
    full = oracle.run(problem, u0, nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, gamma=w.gamma)
    idx = (centre - M // 2 + np.arange(M)) % nx
    win = oracle.run(problem, np.ascontiguousarray(u0[:, idx]), nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, gamma=w.gamma)
    reach = wl.RADIUS[problem] * wl.STAGES[problem] * nsteps
    V = M // 2 - reach
    keep = np.arange(M // 2 - V, M // 2 + V)
    assert np.array_equal(win[:, keep], full[:, idx[keep]])
    # the bound is sharp: the window's outermost points have seen the artificial wrap
    assert not np.array_equal(win[:, :8], full[:, idx[:8]])
