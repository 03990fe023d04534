"""-m gpu parity at BASELINE.json's FULL sizes, in the launch configuration bench.py times (WAVE kernels, launch-free
sweep, tuned tile width, the config's full step count).

The whole field is compared bit for bit with the classic GPU path (north_star: "swept and naive GPU paths must also agree
bit-exactly"), and SAMPLED outputs are compared with the CPU oracle: the value at point i after n timesteps depends only
on the initial values within h*S*n points of i (one stencil radius per sub-timestep), so the oracle, run on a periodic
window of M >= 2*h*S*n + 2*V points cut out of the initial field, reproduces the V points on either side of the
window's centre exactly -- outputs "the oracle can compute one by one" at a cost of M*n instead of nx*n updates.  One
window straddles the periodic seam (index 0), one a tile boundary in the middle of the domain.
"""
import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import TOL, assert_bits_equal, rel_max, run_oracle, solver_for, to_dev

pytestmark = pytest.mark.gpu


def _oracle_window(w, dtype, u0, nsteps, centre, M):
    """Oracle on the periodic window of M points centred at `centre`; returns (global indices, values) of the points whose
    domain of dependence lies inside the window."""
    H, S = wl.RADIUS[w.problem], wl.STAGES[w.problem]
    reach = H * S * nsteps
    V = M // 2 - reach
    assert V >= 64, (M, reach)
    idx = (centre - M // 2 + np.arange(M)) % w.nx
    ref = run_oracle(w, dtype, nsteps, u0=np.ascontiguousarray(u0[:, idx]))
    keep = np.arange(M // 2 - V, M // 2 + V)
    return idx[keep], ref[:, keep]


CASES = [
    # problem, dtype, nx, kind, window M   (nsteps = the config's count)
    pytest.param(wl.HEAT, np.float64, 1 << 22, "noise", 1 << 17, id="heat-f64-2^22-50000-noise"),
    pytest.param(wl.HEAT, np.float32, 1 << 22, "config", 1 << 17, id="heat-f32-2^22-50000-config2"),
    pytest.param(wl.KS, np.float64, 1 << 20, "config", 1 << 18, id="ks-f64-2^20-20000-config3"),
    pytest.param(wl.EULER, np.float64, 1 << 20, "config", 1 << 17, id="euler-f64-2^20-10000-config4"),
]
FULL_STEPS = {wl.HEAT: 50_000, wl.KS: 20_000, wl.EULER: 10_000}


@pytest.mark.parametrize("problem,dtype,nx,kind,M", CASES)
def test_full_size_bench_configuration(problem, dtype, nx, kind, M):
    import torch
    w = wl.make(problem, nx, kind)
    nsteps = FULL_STEPS[problem]
    u0 = w.initial(dtype)
    with solver_for(w, dtype) as s:
        W = s.tune(to_dev(u0))                       # what bench.py does: tuned width, chain on (the default)
        assert s.tile_width_ok(W)
        us, un = to_dev(u0), to_dev(u0)
        s.swept_run(us, nsteps, 0)                   # 0 = the tuned width, on the kernel the tuner measured as fastest for it
        info = s.info()
        ran = "smem" if info["tuned_kernel"] == sw.KERNEL_SMEM else sw.LAUNCH_NAMES[info["last_sweep_launch"]]
        print(f"full-size parity covers: {wl.PROBLEM_NAMES[problem]} {np.dtype(dtype).name} nx=2^{nx.bit_length() - 1} W={W} kernel={ran} "
              f"launches={info['launches_last_call']}")
        # the tuner chooses among the launch-free kernels on these sizes; ring and band carry the remainder inside their ONE launch
        assert info["last_sweep_launch"] in (sw.LAUNCH_RING, sw.LAUNCH_BAND, sw.LAUNCH_CHAIN), info
        if info["last_sweep_launch"] in (sw.LAUNCH_RING, sw.LAUNCH_BAND):
            assert info["launches_last_call"] == 1
        s.naive_run(un, nsteps)
        torch.cuda.synchronize()
        got, naive = us.cpu().numpy(), un.cpu().numpy()
    assert np.all(np.isfinite(naive))
    assert not np.array_equal(naive, u0), "the run must change the field"
    assert_bits_equal(got, naive, f"swept({ran}, W={W}) vs classic at full size")
    # sampled outputs against the oracle: the periodic seam and a tile boundary in mid-domain
    for centre in (0, nx // 2 + W // 2):
        idx, ref = _oracle_window(w, dtype, u0, nsteps, centre, M)
        assert np.all(np.isfinite(ref))
        sample = got.reshape(u0.shape)[:, idx]
        assert rel_max(sample, ref) <= TOL[dtype]
        assert_bits_equal(sample, ref, f"swept vs oracle window at {centre}")


def test_full_size_config5_prefix_and_width_sweep():
    """Config 5 (stress): nx = 2^22 on the 16-mode series; every WAVE width agrees bitwise with the classic path on a
    1 000-step prefix, and the oracle agrees on a window (oracle on a prefix)."""
    import torch
    for problem, dtype in ((wl.HEAT, np.float32), (wl.KS, np.float64), (wl.EULER, np.float32)):
        w = wl.make(problem, 1 << 22, "config5")
        u0 = w.initial(dtype)
        nsteps = 1000
        with solver_for(w, dtype) as s:
            un = to_dev(u0)
            s.naive_run(un, nsteps)
            torch.cuda.synchronize()
            naive = un.cpu().numpy()
            for W in (64, 128, 256, 512, 1024):
                if not s.tile_width_ok(W):
                    continue
                us = to_dev(u0)
                s.swept_run(us, nsteps, W)
                torch.cuda.synchronize()
                assert_bits_equal(us.cpu().numpy(), naive, f"config5 {wl.PROBLEM_NAMES[problem]} W={W}")
        idx, ref = _oracle_window(w, dtype, u0, nsteps, 0, 1 << 14)
        assert_bits_equal(naive.reshape(u0.shape)[:, idx], ref, "config5 oracle window")


CONFIG5 = [(wl.HEAT, np.float64), (wl.HEAT, np.float32), (wl.KS, np.float64), (wl.KS, np.float32), (wl.EULER, np.float64), (wl.EULER, np.float32)]


@pytest.mark.parametrize("problem,dtype", CONFIG5, ids=[f"{wl.PROBLEM_NAMES[p]}-{'f64' if d == np.float64 else 'f32'}" for p, d in CONFIG5])
def test_full_size_config5_full_length(problem, dtype):
    """Config 5 at its FULL length: nx = 2^22, 100 000 timesteps on the 16-mode series, all six
    (problem, dtype) pairs, in the configuration the stress bench times (tuned width, default launch-free option):
    swept == classic bit for bit over the whole field; the oracle on the window of a 1 000-step prefix."""
    import torch
    nx, nsteps, prefix = 1 << 22, 100_000, 1000
    w = wl.make(problem, nx, "config5")
    assert w.nsteps == nsteps
    u0 = w.initial(dtype)
    with solver_for(w, dtype) as s:
        W = s.tune(to_dev(u0))
        s.set_option(sw.OPT_NAIVE_GRAPH, 1)              # same kernels, same order; only the launch mechanism differs
        us, un, up = to_dev(u0), to_dev(u0), to_dev(u0)
        s.swept_run(us, nsteps, 0)
        ran = s.info()["last_sweep_launch"]
        s.naive_run(un, nsteps)
        s.swept_run(up, prefix, 0)
        torch.cuda.synchronize()
        got, naive, pre = us.cpu().numpy(), un.cpu().numpy(), up.cpu().numpy()
    assert ran in (sw.LAUNCH_RING, sw.LAUNCH_BAND, sw.LAUNCH_CHAIN)
    assert np.all(np.isfinite(naive)) and not np.array_equal(naive, u0)
    assert_bits_equal(got, naive, f"config5 full length swept({sw.LAUNCH_NAMES[ran]}, W={W}) vs classic")
    for centre in (0, nx // 2 + W // 2):
        idx, ref = _oracle_window(w, dtype, u0, prefix, centre, 1 << 14)
        sample = pre.reshape(u0.shape)[:, idx]
        assert rel_max(sample, ref) <= TOL[dtype]
        assert_bits_equal(sample, ref, f"config5 prefix vs oracle window at {centre}")
