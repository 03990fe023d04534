"""-m gpu parity of the paper's own heat problem: a rod with insulated ends (Eq. 9; SURVEY.md
section 8(f) NEXT-2).  Classic and swept CUDA paths through the C ABI against the insulated-ends oracle, bit for bit."""
import numpy as np
import pytest

import oracle
import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import TOL, assert_bits_equal, rel_max, solver_for, to_dev

pytestmark = pytest.mark.gpu


def _rod(nx, seed=1612):
    return wl.heat_rod(nx, seed)       # temperature gradient + grid-scale noise: every step changes every value, the ends differ


def _run(w, dtype, nsteps, W=None, chain=None, opts=None):
    import torch
    with solver_for(w, dtype, boundary=sw.BC_INSULATED) as s:
        u = to_dev(w.initial(dtype))
        if W is None:
            s.naive_run(u, nsteps)
        else:
            if chain is not None:
                s.set_option(sw.OPT_CHAIN, chain)
            for k, v in (opts or {}).items():
                s.set_option(k, v)
            s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        return u.cpu().numpy(), s.info()


@pytest.mark.parametrize("dtype", [np.float64, np.float32])
@pytest.mark.parametrize("nx,nsteps", [(8, 3), (1024, 777), (1 << 14, 3000)])
def test_classic_path_equals_the_insulated_oracle(dtype, nx, nsteps):
    w = _rod(nx)
    got, info = _run(w, dtype, nsteps)
    assert info["boundary"] == sw.BC_INSULATED
    ref = oracle.run(w.problem, w.initial(dtype), nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, insulated=True)
    assert rel_max(got, ref) <= TOL[dtype]
    assert_bits_equal(got, ref, "classic insulated vs oracle")
    per = oracle.run(w.problem, w.initial(dtype), nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha)
    assert not np.array_equal(per, ref)                        # the test data tells the two boundary conditions apart


CASES = [
    # nx, W, nsteps                         what it exercises
    (64, 64, 32 * 3),                       # one tile: both boundary tiles of a shifted phase mirror the same tile
    (128, 64, 32 * 4 + 5),                  # two tiles, even number of half-cycles, remainder on the classic kernel
    (1 << 12, 128, 64 * 7 + 33),            # odd number of half-cycles: the closing phase is a shifted one with boundary tiles
    (1 << 12, 256, 128 * 6 + 77),           # remainder half-cycles on narrower tiles (upright + closing at W = 128, 64)
    (1 << 16, 1024, 512 * 5),
    (1 << 20, 256, 128 * 9 + 1),            # far more tiles than resident warps
]


@pytest.mark.parametrize("chain", [0, 1, 2], ids=["per-launch", "tile-flags", "default"])
@pytest.mark.parametrize("nx,W,nsteps", CASES)
def test_swept_paths_equal_the_classic_path_and_the_oracle(nx, W, nsteps, chain):
    w = _rod(nx)
    for dtype in (np.float64, np.float32):
        got, info = _run(w, dtype, nsteps, W, chain)
        if chain == 2 and nsteps >= W // 2:
            # the band schedule needs a periodic domain: the default falls back to the tile-flag kernel
            assert info["last_sweep_launch"] == sw.LAUNCH_CHAIN
        naive, _ = _run(w, dtype, nsteps)
        assert_bits_equal(got, naive, f"swept insulated nx={nx} W={W} chain={chain} vs classic")
        if nx <= (1 << 16):
            ref = oracle.run(w.problem, w.initial(dtype), nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, insulated=True)
            assert rel_max(got, ref) <= TOL[dtype]
            assert_bits_equal(got, ref, f"swept insulated nx={nx} W={W} chain={chain} vs oracle")


def test_launch_shapes_and_tuner_on_the_rod():
    w = _rod(1 << 15)
    nsteps = 64 * 11 + 3
    ref, _ = _run(w, np.float64, nsteps)
    for wpb, cap in ((1, 0), (2, 3), (8, 1)):
        got, _ = _run(w, np.float64, nsteps, 128, 1, opts={sw.OPT_WARPS_PER_BLOCK: wpb, sw.OPT_BLOCKS_PER_SM: cap})
        assert_bits_equal(got, ref, f"insulated wpb={wpb} cap={cap}")
    import torch
    with solver_for(w, np.float64, boundary=sw.BC_INSULATED) as s:
        W = s.tune(to_dev(w.initial(np.float64)))
        u = to_dev(w.initial(np.float64))
        s.swept_run(u, nsteps, 0)
        torch.cuda.synchronize()
        assert s.tile_width_ok(W)
        assert_bits_equal(u.cpu().numpy(), ref, "tuned width on the rod")


def test_insulated_ends_are_heat_only_and_need_the_wave_kernels():
    w = wl.ks_noise(1 << 12)
    with pytest.raises(sw.SweptError):
        solver_for(w, np.float64, boundary=sw.BC_INSULATED)
    with pytest.raises(sw.SweptError):
        solver_for(_rod(1 << 12), np.float64, boundary=7)
    with solver_for(_rod(1 << 12), np.float64, boundary=sw.BC_INSULATED) as s:
        s.set_option(sw.OPT_KERNEL, sw.KERNEL_SMEM)
        assert not s.tile_width_ok(128)
        s.set_option(sw.OPT_KERNEL, sw.KERNEL_WAVE)
        assert s.tile_width_ok(128)


def test_full_size_rod_in_the_bench_configuration():
    """nx = 2^22, the config's 50 000 timesteps, tuned width (what `bench.py --boundary insulated` times): swept = classic bit for
    bit, and the left end (where the mirror matters) against the oracle on a window that the far side cannot reach: values at
    x < M - nsteps of an M-point rod depend only on the first M points."""
    import torch
    nx, nsteps, M, V = 1 << 22, 50_000, 1 << 16, 4096
    w = _rod(nx)
    u0 = w.initial(np.float64)
    with solver_for(w, np.float64, boundary=sw.BC_INSULATED) as s:
        W = s.tune(to_dev(u0))
        us, un = to_dev(u0), to_dev(u0)
        s.swept_run(us, nsteps, 0)
        s.naive_run(un, nsteps)
        torch.cuda.synchronize()
        got, naive = us.cpu().numpy(), un.cpu().numpy()
    assert_bits_equal(got, naive, f"rod, full size, W={W}")
    ref = oracle.heat_insulated(u0[0, :M].copy(), nsteps, w.alpha, w.dx, w.dt)
    assert M - nsteps >= V
    assert_bits_equal(got[0, :V], ref[:V], "left end of the rod vs the insulated oracle")
    ref = oracle.heat_insulated(u0[0, nx - M:].copy(), nsteps, w.alpha, w.dx, w.dt)
    assert_bits_equal(got[0, nx - V:], ref[M - V:], "right end of the rod vs the insulated oracle")
