"""-m gpu parity of the 2-D swept rule (include/swept2d.h): classic 2-D kernel == CPU oracle and swept == classic, bit for bit."""
import numpy as np
import pytest

import oracle
import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import TOL, assert_bits_equal, rel_max, to_dev

pytestmark = pytest.mark.gpu


KERNELS = {"warp": sw.KERNEL2D_WARP, "smem": sw.KERNEL2D_SMEM, "column": sw.KERNEL2D_COLUMN}     # W = 32 only; narrower tiles always run on the shared-memory kernels


def _run(nx, ny, dtype, nsteps, W=None, fo=0.2, u0=None, kernel="warp"):
    import torch
    dx, dt = wl.heat2d_grid(max(nx, ny), fo)
    u0 = wl.heat2d_field(nx, ny).astype(dtype) if u0 is None else u0
    with sw.Solver2D(nx, ny, dx, dt, dtype=sw.F64 if dtype == np.float64 else sw.F32) as s:
        u = to_dev(u0)
        s.set_option(sw.OPT2D_KERNEL, KERNELS[kernel])
        if W is None:
            s.naive_run(u, nsteps)
        else:
            s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        return u.cpu().numpy(), s.info()


@pytest.mark.parametrize("dtype", [np.float64, np.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("nx,ny,nsteps", [(8, 8, 3), (64, 32, 37), (256, 512, 20)])
def test_classic_2d_matches_oracle(nx, ny, nsteps, dtype):
    got, _ = _run(nx, ny, dtype, nsteps)
    dx, dt = wl.heat2d_grid(max(nx, ny), 0.2)
    ref = oracle.heat2d(wl.heat2d_field(nx, ny).astype(dtype), nsteps, 1.0, dx, dt)
    assert rel_max(got[None], ref[None]) <= TOL[dtype]
    assert_bits_equal(got, ref, f"classic 2-D vs oracle {nx}x{ny}")


@pytest.mark.parametrize("dtype", [np.float64, np.float32], ids=["f64", "f32"])
@pytest.mark.parametrize("nx,ny,W,nsteps", [
    (8, 8, 8, 4),            # one tile wrapping onto itself in both directions, one half-cycle
    (16, 8, 8, 4 * 3 + 1),   # three half-cycles (closes on the shifted alignment) + a remainder step
    (64, 128, 16, 8 * 4),    # even half-cycle count
    (128, 64, 32, 16 * 2 + 7),
    (512, 512, 32, 16 * 5 + 3),
    (256, 1024, 16, 8 * 7),
    (32, 32, 32, 16 * 3),    # one 32 x 32 tile wrapping onto itself: every halo of the register kernel is the tile's own far side
    (64, 32, 32, 16),        # one half-cycle: pyramid, bridges, inverted pyramid
    (32, 128, 32, 16 * 4 + 1),
])
@pytest.mark.parametrize("kernel", ["warp", "column", "smem"])
def test_swept_2d_equals_classic_and_oracle(nx, ny, W, nsteps, dtype, kernel):
    if kernel != "warp" and W != 32:
        pytest.skip("W < 32 has one kernel family")
    got, info = _run(nx, ny, dtype, nsteps, W=W, kernel=kernel)
    ref, _ = _run(nx, ny, dtype, nsteps)
    L = W // 2
    assert info["launches_last_call"] == nsteps % L + 1 + 2 * (nsteps // L)       # remainder + pyramids + (bridges, octahedra) per half-cycle
    assert_bits_equal(got, ref, f"swept 2-D vs classic {nx}x{ny} W={W}")
    dx, dt = wl.heat2d_grid(max(nx, ny), 0.2)
    orc = oracle.heat2d(wl.heat2d_field(nx, ny).astype(dtype), nsteps, 1.0, dx, dt)
    assert rel_max(got[None], orc[None]) <= TOL[dtype]
    assert_bits_equal(got, orc, "swept 2-D vs oracle")


def test_swept_2d_full_size_sampled_against_the_oracle():
    """nx = ny = 4096 (128 MiB of fp64: HBM-resident), 400 timesteps: whole field == classic; the oracle on a periodic window whose
    centre block lies outside the reach of the window's seam."""
    n, nsteps, M = 4096, 400, 1024
    rng = np.random.default_rng(3)
    u0 = rng.uniform(-1, 1, (n, n))
    got, _ = _run(n, n, np.float64, nsteps, W=32, u0=u0)
    ref, _ = _run(n, n, np.float64, nsteps, u0=u0)
    assert_bits_equal(got, ref, "swept 2-D (register kernel) vs classic at 4096^2")
    for kern in ("column", "smem"):
        other, _ = _run(n, n, np.float64, nsteps, W=32, u0=u0, kernel=kern)
        assert_bits_equal(other, ref, f"swept 2-D ({kern} kernel) vs classic at 4096^2")
    dx, dt = wl.heat2d_grid(n, 0.2)
    for cy, cx in ((0, 0), (n // 2 + 16, n // 2 + 16)):
        iy, ix = (cy - M // 2 + np.arange(M)) % n, (cx - M // 2 + np.arange(M)) % n
        win = oracle.heat2d(np.ascontiguousarray(u0[np.ix_(iy, ix)]), nsteps, 1.0, dx, dt)
        V = M // 2 - nsteps - 8
        keep = np.arange(M // 2 - V, M // 2 + V)
        assert_bits_equal(got[np.ix_(iy[keep], ix[keep])], win[np.ix_(keep, keep)], f"oracle window at ({cy}, {cx})")


def test_illegal_arguments_2d():
    with pytest.raises(sw.SweptError):
        sw.Solver2D(100, 64, 0.01, 1e-5)
    dx, dt = wl.heat2d_grid(64)
    with sw.Solver2D(64, 64, dx, dt) as s:
        u = to_dev(wl.heat2d_field(64, 64))
        for bad in (4, 12, 64, -8):
            with pytest.raises(sw.SweptError):
                s.swept_run(u, 10, bad)
        with pytest.raises(sw.SweptError):
            s.naive_run(u.float(), 1)
        with pytest.raises(sw.SweptError):
            s.set_option(sw.OPT2D_KERNEL, 7)


def test_skinny_2d_grid_at_the_row_limit():
    """ny = 2^18 is the tallest grid the header allows (ny / 8 rows of blocks on blockIdx.y): every path launches and agrees;
    one row more is refused at creation instead of failing at launch."""
    nx, ny = 8, 1 << 18
    u0 = wl.heat2d_field(nx, ny)
    want, _ = _run(nx, ny, np.float64, 5, None, u0=u0)
    assert np.isfinite(want).all()
    got, _ = _run(nx, ny, np.float64, 5, 8, u0=u0)                # one classic remainder step, then one half-cycle of W = 8 (4 timesteps)
    assert_bits_equal(got, want, "swept W = 8 on 8 x 2^18")
    with pytest.raises(sw.SweptError):
        sw.Solver2D(8, 1 << 19, 1.0, 0.1)


def test_run_host_2d_equals_the_device_path():
    nx, ny, nsteps = 256, 128, 37
    u0 = wl.heat2d_field(nx, ny)
    want, _ = _run(nx, ny, np.float64, nsteps, 32, u0=u0)
    dx, dt = wl.heat2d_grid(max(nx, ny), 0.2)
    with sw.Solver2D(nx, ny, dx, dt) as s:
        h = u0.copy()
        s.run_host(h, nsteps, 32)
        assert_bits_equal(h, want, "swept2d_run_host, swept")
        h = u0.copy()
        s.run_host(h, nsteps, use_swept=False)
        assert_bits_equal(h, want, "swept2d_run_host, classic")
        with pytest.raises(sw.SweptError):
            s.run_host(u0[:64].copy(), nsteps)


def test_the_two_2d_kernels_agree():
    """The register kernel and the shared-memory kernel run the same regions in the same tier order with the same store rule:
    identical fields after 1, 2 and 3 half-cycles (odd and even closing alignment)."""
    import torch
    nx = ny = 128
    dx, dt = wl.heat2d_grid(nx, 0.2)
    u0 = wl.heat2d_field(nx, ny)
    for K in (1, 2, 3):
        outs = []
        for kern in ("warp", "column", "smem"):
            with sw.Solver2D(nx, ny, dx, dt) as s:
                s.set_option(sw.OPT2D_KERNEL, KERNELS[kern])
                u = to_dev(u0)
                s.swept_run(u, 16 * K, 32)
                torch.cuda.synchronize()
                outs.append(u.cpu().numpy())
        assert_bits_equal(outs[0], outs[1], f"folded vs column register kernels, {K} half-cycles")
        assert_bits_equal(outs[0], outs[2], f"register vs shared-memory 2-D kernels, {K} half-cycles")


def test_random_2d_configurations_match_the_classic_path_bitwise():
    """Seeded random (nx, ny, tile width, kernel, step count, dtype): swept == classic bit for bit."""
    import torch
    rng = np.random.default_rng(2495)
    ran = 0
    for _ in range(60):
        nx, ny = (1 << int(rng.integers(3, 10))), (1 << int(rng.integers(3, 10)))
        W = int(rng.choice([8, 16, 32]))
        kern = str(rng.choice(["warp", "column", "smem"]))
        dtype = np.float64 if rng.random() < 0.5 else np.float32
        nsteps = int(rng.integers(1, 5 * W))
        if W > min(nx, ny):
            continue
        u0 = rng.uniform(-1, 1, (ny, nx)).astype(dtype)
        got, _ = _run(nx, ny, dtype, nsteps, W=W, u0=u0, kernel=kern)
        ref, _ = _run(nx, ny, dtype, nsteps, u0=u0)
        assert_bits_equal(got, ref, f"2-D {nx}x{ny} W={W} {kern} {np.dtype(dtype).name} nsteps={nsteps}")
        ran += 1
    assert ran >= 30
