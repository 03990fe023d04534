"""-m gpu parity of the 1-D heat kernels at Fourier numbers that are NOT a power of two.

Every other heat test of the suite runs the configs' Fo = alpha dt / dx^2 = 1/4 (BASELINE.json; reading S2), for which
both products of `fma(Fo, l + r, c0 * u)` are exact in binary: fused or not, in any order, the bits come out the same, so "the
CUDA path rounds exactly as the oracle does" is not exercised.  The C ABI takes any alpha, dx, dt; here Fo = 0.3 and 0.1237 with
alpha = 1 and 0.7 go through the classic kernel, every swept kernel family, the packed f32x2 band pairs and the insulated-ends
tiles, each asserted bit for bit against the CPU oracle (which is stronger than north_star's 1e-12 / 1e-5).
"""
import numpy as np
import pytest

import oracle
import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import (BAND, VARIANTS, VARIANT_IDS, TOL, assert_bits_equal, rel_max, run_naive, run_oracle, run_swept, solver_for, to_dev,
                      width_ok)

pytestmark = pytest.mark.gpu

FOURIER = [(0.3, 1.0), (0.1237, 0.7)]            # (Fo, alpha): neither Fo nor 1 - 2 Fo is a dyadic rational
FIDS = ["Fo0.3", "Fo0.1237-alpha0.7"]
DTYPES = [np.float64, np.float32]


@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("r,alpha", FOURIER, ids=FIDS)
@pytest.mark.parametrize("nx,nsteps", [(64, 37), (4096, 101)])
def test_classic_heat_kernel_equals_the_oracle_at_non_dyadic_fourier_numbers(r, alpha, dtype, nx, nsteps):
    w = wl.heat_noise(nx, r=r, alpha=alpha)
    got, ref = run_naive(w, dtype, nsteps), run_oracle(w, dtype, nsteps)
    assert rel_max(got, ref) <= TOL[dtype]
    assert_bits_equal(got, ref, f"classic vs oracle, Fo = {r}, alpha = {alpha}")
    # the case is not vacuous: an unfused evaluation of the same formula differs somewhere
    u = w.initial(dtype)
    fo, c0 = dtype(alpha * w.dt / (w.dx * w.dx)), dtype(1.0 - 2.0 * alpha * w.dt / (w.dx * w.dx))
    unfused = (fo * (np.roll(u, 1, axis=1) + np.roll(u, -1, axis=1)) + c0 * u).astype(dtype)
    one = run_oracle(w, dtype, 1)
    assert np.max(np.abs(unfused.astype(np.float64) - one.astype(np.float64))) <= 4 * np.finfo(dtype).eps * np.max(np.abs(one))
    if nx >= 4096:
        assert not np.array_equal(unfused, one), "Fo is exactly representable here: the case would not test rounding"


@pytest.mark.parametrize("kernel", VARIANTS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("r,alpha", FOURIER, ids=FIDS)
def test_every_swept_family_equals_the_oracle_at_non_dyadic_fourier_numbers(r, alpha, dtype, kernel):
    nx, W = 1 << 13, 256
    w = wl.heat_noise(nx, r=r, alpha=alpha)
    assert width_ok(w, dtype, W, kernel)
    nsteps = 3 * wl.steps_per_half_cycle(wl.HEAT, W) + 41          # three half-cycles + a remainder
    got = run_swept(w, dtype, nsteps, W, kernel)
    assert_bits_equal(got, run_oracle(w, dtype, nsteps), f"swept vs oracle, Fo = {r}, alpha = {alpha}")


@pytest.mark.parametrize("r,alpha", FOURIER, ids=FIDS)
@pytest.mark.parametrize("nx,W,q", [(1 << 12, 128, 3), (1 << 17, 128, 5)])
def test_packed_band_pairs_equal_the_oracle_at_non_dyadic_fourier_numbers(r, alpha, nx, W, q):
    """fma.rn.f32x2 rounds each component as a scalar fma does."""
    import torch
    w = wl.heat_noise(nx, r=r, alpha=alpha)
    nsteps = q * wl.steps_per_half_cycle(wl.HEAT, W) + 7
    with solver_for(w, np.float32) as s:
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
        s.set_option(sw.OPT_PACK, sw.PACK_ON)
        u = to_dev(w.initial(np.float32))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        assert s.info()["last_sweep_launch"] == sw.LAUNCH_BAND
        got = u.cpu().numpy()
    assert_bits_equal(got, run_oracle(w, np.float32, nsteps), f"packed pairs vs oracle, Fo = {r}")


@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("r,alpha", FOURIER, ids=FIDS)
def test_insulated_rod_equals_the_oracle_at_non_dyadic_fourier_numbers(r, alpha, dtype):
    import torch
    w = wl.heat_rod(1 << 12, r=r, alpha=alpha)
    nsteps = 3 * 64 + 29
    ref = oracle.run(w.problem, w.initial(dtype), nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, insulated=True)
    with solver_for(w, dtype, boundary=sw.BC_INSULATED) as s:
        us, un = to_dev(w.initial(dtype)), to_dev(w.initial(dtype))
        s.swept_run(us, nsteps, 128)
        s.naive_run(un, nsteps)
        torch.cuda.synchronize()
        assert_bits_equal(un.cpu().numpy(), ref, f"rod, classic vs oracle, Fo = {r}")
        assert_bits_equal(us.cpu().numpy(), ref, f"rod, swept (mirror tiles) vs oracle, Fo = {r}")


def test_static_entry_point_at_a_non_dyadic_fourier_number():
    import torch
    w = wl.heat_noise(1 << 13, r=0.3, alpha=0.7)
    u = to_dev(w.initial(np.float64))
    sw.swept_run_static(w.problem, u, 200, w.dx, w.dt, tile_width=256, alpha=w.alpha)
    torch.cuda.synchronize()
    assert_bits_equal(u.cpu().numpy(), run_oracle(w, np.float64, 200), "swept_run_static vs oracle")
