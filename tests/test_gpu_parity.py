"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, element by element, and the swept
kernels against the classic kernel bit for bit (include/swept1d.h guarantee; north_star).

Tolerance (north_star): relative max-norm <= 1e-12 (fp64) / 1e-5 (fp32) against the oracle.  Oracle and CUDA path
evaluate the same canonical operation order with explicit fma and no contraction, so the
tests additionally assert the stronger statement that holds by construction: identical bits.
"""
import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import SMEM as SMEM_V, BAND as BAND_V
from gpu_util import (VARIANTS, VARIANT_IDS, TOL, assert_bits_equal, rel_max, run_naive, run_oracle, run_swept, solver_for, to_dev, width_ok)

pytestmark = pytest.mark.gpu

PROBLEMS = [wl.HEAT, wl.KS, wl.EULER]
DTYPES = [np.float64, np.float32]
KERNELS = VARIANTS            # (kernel family, chain): smem, wave (one launch per half-cycle), chain (launch-free sweep)
KNAME = dict(zip(VARIANTS, VARIANT_IDS))


def _noise(problem, nx):
    return wl.make(problem, nx, "noise")


# ------------------------------------------------------------------------------------------------------------
# classic (naive) path vs oracle
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("nx,nsteps", [(8, 3), (64, 37), (4096, 101), (1 << 16, 12)])
def test_naive_matches_oracle(problem, dtype, nx, nsteps):
    w = _noise(problem, nx)
    got = run_naive(w, dtype, nsteps)
    ref = run_oracle(w, dtype, nsteps)
    assert np.all(np.isfinite(ref))
    assert rel_max(got, ref) <= TOL[dtype]
    assert_bits_equal(got, ref, f"naive vs oracle {wl.PROBLEM_NAMES[problem]} nx={nx}")


@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
def test_naive_zero_steps_is_identity_and_graph_matches_plain(problem):
    w = _noise(problem, 1024)
    u0 = w.initial(np.float64)
    assert_bits_equal(run_naive(w, np.float64, 0), u0, "0 steps")
    assert_bits_equal(run_naive(w, np.float64, 57, graph=True), run_naive(w, np.float64, 57), "graph vs plain")


# ------------------------------------------------------------------------------------------------------------
# swept vs classic: bit-exact for every legal tile width, remainder, alignment, single-tile wrap
# ------------------------------------------------------------------------------------------------------------
def _sph(problem, W):
    return wl.steps_per_half_cycle(problem, W)


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("W", [8, 32, 64, 128, 256, 512, 1024, 2048])
def test_swept_matches_naive_bitwise(problem, dtype, W, kernel):
    nx = max(4 * W, 2048)
    w = _noise(problem, nx)
    if not width_ok(w, dtype, W, kernel):
        pytest.skip(f"W={W} not offered by the {KNAME[kernel]} kernel for this problem")
    sph = _sph(problem, W)
    # 3 half-cycles (odd: closes on the shifted alignment) plus a remainder that needs narrower tiles and a classic step
    nsteps = 3 * sph + (sph // 2 + 1 if sph > 1 else 0)
    got = run_swept(w, dtype, nsteps, W, kernel)
    ref = run_naive(w, dtype, nsteps)
    assert np.all(np.isfinite(ref))
    assert_bits_equal(got, ref, f"swept({KNAME[kernel]}) vs naive W={W}")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("q", [1, 2, 4, 5])
def test_swept_half_cycle_counts(problem, q, kernel):
    """Odd and even half-cycle counts both write out correctly (reading S4), q = 1 is up + down only."""
    W, nx = 64, 1024
    w = _noise(problem, nx)
    if not width_ok(w, np.float64, W, kernel):
        pytest.skip("width not offered")
    nsteps = q * _sph(problem, W)
    assert_bits_equal(run_swept(w, np.float64, nsteps, W, kernel), run_naive(w, np.float64, nsteps), f"q={q}")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
def test_swept_single_tile_wraps_onto_itself(problem, kernel):
    W = nx = 256
    w = _noise(problem, nx)
    if not width_ok(w, np.float64, W, kernel):
        pytest.skip("width not offered")
    nsteps = 3 * _sph(problem, W) + 1
    assert_bits_equal(run_swept(w, np.float64, nsteps, W, kernel), run_naive(w, np.float64, nsteps), "nx == W")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
def test_swept_translation_equivariance_bitwise(problem, kernel):
    """A circular shift by a non-multiple of W commutes with the swept run bit for bit (exposes tile-edge bugs)."""
    W, nx, shift = 128, 2048, 37
    w = _noise(problem, nx)
    if not width_ok(w, np.float64, W, kernel):
        pytest.skip("width not offered")
    nsteps = 2 * _sph(problem, W) + 3
    u0 = w.initial(np.float64)
    a = run_swept(w, np.float64, nsteps, W, kernel, u0=u0)
    b = run_swept(w, np.float64, nsteps, W, kernel, u0=np.ascontiguousarray(np.roll(u0, shift, axis=1)))
    assert_bits_equal(b.reshape(u0.shape), np.roll(a.reshape(u0.shape), shift, axis=1), "shift equivariance")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
def test_result_independent_of_tile_width(kernel):
    w = _noise(wl.KS, 4096)
    outs = []
    for W in (32, 64, 256, 1024):
        if width_ok(w, np.float64, W, kernel):
            outs.append(run_swept(w, np.float64, 300, W, kernel))
    if len(outs) < 2:
        pytest.skip("fewer than two widths offered")
    for o in outs[1:]:
        assert_bits_equal(o, outs[0], "tile-width independence")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
def test_swept_graph_replay_matches_plain(kernel):
    w = _noise(wl.HEAT, 4096)
    if not width_ok(w, np.float64, 128, kernel):
        pytest.skip("width not offered")
    a = run_swept(w, np.float64, 500, 128, kernel, graph=True)
    assert_bits_equal(a, run_naive(w, np.float64, 500), "graph replay")


# ------------------------------------------------------------------------------------------------------------
# swept vs oracle on the configs (BASELINE.json)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
def test_config1_heat_full_run_matches_oracle(kernel):
    """Config 1 exactly: heat fp64, nx=1024, r=0.25, 10 000 steps, W=64 (312 half-cycles + 16 remainder steps)."""
    w = wl.heat_config1()
    if not width_ok(w, np.float64, w.tile_width, kernel):
        pytest.skip("width not offered")
    got = run_swept(w, np.float64, w.nsteps, w.tile_width, kernel)
    ref = run_oracle(w, np.float64, w.nsteps)
    assert rel_max(got, ref) <= 1e-12
    assert_bits_equal(got, ref, "config 1")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("problem,nx,nsteps,W", [(wl.HEAT, 1 << 14, 3000, 256), (wl.KS, 1 << 14, 2000, 256), (wl.EULER, 1 << 12, 1500, 128)],
                         ids=["heat-c2", "ks-c3", "euler-c4"])
def test_config_workloads_match_oracle(problem, nx, nsteps, W, dtype, kernel):
    """Configs 2-4 initial data at their smallest nx on a prefix of the run the oracle finishes in seconds."""
    w = wl.make(problem, nx, "config")
    if not width_ok(w, dtype, W, kernel):
        pytest.skip("width not offered")
    got = run_swept(w, dtype, nsteps, W, kernel)
    ref = run_oracle(w, dtype, nsteps)
    assert np.all(np.isfinite(ref))
    assert rel_max(got, ref) <= TOL[dtype]
    assert_bits_equal(got, ref, "config workload")


# ------------------------------------------------------------------------------------------------------------
# boundary behaviour
# ------------------------------------------------------------------------------------------------------------
def test_illegal_arguments_are_rejected():
    import torch
    w = _noise(wl.KS, 1024)
    with solver_for(w, np.float64) as s:
        s.set_option(sw.OPT_KERNEL, sw.KERNEL_SMEM)
        u = to_dev(w.initial(np.float64))
        for bad in (3, 4, 48, 2048, -8):
            with pytest.raises(sw.SweptError) as ei:
                s.swept_run(u, 10, bad)
            assert ei.value.code == sw.EINVAL
        with pytest.raises(sw.SweptError):
            s.swept_run(u, -1, 64)
        with pytest.raises(sw.SweptError):
            s.naive_run(u.float(), 1)
        with pytest.raises(sw.SweptError):
            s.set_option(99, 0)
        torch.cuda.synchronize()
        assert_bits_equal(u.cpu().numpy(), w.initial(np.float64), "rejected calls must not touch the field")


def test_run_host_round_trip_and_info():
    import torch
    w = _noise(wl.EULER, 2048)
    with solver_for(w, np.float64) as s:
        s.set_option(sw.OPT_KERNEL, sw.KERNEL_SMEM)
        h = torch.from_numpy(w.initial(np.float64)).pin_memory()
        s.run_host(h, 40, 64, use_swept=True)
        info = s.info()
        assert info["ncomp"] == 3 and info["radius"] == 2 and info["stages"] == 2 and info["nx"] == 2048
        assert info["launches_last_call"] == 40 // 8 + 1
        assert_bits_equal(h.numpy(), run_naive(w, np.float64, 40), "run_host")


@pytest.mark.parametrize("kernel", KERNELS, ids=VARIANT_IDS)
def test_tuner_returns_a_legal_width_and_default_run_uses_it(kernel):
    import torch
    w = _noise(wl.HEAT, 1 << 14)
    with solver_for(w, np.float32, max_tile_width=512) as s:
        s.set_option(sw.OPT_KERNEL, kernel[0])
        s.set_option(sw.OPT_CHAIN, kernel[1])
        if not any(s.tile_width_ok(W) for W in (32, 64, 128, 256, 512)):
            pytest.skip("kernel offers no width")
        scratch = to_dev(w.initial(np.float32))
        best = s.tune(scratch)
        assert s.tile_width_ok(best) and best <= 512
        assert s.info()["tuned_tile_width"] == best
        u = to_dev(w.initial(np.float32))
        s.swept_run(u, 777, 0)
        torch.cuda.synchronize()
        assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float32, 777), "tuned width run")


@pytest.mark.parametrize("dtype", [np.float64, np.float32], ids=["f64", "f32"])
def test_classic_euler_with_shared_faces_is_bit_identical(dtype):
    """SWEPT_OPT_NAIVE_SHARE: the classic kernel evaluates the faces between a thread's cells once.  Same bits as the per-point
    kernel and the oracle -- plain launches, graph replay, and as the remainder steps of a swept run."""
    import torch
    w = _noise(wl.EULER, 1 << 12)
    nsteps = 137
    ref = run_naive(w, dtype, nsteps)
    assert_bits_equal(ref, run_oracle(w, dtype, nsteps), "per-point classic vs oracle")
    for graph in (0, 1):
        with solver_for(w, dtype) as s:
            s.set_option(sw.OPT_NAIVE_SHARE, 1)
            s.set_option(sw.OPT_NAIVE_GRAPH, graph)
            u = to_dev(w.initial(dtype))
            s.naive_run(u, nsteps)
            torch.cuda.synchronize()
            assert_bits_equal(u.cpu().numpy(), ref, f"shared-face classic (graph={graph}) vs per-point classic")
            u = to_dev(w.initial(dtype))
            s.set_option(sw.OPT_CHAIN, sw.CHAIN_TILES)
            s.swept_run(u, nsteps, 256)              # 137 = 4 x 32 + 9: the remainder's classic steps take the option too
            torch.cuda.synchronize()
            assert_bits_equal(u.cpu().numpy(), ref, "swept run with shared-face remainder steps")
    with solver_for(_noise(wl.HEAT, 1 << 10), np.float64) as s:
        s.set_option(sw.OPT_NAIVE_SHARE, 1)           # accepted and ignored
        with pytest.raises(sw.SweptError):
            s.set_option(sw.OPT_NAIVE_SHARE, 2)


def test_alu_peak_microbenchmark_is_plausible():
    p64 = sw.measure_alu_peak(sw.F64)["instr_per_s"]
    p32 = sw.measure_alu_peak(sw.F32)["instr_per_s"]
    assert 1e12 < p64 < 1e14 and 1e12 < p32 < 2e14


def test_smem_peak_and_latency_probes_are_plausible():
    """swept_measure_smem_peak / swept_measure_latencies (include/swept1d.h): the denominators and bounds DESIGN.md quotes."""
    bw = sw.measure_smem_peak()["bytes_per_s"]
    assert 5e12 < bw < 1e14
    lat = sw.measure_latencies()
    assert set(lat) == {"dfma", "dadd_dfma", "shfl64", "lockstep_tier_2shfl_dadd_dfma", "smem_tier_1barrier_256thr"}
    assert all(np.isfinite(v) and 1.0 < v < 2000.0 for v in lat.values()), lat
    assert lat["dfma"] < lat["dadd_dfma"] < lat["lockstep_tier_2shfl_dadd_dfma"], lat       # one op < two dependent ops < shuffle + two ops
    assert lat["shfl64"] < lat["lockstep_tier_2shfl_dadd_dfma"] < lat["smem_tier_1barrier_256thr"], lat


# ------------------------------------------------------------------------------------------------------------
# launch-free sweep (SWEPT_OPT_CHAIN): flag-ordered persistent kernel
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("nx,W,q", [(128, 128, 9), (256, 128, 12), (1 << 12, 128, 40), (1 << 20, 128, 5), (1 << 16, 512, 7)])
def test_chain_many_phases_few_and_many_tiles(problem, nx, W, q):
    """One tile wrapping onto itself, two tiles (each the other's both neighbours), fewer tiles than SMs, and far more
    tiles than resident warps (8192 tiles: items of several phases in flight at once): the chained launch equals the
    classic path bit for bit."""
    from gpu_util import CHAIN
    w = _noise(problem, nx)
    if not width_ok(w, np.float64, W, CHAIN):
        pytest.skip("width not offered")
    nsteps = q * _sph(problem, W)
    assert_bits_equal(run_swept(w, np.float64, nsteps, W, CHAIN), run_naive(w, np.float64, nsteps), f"chain nx={nx} W={W} q={q}")


@pytest.mark.parametrize("wpb", [1, 2, 4, 8])
@pytest.mark.parametrize("cap", [0, 1, 3])
def test_chain_launch_shapes(wpb, cap):
    from gpu_util import CHAIN
    w = _noise(wl.KS, 1 << 15)
    nsteps = 11 * _sph(wl.KS, 256) + 5
    got = run_swept(w, np.float32, nsteps, 256, CHAIN, opts={sw.OPT_WARPS_PER_BLOCK: wpb, sw.OPT_BLOCKS_PER_SM: cap})
    assert_bits_equal(got, run_naive(w, np.float32, nsteps), f"chain wpb={wpb} cap={cap}")


def test_chain_repeated_calls_reuse_the_flags_and_plan_matches_launch_count():
    import torch
    w = _noise(wl.HEAT, 1 << 13)
    with solver_for(w, np.float64) as s:
        u = to_dev(w.initial(np.float64))
        total = 0
        for nsteps in (64 * 3, 64 * 8 + 17, 5, 64):
            s.swept_run(u, nsteps, 128)
            total += nsteps
            kinds = [k for k, *_ in sw.plan(wl.HEAT, w.nx, nsteps, 128)]
            assert s.info()["launches_last_call"] == sum(
                c if k in (sw.LAUNCH_CLASSIC, sw.LAUNCH_DIAMOND) else 1 for k, _, _, c in sw.plan(wl.HEAT, w.nx, nsteps, 128)), kinds
        torch.cuda.synchronize()
        assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float64, total), "four chained calls back to back")


def test_chain_graph_replay_and_two_streams():
    """Two solvers on two streams run chained sweeps concurrently (each handle owns its flags)."""
    import torch
    w = _noise(wl.HEAT, 1 << 14)
    s1, s2 = solver_for(w, np.float64), solver_for(w, np.float64)
    s2.set_option(sw.OPT_SWEPT_GRAPH, 1)
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    u1, u2 = to_dev(w.initial(np.float64)), to_dev(w.initial(np.float64))
    torch.cuda.synchronize()
    for _ in range(3):
        s1.swept_run(u1, 1000, 256, stream=st1)
        s2.swept_run(u2, 1000, 256, stream=st2)
    torch.cuda.synchronize()
    ref = run_naive(w, np.float64, 3000)
    assert_bits_equal(u1.cpu().numpy(), ref, "stream 1")
    assert_bits_equal(u2.cpu().numpy(), ref, "stream 2 (graph replay)")
    s1.close(); s2.close()


# ------------------------------------------------------------------------------------------------------------
# streaming bands (SWEPT_OPT_CHAIN = 2, the default): columns resident across half-cycles, progress counters
# ------------------------------------------------------------------------------------------------------------
BAND_CASES = [
    # problem, dtype, nx, W, q                      what it exercises
    (wl.HEAT, np.float64, 512, 256, 9),             # two bands, each the other's neighbour on both sides
    (wl.HEAT, np.float64, 1 << 12, 128, 1),         # q = 1: upright triangle straight into the closing triangle
    (wl.HEAT, np.float64, 1 << 12, 128, 2),
    (wl.HEAT, np.float32, 1 << 16, 256, 40),        # one band per warp, many phases (SR = 2 iterations)
    (wl.HEAT, np.float64, 1 << 22, 1024, 5),        # 4096 bands: warps own 1 or 2 bands, parked columns in shared memory
    (wl.HEAT, np.float32, 1 << 22, 256, 5),         # 16384 bands: up to 6 bands per warp, rotating parked buffers
    (wl.HEAT, np.float64, 1 << 21, 128, 6),         # SR = 1 heat tiles, 16384 bands
    (wl.KS, np.float64, 1 << 14, 256, 11),
    (wl.KS, np.float32, 1 << 21, 256, 4),           # 8192 bands, several per warp
    (wl.KS, np.float64, 1 << 20, 1024, 3),
    (wl.EULER, np.float64, 1 << 13, 256, 7),
    (wl.EULER, np.float32, 1 << 20, 256, 3),        # 4096 bands on few resident warps
    (wl.EULER, np.float64, 1 << 18, 512, 2),
    (wl.HEAT, np.float32, 1 << 22, 512, 5),         # four super-rows per iteration, 8192 bands: 3 per warp, swaps in the steady loop
    (wl.HEAT, np.float64, 1 << 21, 512, 3),         # four super-rows per iteration, 2 bands per warp
    (wl.KS, np.float32, 1 << 22, 512, 3),           # two super-rows per iteration (KS), 8192 bands
    (wl.KS, np.float64, 1 << 20, 512, 7),           # two super-rows per iteration, one band per warp
    (wl.EULER, np.float64, 1 << 19, 256, 3),        # the 16-warp build of the Euler fp64 band kernel
]


@pytest.mark.parametrize("problem,dtype,nx,W,q", BAND_CASES)
def test_band_kernel_equals_classic(problem, dtype, nx, W, q):
    import torch
    from gpu_util import BAND
    w = _noise(problem, nx)
    nsteps = q * _sph(problem, W) + 3                      # + a remainder that runs before the band launch
    with solver_for(w, dtype) as s:
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
        assert s.tile_width_ok(W)
        u = to_dev(w.initial(dtype))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        assert s.info()["last_sweep_launch"] == sw.LAUNCH_BAND, "this case must run on swept_band_kernel, not fall back"
        got = u.cpu().numpy()
    assert_bits_equal(got, run_naive(w, dtype, nsteps), f"band nx={nx} W={W} q={q}")


def test_band_falls_back_to_tile_flags_where_the_schedule_does_not_fit():
    """One 32-iteration chunk per tile (heat W = 64) and a single band (nx = W) can run neither on the ring kernel nor as
    streaming bands: the same half-cycles run on swept_chain_kernel, with the same result."""
    import torch
    for nx, W in ((1 << 12, 64), (256, 256)):
        w = _noise(wl.HEAT, nx)
        with solver_for(w, np.float64) as s:
            u = to_dev(w.initial(np.float64))
            s.swept_run(u, 5 * _sph(wl.HEAT, W), W)
            torch.cuda.synchronize()
            assert s.info()["last_sweep_launch"] == sw.LAUNCH_CHAIN
            assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float64, 5 * _sph(wl.HEAT, W)), f"fallback nx={nx} W={W}")


def test_band_repeated_calls_two_streams_and_graph_replay():
    """Band launches are cooperative (every warp resident): two solvers on two streams, one replaying a CUDA graph."""
    import torch
    w = _noise(wl.HEAT, 1 << 20)
    s1, s2 = solver_for(w, np.float64), solver_for(w, np.float64)
    s1.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
    s2.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
    s2.set_option(sw.OPT_SWEPT_GRAPH, 1)
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    u1, u2 = to_dev(w.initial(np.float64)), to_dev(w.initial(np.float64))
    torch.cuda.synchronize()
    for _ in range(3):
        s1.swept_run(u1, 1100, 512, stream=st1)
        s2.swept_run(u2, 1100, 512, stream=st2)
    torch.cuda.synchronize()
    assert s1.info()["last_sweep_launch"] == sw.LAUNCH_BAND
    ref = run_naive(w, np.float64, 3300)
    assert_bits_equal(u1.cpu().numpy(), ref, "stream 1")
    assert_bits_equal(u2.cpu().numpy(), ref, "stream 2 (graph replay)")
    s1.close(); s2.close()


def test_tuner_chooses_between_bands_and_tile_flags():
    w = _noise(wl.EULER, 1 << 16)
    with solver_for(w, np.float64) as s:
        W = s.tune(to_dev(w.initial(np.float64)))
        info = s.info()
        assert info["tuned_tile_width"] == W
        nsteps = 7 * _sph(wl.EULER, W) + 1
        if info["tuned_kernel"] == sw.KERNEL_SMEM:      # small Euler grids: the paper-style kernels (a thread per cell) can win
            assert info["tuned_chain"] == 0
            variant = (sw.KERNEL_SMEM, sw.CHAIN_OFF)
        else:
            assert info["tuned_kernel"] == -1 and info["tuned_chain"] in (sw.CHAIN_TILES, sw.CHAIN_BANDS, sw.CHAIN_RING)
            variant = (sw.KERNEL_WAVE, info["tuned_chain"])
        assert_bits_equal(run_swept(w, np.float64, nsteps, W, variant), run_naive(w, np.float64, nsteps), "tuned variant")
        # the default run (tile_width 0, and the tuned width given explicitly) uses what the tuner chose
        import torch
        for tw in (0, W):
            u = to_dev(w.initial(np.float64))
            s.swept_run(u, nsteps, tw)
            torch.cuda.synchronize()
            assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float64, nsteps), f"default run after tune, tile_width={tw}")
            ran = s.info()["last_sweep_launch"]
            assert (ran == sw.LAUNCH_DIAMOND) == (info["tuned_kernel"] == sw.KERNEL_SMEM)


def test_tuner_picks_the_shared_memory_kernels_for_a_small_euler_grid():
    """nx = 2^12 Euler: 16 tiles of 256 cells give the register kernels 16 warps of 8 cells per lane; the paper-style kernels run a
    thread per cell.  The tuner measures both families under the default options and swept_run follows it."""
    import torch
    w = _noise(wl.EULER, 1 << 12)
    with solver_for(w, np.float64) as s:
        W = s.tune(to_dev(w.initial(np.float64)))
        info = s.info()
        assert info["tuned_kernel"] == sw.KERNEL_SMEM and info["tuned_chain"] == 0 and info["tuned_tile_width"] == W
        u = to_dev(w.initial(np.float64))
        s.swept_run(u, 301, 0)
        torch.cuda.synchronize()
        assert s.info()["last_sweep_launch"] == sw.LAUNCH_DIAMOND
        assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float64, 301), "tuned shared-memory run")
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)       # an explicit choice of kernel overrides the tuner's family
        s.swept_run(u, 64, 256)
        torch.cuda.synchronize()
        assert s.info()["last_sweep_launch"] != sw.LAUNCH_DIAMOND


# ------------------------------------------------------------------------------------------------------------
# one handle, several streams; grids narrower than the narrowest register tile
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("chain", [sw.CHAIN_RING, sw.CHAIN_BANDS, sw.CHAIN_TILES], ids=["ring", "band", "chain"])
def test_one_handle_from_two_streams_is_serialised_not_corrupted(chain):
    """include/swept1d.h: calls on one handle from different streams run one after the other (each call's stream waits for
    the handle's previous call), so the flags / counters the launch-free kernels share are never re-zeroed under a running
    kernel.  Two fields advance alternately on two streams through ONE handle; a CUDA graph replay joins in."""
    import torch
    w = _noise(wl.HEAT, 1 << 16)
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    with solver_for(w, np.float64) as s:
        s.set_option(sw.OPT_CHAIN, chain)
        u1, u2 = to_dev(w.initial(np.float64)), to_dev(w.initial(np.float64))
        torch.cuda.synchronize()
        for i in range(6):
            s.set_option(sw.OPT_SWEPT_GRAPH, i % 2)
            s.swept_run(u1, 700, 256, stream=st1)
            s.swept_run(u2, 700, 256, stream=st2)
        s.naive_run(u2, 5, stream=st1)
        s.naive_run(u1, 5, stream=st2)
        torch.cuda.synchronize()
        ref = run_naive(w, np.float64, 6 * 700 + 5)
        assert_bits_equal(u1.cpu().numpy(), ref, "field 1")
        assert_bits_equal(u2.cpu().numpy(), ref, "field 2")


@pytest.mark.parametrize("problem", PROBLEMS, ids=["heat", "ks", "euler"])
@pytest.mark.parametrize("nx", [8, 32])
def test_default_width_on_grids_narrower_than_a_register_tile(problem, nx):
    """swept_run(tile_width = 0) on a grid too small for the WAVE kernels falls back to the shared-memory kernels."""
    import torch
    w = _noise(problem, nx)
    with solver_for(w, np.float64) as s:
        u = to_dev(w.initial(np.float64))
        s.swept_run(u, 23, 0)
        torch.cuda.synchronize()
        assert_bits_equal(u.cpu().numpy(), run_naive(w, np.float64, 23), f"default width nx={nx}")


# ------------------------------------------------------------------------------------------------------------
# Euler: the batched reciprocal / square root (stencils.cuh fp<T>::rcp_fast / sqrt_fast) must equal IEEE division and
# square root for EVERY operand, also those that leave the fast path (subnormal / huge densities, tiny sound speeds)
# ------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("dtype", DTYPES, ids=["f64", "f32"])
@pytest.mark.parametrize("case", ["tiny-density", "huge-density", "tiny-sound-speed"])
def test_batched_rcp_sqrt_fallback(case, dtype):
    nx, nsteps = 2048, 24
    rng = np.random.default_rng(7)
    big = 1000 if dtype == np.float64 else 120
    rho = 1 + 0.3 * rng.uniform(-1, 1, nx)
    vel = 0.3 * rng.uniform(-1, 1, nx)
    p = 1 + 0.3 * rng.uniform(-1, 1, nx)
    if case == "tiny-density":        # rho, m, E all scaled by 2^-big: 1 / rho leaves the fast path's exponent range (f64)
        scale_rho, scale_p = 2.0 ** -big, 2.0 ** -big
    elif case == "huge-density":      # 1 / rho is subnormal
        big = 1022 if dtype == np.float64 else 126
        scale_rho, scale_p = 2.0 ** big, 2.0 ** big
        vel, p = 0.01 * vel, 0.01 * p
    else:                             # c^2 = gamma p / rho below the square root's fast range
        scale_rho, scale_p = 1.0, 2.0 ** -(big + 10)
        vel = 0.0 * vel
    U0 = wl.euler_conserved(rho * scale_rho, vel, p * scale_p).astype(dtype)
    assert np.all(np.isfinite(U0)) and np.all(U0[0] > 0)
    w = wl.Workload(wl.EULER, nx, 1.0 / nx, 0.2 / nx, U0.astype(np.float64), name="euler-" + case)
    ref = run_oracle(w, dtype, nsteps, u0=U0)
    assert np.all(np.isfinite(ref)) and not np.array_equal(ref, U0)
    assert_bits_equal(run_naive(w, dtype, nsteps, u0=U0), ref, f"classic vs oracle, {case}")
    for kernel in (SMEM_V, BAND_V):
        assert_bits_equal(run_swept(w, dtype, nsteps, 256, kernel, u0=U0), ref, f"swept vs oracle, {case}")


# ------------------------------------------------------------------------------------------------------------
# ring kernel (SWEPT_OPT_CHAIN = 3, the default): communication warp, cp.async-staged exchange, remainder inside the launch
# ------------------------------------------------------------------------------------------------------------
RING_CASES = [
    # problem, dtype, nx, W, q, r                   what it exercises
    (wl.HEAT, np.float64, 256, 128, 9, 0),          # two bands, each the other's neighbour on both sides; 16-iteration chunks
    (wl.HEAT, np.float64, 1 << 11, 128, 5, 37),     # odd remainder: truncated closing cycle, final values from two alignments
    (wl.HEAT, np.float64, 1 << 12, 128, 1, 0),      # q = 1: upright triangle straight into the closing triangle
    (wl.HEAT, np.float64, 1 << 12, 128, 0, 63),     # q = 0: only the truncated cycle, remainder L - 1
    (wl.HEAT, np.float64, 1 << 12, 256, 0, 1),
    (wl.HEAT, np.float64, 1 << 12, 256, 2, 127),
    (wl.HEAT, np.float32, 1 << 16, 256, 40, 3),     # one band per warp, many phases (SR = 2 iterations)
    (wl.HEAT, np.float64, 1 << 22, 1024, 5, 336),   # 4096 bands on 148 x 15 warps: 1 or 2 bands per warp, parked columns
    (wl.HEAT, np.float32, 1 << 22, 256, 5, 100),    # 16384 bands: several bands per warp, rotating parked buffers
    (wl.HEAT, np.float64, 1 << 21, 128, 6, 11),     # SR = 1 tiles, 16384 bands
    (wl.HEAT, np.float32, 1 << 22, 512, 5, 255),    # four super-rows per iteration
    (wl.HEAT, np.float64, 1 << 21, 512, 3, 2),
    (wl.HEAT, np.float64, 1 << 16, 512, 7, 77),     # roomy build (no more bands than 3 warps per SM)
    (wl.KS, np.float64, 1 << 14, 256, 11, 5),
    (wl.KS, np.float32, 1 << 21, 256, 4, 31),       # 8192 bands, several per warp
    (wl.KS, np.float64, 1 << 20, 1024, 3, 100),
    (wl.KS, np.float64, 1 << 22, 512, 2, 63),       # the size the band kernel could not hold in shared memory (per-warp packing)
    (wl.KS, np.float32, 1 << 22, 512, 3, 1),
    (wl.EULER, np.float64, 1 << 13, 256, 7, 3),
    (wl.EULER, np.float32, 1 << 20, 256, 3, 17),
    (wl.EULER, np.float64, 1 << 18, 512, 2, 50),
    (wl.EULER, np.float64, 1 << 20, 256, 3, 9),     # config 4's largest grid: 4096 bands, parked columns packed per warp
    (wl.EULER, np.float32, 1 << 21, 512, 2, 0),      # 4096 bands of 3 fields: 3 or 2 bands per warp
]


@pytest.mark.parametrize("problem,dtype,nx,W,q,r", RING_CASES)
def test_ring_kernel_equals_classic(problem, dtype, nx, W, q, r):
    import torch
    w = _noise(problem, nx)
    assert r < _sph(problem, W)
    nsteps = q * _sph(problem, W) + r
    with solver_for(w, dtype) as s:
        assert s.tile_width_ok(W)
        u = to_dev(w.initial(dtype))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        info = s.info()
        assert info["last_sweep_launch"] == sw.LAUNCH_RING, "this case must run on swept_ring_kernel, not fall back"
        assert info["launches_last_call"] == 1, "remainder included, a swept_run is one launch"
        got = u.cpu().numpy()
    assert_bits_equal(got, run_naive(w, dtype, nsteps), f"ring nx={nx} W={W} q={q} r={r}")


def test_ring_repeated_calls_two_handles_two_streams_and_graph_replay():
    import torch
    w = _noise(wl.KS, 1 << 18)
    s1, s2 = solver_for(w, np.float64), solver_for(w, np.float64)
    s2.set_option(sw.OPT_SWEPT_GRAPH, 1)
    st1, st2 = torch.cuda.Stream(), torch.cuda.Stream()
    u1, u2 = to_dev(w.initial(np.float64)), to_dev(w.initial(np.float64))
    torch.cuda.synchronize()
    for _ in range(3):
        s1.swept_run(u1, 333, 256, stream=st1)
        s2.swept_run(u2, 333, 256, stream=st2)
    torch.cuda.synchronize()
    assert s1.info()["last_sweep_launch"] == sw.LAUNCH_RING
    ref = run_naive(w, np.float64, 999)
    assert_bits_equal(u1.cpu().numpy(), ref, "stream 1")
    assert_bits_equal(u2.cpu().numpy(), ref, "stream 2 (graph replay)")
    s1.close(); s2.close()


# ------------------------------------------------------------------------------------------------------------
# packed pairs of bands (SWEPT_OPT_PACK = 2): heat fp32 on the band kernel, two bands per warp slot on f32x2 arithmetic
# ------------------------------------------------------------------------------------------------------------
PACK_CASES = [
    # nx, W, q                        what it exercises
    (512, 128, 9),                    # four bands = two slots: each slot is the other's left neighbour, components swapped at the wrap
    (1 << 12, 128, 1),                # q = 1
    (1 << 16, 256, 40),               # one slot per warp, many phases
    (1 << 20, 512, 7),                # four super-rows per iteration
    (1 << 22, 1024, 5),               # the bench size: 2048 slots on 148 x 16 warps
    (1 << 22, 256, 5),                # 8192 slots: several per warp, parked pairs swapped through shared memory
    (1 << 21, 128, 6),
]


@pytest.mark.parametrize("nx,W,q", PACK_CASES)
def test_packed_band_pairs_equal_classic(nx, W, q):
    import torch
    w = _noise(wl.HEAT, nx)
    nsteps = q * _sph(wl.HEAT, W) + 3
    with solver_for(w, np.float32) as s:
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
        s.set_option(sw.OPT_PACK, sw.PACK_ON)
        u = to_dev(w.initial(np.float32))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        assert s.info()["last_sweep_launch"] == sw.LAUNCH_BAND
        got = u.cpu().numpy()
    assert_bits_equal(got, run_naive(w, np.float32, nsteps), f"packed band pairs nx={nx} W={W} q={q}")
    # and the same run with one band per slot gives the same bits
    assert_bits_equal(got, run_swept(w, np.float32, nsteps, W, BAND_V, opts={sw.OPT_PACK: sw.PACK_OFF}), "packed vs one band per slot")


@pytest.mark.parametrize("nx,W,q,r", [
    (1 << 10, 256, 5, 0),             # four bands = two slots (KS band tiles start at W = 256: 64 iterations per tile)
    (1 << 12, 256, 1, 3),             # q = 1 + a remainder (truncated closing cycle)
    (1 << 16, 256, 9, 17),
    (1 << 20, 512, 4, 63),
    (1 << 22, 1024, 3, 100),          # the config-5 size: 2048 slots
    (1 << 22, 256, 3, 5),             # 8192 slots: several per warp, parked pairs
    (1 << 12, 256, 0, 15),            # q = 0: only the truncated cycle
])
def test_packed_band_pairs_ks_equal_classic(nx, W, q, r):
    """KS fp32 on packed f32x2 arithmetic (two sub-timesteps per timestep, radius 2, immediate and negated operands): same bits."""
    import torch
    w = _noise(wl.KS, nx)
    nsteps = q * _sph(wl.KS, W) + r
    with solver_for(w, np.float32) as s:
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
        s.set_option(sw.OPT_PACK, sw.PACK_ON)
        u = to_dev(w.initial(np.float32))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        info = s.info()
        assert info["last_sweep_launch"] == sw.LAUNCH_BAND and info["launches_last_call"] == 1
        got = u.cpu().numpy()
    assert_bits_equal(got, run_naive(w, np.float32, nsteps), f"KS packed band pairs nx={nx} W={W} q={q} r={r}")
    assert_bits_equal(got, run_swept(w, np.float32, nsteps, W, BAND_V, opts={sw.OPT_PACK: sw.PACK_OFF}), "packed vs one band per slot")
    if nx <= 1 << 16:
        assert_bits_equal(got, run_oracle(w, np.float32, nsteps), "KS packed pairs vs oracle")


@pytest.mark.parametrize("problem,dtype,nx,W,q,r,pack", [
    (wl.HEAT, np.float64, 1 << 11, 128, 5, 37, 0),       # odd remainder
    (wl.HEAT, np.float64, 1 << 12, 128, 0, 63, 0),       # q = 0: only the truncated cycle, remainder L - 1
    (wl.HEAT, np.float64, 1 << 22, 1024, 3, 336, 0),     # the bench shape: 1 or 2 bands per warp
    (wl.HEAT, np.float32, 1 << 22, 1024, 3, 335, 2),     # packed pairs, odd remainder
    (wl.HEAT, np.float32, 1 << 21, 128, 4, 11, 2),       # packed pairs, several slots per warp
    (wl.KS, np.float64, 1 << 20, 512, 3, 63, 0),
    (wl.EULER, np.float64, 1 << 18, 256, 2, 17, 0),
])
def test_band_kernel_runs_the_remainder_as_a_truncated_closing_cycle(problem, dtype, nx, W, q, r, pack):
    import torch
    w = _noise(problem, nx)
    nsteps = q * _sph(problem, W) + r
    with solver_for(w, dtype) as s:
        s.set_option(sw.OPT_CHAIN, sw.CHAIN_BANDS)
        if pack:
            s.set_option(sw.OPT_PACK, pack)
        u = to_dev(w.initial(dtype))
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        info = s.info()
        assert info["last_sweep_launch"] == sw.LAUNCH_BAND and info["launches_last_call"] == 1
        got = u.cpu().numpy()
    assert_bits_equal(got, run_naive(w, dtype, nsteps), f"band, truncated cycle nx={nx} W={W} q={q} r={r}")
