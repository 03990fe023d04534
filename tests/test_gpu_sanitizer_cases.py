"""-m gpu: one SMALL case per kernel family and per synchronisation mechanism, sized so that the whole file also finishes
under compute-sanitizer (memcheck / racecheck / synccheck slow a kernel down by one to two orders of magnitude):

    compute-sanitizer --tool racecheck python -m pytest tests/test_gpu_sanitizer_cases.py -m gpu -q

(summaries of those runs: profiles/r2_sanitizer.md).  The cases are ordinary bit-exactness tests and run in the normal suite too.
"""
import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import BAND, CHAIN, SMEM, WAVE, assert_bits_equal, run_naive, run_swept, solver_for, to_dev

pytestmark = pytest.mark.gpu

CASES = [
    # id, problem, dtype, nx, W, half-cycles, variant, options
    ("band-heat-f64-1-band-per-warp", wl.HEAT, np.float64, 1 << 13, 256, 3, BAND, {}),
    ("band-heat-f32-sr4", wl.HEAT, np.float32, 1 << 13, 512, 2, BAND, {}),
    ("band-ks-f64", wl.KS, np.float64, 1 << 13, 256, 2, BAND, {}),
    ("band-euler-f64", wl.EULER, np.float64, 1 << 12, 256, 2, BAND, {}),
    # 1024 bands on 148 x 4 warps: two bands per warp, parked columns swapped through shared memory
    ("band-heat-f32-2-bands-per-warp", wl.HEAT, np.float32, 1 << 17, 128, 3, BAND, {sw.OPT_BLOCKS_PER_SM: 1}),
    ("chain-heat-f64", wl.HEAT, np.float64, 1 << 12, 128, 3, CHAIN, {}),
    ("chain-euler-f32", wl.EULER, np.float32, 1 << 12, 128, 2, CHAIN, {}),
    ("wave-ks-f32", wl.KS, np.float32, 1 << 12, 128, 3, WAVE, {}),
    ("smem-heat-f64", wl.HEAT, np.float64, 1 << 12, 256, 3, SMEM, {}),
    ("smem-euler-f64", wl.EULER, np.float64, 1 << 11, 128, 2, SMEM, {}),
]


@pytest.mark.parametrize("name,problem,dtype,nx,W,q,variant,opts", CASES, ids=[c[0] for c in CASES])
def test_small_case_per_kernel_family(name, problem, dtype, nx, W, q, variant, opts):
    w = wl.make(problem, nx, "noise")
    nsteps = q * wl.steps_per_half_cycle(problem, W) + 3          # + a remainder: narrower tiles and a classic step
    got = run_swept(w, dtype, nsteps, W, variant, opts=opts)
    assert_bits_equal(got, run_naive(w, dtype, nsteps), name)


def test_small_rod_with_insulated_ends():
    import torch
    w = wl.heat_rod(1 << 12)
    u0 = w.initial(np.float64)
    with sw.Solver(w.problem, w.nx, w.dx, w.dt, dtype=sw.F64, alpha=w.alpha, boundary=sw.BC_INSULATED) as s:
        us, un = to_dev(u0), to_dev(u0)
        s.swept_run(us, 3 * 64 + 5, 128)
        s.naive_run(un, 3 * 64 + 5)
        torch.cuda.synchronize()
        assert_bits_equal(us.cpu().numpy(), un.cpu().numpy(), "rod, tile-flag kernel for insulated ends")
