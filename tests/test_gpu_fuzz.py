"""-m gpu: seeded random sampling of the (problem, dtype, nx, tile width, kernel variant, step count, options) space:
swept_run == naive_run bit for bit.  The hand-picked parity cases cover the corners the design names; this covers the
combinations nobody thought of (odd remainders on many-band grids, one tile, two tiles, narrow tiles on large grids, caps).
FUZZ_CASES (environment) raises the number of cases for a soak run; the default finishes in about a minute.
"""
import os

import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import VARIANT_IDS, VARIANTS, assert_bits_equal, solver_for, to_dev

pytestmark = pytest.mark.gpu

N_CASES = int(os.environ.get("FUZZ_CASES", "400"))


def _cases(n, seed=16122495):
    rng = np.random.default_rng(seed)
    out = []
    while len(out) < n:
        problem = int(rng.choice([wl.HEAT, wl.KS, wl.EULER], p=[0.45, 0.3, 0.25]))
        dtype = np.float64 if rng.random() < 0.6 else np.float32
        lg = int(rng.integers(7, 18 if problem != wl.EULER else 16))
        vi = int(rng.integers(0, len(VARIANTS)))
        W = 1 << int(rng.integers(3, 12))
        if W > (1 << lg):
            continue
        halfs = int(rng.integers(0, 6))
        rem = int(rng.integers(0, max(1, wl.steps_per_half_cycle(problem, W))))
        opts = {}
        if rng.random() < 0.25:
            opts[sw.OPT_BLOCKS_PER_SM] = int(rng.integers(1, 5))
        if problem == wl.HEAT and dtype == np.float32 and rng.random() < 0.5:
            opts[sw.OPT_PACK] = int(rng.integers(1, 3))
        out.append((problem, dtype, lg, vi, W, halfs, rem, opts))
    return out


CASES = _cases(N_CASES)


@pytest.mark.parametrize("chunk", range((len(CASES) + 19) // 20))
def test_random_configurations_match_the_classic_path_bitwise(chunk):
    import torch
    ran = 0
    for problem, dtype, lg, vi, W, halfs, rem, opts in CASES[20 * chunk: 20 * chunk + 20]:
        w = wl.make(problem, 1 << lg, "noise")
        sph = wl.steps_per_half_cycle(problem, W)
        if sph < 1:
            continue
        nsteps = halfs * sph + rem
        if nsteps == 0 or nsteps > 6000:
            continue
        u0 = w.initial(dtype)
        with solver_for(w, dtype) as s:
            s.set_option(sw.OPT_KERNEL, VARIANTS[vi][0])
            s.set_option(sw.OPT_CHAIN, VARIANTS[vi][1])
            if not s.tile_width_ok(W):
                continue
            for k, v in opts.items():
                s.set_option(k, v)
            us, un = to_dev(u0), to_dev(u0)
            s.swept_run(us, nsteps, W)
            s.naive_run(un, nsteps)
            torch.cuda.synchronize()
            what = (f"{wl.PROBLEM_NAMES[problem]} {np.dtype(dtype).name} nx=2^{lg} W={W} {VARIANT_IDS[vi]} nsteps={nsteps} "
                    f"({halfs} half-cycles + {rem}) opts={opts} ran={sw.LAUNCH_NAMES.get(s.info()['last_sweep_launch'], '-')}")
            assert_bits_equal(us.cpu().numpy(), un.cpu().numpy(), what)
            ran += 1
    print(f"fuzz chunk {chunk}: {ran} of 20 sampled configurations were legal and ran")
    assert ran >= 3, ran
