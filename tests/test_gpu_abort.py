"""-m gpu: the error path of the bounded waits (include/swept1d.h, "Conventions"): a launch-free sweep that gave up a wait marks
the handle; the mark is reported once as SWEPT_ECUDA -- by swept_check, by the next call made after the launch has finished, by
swept_run_host -- and the handle works afterwards.  The mark is injected (SWEPT_OPT_INJECT_ABORT): a real one needs a hung GPU."""
import numpy as np
import pytest

import paper_1612_02495_b200 as sw
import workloads as wl
from gpu_util import assert_bits_equal, solver_for, to_dev

pytestmark = pytest.mark.gpu

NSTEPS, W = 300, 256


def _good(s, u0):
    import torch
    u = to_dev(u0)
    s.swept_run(u, NSTEPS, W)
    s.check()
    torch.cuda.synchronize()
    return u.cpu().numpy()


@pytest.mark.parametrize("chain", [sw.CHAIN_RING, sw.CHAIN_BANDS, sw.CHAIN_TILES], ids=["ring", "band", "chain"])
def test_abort_is_reported_exactly_once_and_the_handle_recovers(chain):
    import torch
    w = wl.heat_noise(1 << 14)
    u0 = w.initial(np.float64)
    with solver_for(w, np.float64) as s:
        s.set_option(sw.OPT_CHAIN, chain)
        want = _good(s, u0)
        s.check()                                            # nothing to report on a healthy handle

        # reported by swept_check
        s.set_option(sw.OPT_INJECT_ABORT, 1)
        s.swept_run(to_dev(u0), NSTEPS, W)                   # this field is invalid
        with pytest.raises(sw.SweptError) as ei:
            s.check()
        assert ei.value.code == sw.ECUDA and "gave up" in str(ei.value)
        s.check()                                            # once only
        assert_bits_equal(_good(s, u0), want, "after swept_check reported the abort")

        # reported by the next call made after the marked launch has finished
        s.set_option(sw.OPT_INJECT_ABORT, 1)
        s.swept_run(to_dev(u0), NSTEPS, W)
        torch.cuda.synchronize()
        with pytest.raises(sw.SweptError) as ei:
            s.swept_run(to_dev(u0), NSTEPS, W)
        assert ei.value.code == sw.ECUDA
        assert_bits_equal(_good(s, u0), want, "after swept_run reported the abort")

        # reported by swept_run_host itself, which hands back the invalid field
        s.set_option(sw.OPT_INJECT_ABORT, 1)
        h = u0.copy()
        with pytest.raises(sw.SweptError) as ei:
            s.run_host(h, NSTEPS, W)
        assert ei.value.code == sw.ECUDA
        h = u0.copy()
        s.run_host(h, NSTEPS, W)
        assert_bits_equal(h, want, "swept_run_host after it reported the abort")
        s.check()


def test_tile_width_ok_agrees_with_swept_run_after_tuning():
    """swept_tune may choose the paper-style shared-memory kernels (small Euler grids); swept_tile_width_ok answers for the family
    swept_run will use for that width."""
    import torch
    w = wl.euler_noise(1 << 12)
    with solver_for(w, np.float64) as s:
        scratch = to_dev(w.initial(np.float64))
        best = s.tune(scratch)
        assert s.tile_width_ok(best), (best, s.info())
        u = to_dev(w.initial(np.float64))
        s.swept_run(u, 64, best)
        torch.cuda.synchronize()
