"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding, return numpy arrays."""
from __future__ import annotations

import numpy as np

import oracle
import paper_1612_02495_b200 as sw
import workloads as wl

TOL = {np.float64: 1e-12, np.float32: 1e-5}     # north_star: relative max-norm vs the oracle


def solver_for(w: wl.Workload, dtype, **kw) -> sw.Solver:
    return sw.Solver(w.problem, w.nx, w.dx, w.dt, dtype=sw.F64 if dtype == np.float64 else sw.F32,
                     alpha=w.alpha, gamma=w.gamma, **kw)


def to_dev(a: np.ndarray):
    import torch
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def run_naive(w: wl.Workload, dtype, nsteps: int, u0=None, graph: bool = False) -> np.ndarray:
    import torch
    with solver_for(w, dtype) as s:
        if graph:
            s.set_option(sw.OPT_NAIVE_GRAPH, 1)
        u = to_dev(w.initial(dtype) if u0 is None else u0)
        s.naive_run(u, nsteps)
        torch.cuda.synchronize()
        return u.cpu().numpy()


# the swept kernel variants every parity test runs: (kernel family, chain option)
SMEM, WAVE, CHAIN, BAND, RING = (sw.KERNEL_SMEM, 0), (sw.KERNEL_WAVE, 0), (sw.KERNEL_WAVE, 1), (sw.KERNEL_WAVE, 2), (sw.KERNEL_WAVE, 3)
VARIANTS = [SMEM, WAVE, CHAIN, BAND, RING]
VARIANT_IDS = ["smem", "wave", "chain", "band", "ring"]


def _select(s: sw.Solver, kernel) -> None:
    if isinstance(kernel, tuple):
        s.set_option(sw.OPT_KERNEL, kernel[0])
        s.set_option(sw.OPT_CHAIN, kernel[1])
    else:
        s.set_option(sw.OPT_KERNEL, kernel)


def run_swept(w: wl.Workload, dtype, nsteps: int, W: int, kernel, u0=None, graph: bool = False, opts=None) -> np.ndarray:
    import torch
    with solver_for(w, dtype) as s:
        _select(s, kernel)
        if graph:
            s.set_option(sw.OPT_SWEPT_GRAPH, 1)
        for k, v in (opts or {}).items():
            s.set_option(k, v)
        u = to_dev(w.initial(dtype) if u0 is None else u0)
        s.swept_run(u, nsteps, W)
        torch.cuda.synchronize()
        return u.cpu().numpy()


def width_ok(w: wl.Workload, dtype, W: int, kernel) -> bool:
    with solver_for(w, dtype) as s:
        _select(s, kernel)
        return s.tile_width_ok(W)


def run_oracle(w: wl.Workload, dtype, nsteps: int, u0=None) -> np.ndarray:
    a = w.initial(dtype) if u0 is None else np.ascontiguousarray(u0)
    return oracle.run(w.problem, a, nsteps, dx=w.dx, dt=w.dt, alpha=w.alpha, gamma=w.gamma)


def rel_max(a: np.ndarray, b: np.ndarray) -> float:
    """Reading S7: max|a-b| / max|b| per field, worst field (b = oracle)."""
    a = a.reshape(b.shape)
    worst = 0.0
    for k in range(b.shape[0]):
        den = max(float(np.max(np.abs(b[k]))), np.finfo(b.dtype).tiny)
        worst = max(worst, float(np.max(np.abs(a[k].astype(np.float64) - b[k].astype(np.float64)))) / den)
    return worst


def assert_bits_equal(a: np.ndarray, b: np.ndarray, what: str = "") -> None:
    a = a.reshape(b.shape)
    ai = a.view(np.uint64 if a.dtype == np.float64 else np.uint32)
    bi = b.view(np.uint64 if b.dtype == np.float64 else np.uint32)
    if not np.array_equal(ai, bi):
        bad = np.argwhere(ai != bi)
        raise AssertionError(f"{what}: {len(bad)} of {a.size} values differ bitwise; first at {bad[0].tolist()}: "
                             f"{a[tuple(bad[0])]!r} vs {b[tuple(bad[0])]!r}; rel max {rel_max(a, b):.3e}")
