"""paper_1612_02495_b200 -- B200-native swept time-space decomposition for explicit 1-D PDE time stepping.

Thin ctypes binding of the C ABI in include/swept1d.h (libswept1d.so, hand-written CUDA for sm_100a).
Argument marshalling only: every step of the hot path -- the upright-triangle, diamond and closing
inverted-triangle kernels (Fig. 5), the edge-exchange staircases, the
classic one-kernel-per-sub-timestep path (Fig. 6) and the tile-width tuner --
runs inside the library.  torch is used for device memory and streams only.

There is no CPU fallback: importing works without a GPU (so the symbols can be checked), but every compute
call raises `SweptError` if the library or a CUDA device is missing.
"""
from __future__ import annotations

import ctypes
import os
from typing import Optional

HEAT, KS, EULER = 0, 1, 2
F32, F64 = 0, 1
KERNEL_SMEM, KERNEL_WAVE = 0, 1
OPT_KERNEL, OPT_NAIVE_GRAPH, OPT_BLOCKS_PER_SM, OPT_WARPS_PER_BLOCK, OPT_SWEPT_GRAPH, OPT_CHAIN, OPT_PACK, OPT_NAIVE_SHARE, OPT_INJECT_ABORT = 0, 1, 2, 3, 4, 5, 6, 7, 8
PACK_AUTO, PACK_OFF, PACK_ON = 0, 1, 2
LAUNCH_CLASSIC, LAUNCH_UP, LAUNCH_DIAMOND, LAUNCH_DOWN, LAUNCH_CHAIN, LAUNCH_BAND, LAUNCH_RING = 0, 1, 2, 3, 4, 5, 6
LAUNCH_NAMES = {0: "classic", 1: "up", 2: "diamond", 3: "down", 4: "chain", 5: "band", 6: "ring"}
BC_PERIODIC, BC_INSULATED = 0, 1
OPT2D_KERNEL, KERNEL2D_WARP, KERNEL2D_SMEM, KERNEL2D_COLUMN = 0, 0, 1, 2      # include/swept2d.h: swept2d_set_option
CHAIN_OFF, CHAIN_TILES, CHAIN_BANDS, CHAIN_RING = 0, 1, 2, 3     # values of OPT_CHAIN (include/swept1d.h); CHAIN_RING is the default
OK, EINVAL, ENOMEM, ECUDA = 0, -1, -2, -3
PROBLEMS = {"heat": HEAT, "ks": KS, "euler": EULER}

# every symbol include/swept1d.h declares
SYMBOLS = (
    "swept_create", "swept_run", "naive_run", "swept_tune", "swept_run_host", "swept_set_option", "swept_get_info",
    "swept_tile_width_ok", "swept_measure_alu_peak", "swept_destroy", "swept_last_error", "swept_version", "swept_plan",
    "swept_band_layout", "swept_band_owner", "swept_problem_info", "swept_measure_smem_peak", "swept_measure_latencies",
    "swept_run_static", "swept_check",
    # include/swept2d.h
    "swept2d_create", "swept2d_run", "naive2d_run", "swept2d_set_option", "swept2d_get_info", "swept2d_destroy", "swept2d_run_host",
)

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libswept1d.so")


class SweptError(RuntimeError):
    def __init__(self, code: int, message: str):
        super().__init__(f"[{code}] {message}")
        self.code = code


class _Params(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("alpha", ctypes.c_double), ("gamma", ctypes.c_double), ("max_tile_width", ctypes.c_int),
                ("boundary", ctypes.c_int)]


class _Info(ctypes.Structure):
    _fields_ = [
        ("problem", ctypes.c_int), ("dtype", ctypes.c_int), ("radius", ctypes.c_int), ("stages", ctypes.c_int), ("ncomp", ctypes.c_int),
        ("nx", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64), ("tuned_tile_width", ctypes.c_int),
        ("launches_last_call", ctypes.c_int64), ("launches_total", ctypes.c_int64), ("sm_count", ctypes.c_int),
        ("max_smem_per_block", ctypes.c_int), ("last_sweep_launch", ctypes.c_int), ("boundary", ctypes.c_int), ("tuned_chain", ctypes.c_int), ("tuned_blocks_per_sm", ctypes.c_int),
        ("tuned_pack", ctypes.c_int), ("tuned_kernel", ctypes.c_int),
    ]


class _Launch(ctypes.Structure):
    _fields_ = [("kind", ctypes.c_int), ("tile_width", ctypes.c_int), ("offset", ctypes.c_int64), ("count", ctypes.c_int64)]


class _BandLayout(ctypes.Structure):
    _fields_ = [(n, ctypes.c_int) for n in ("blocks", "warps_per_block", "slots_per_block", "warps_per_slot", "slots", "max_bands_per_warp", "ntiles")]


class _Params2D(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("alpha", ctypes.c_double)]


class _Info2D(ctypes.Structure):
    _fields_ = [("dtype", ctypes.c_int), ("nx", ctypes.c_int64), ("ny", ctypes.c_int64), ("workspace_bytes", ctypes.c_int64),
                ("launches_last_call", ctypes.c_int64), ("launches_total", ctypes.c_int64)]


_lib = None


def build(force: bool = False) -> str:
    """Compile the CUDA sources in-tree (nvcc, sm_100a)."""
    from . import _build
    return _build.build(force=force)


def lib() -> ctypes.CDLL:
    """Load libswept1d.so (building it if the sources are newer).  Raises if it cannot be had."""
    global _lib
    if _lib is not None:
        return _lib
    if not os.path.exists(LIB_PATH) or os.environ.get("SWEPT1D_REBUILD"):
        build()
    if not os.path.exists(LIB_PATH):
        raise SweptError(ECUDA, f"{LIB_PATH} is missing and could not be built; there is no CPU fallback")
    L = ctypes.CDLL(LIB_PATH)
    vp, i64, ci, dbl = ctypes.c_void_p, ctypes.c_int64, ctypes.c_int, ctypes.c_double
    L.swept_create.argtypes = [ctypes.POINTER(vp), ci, i64, dbl, dbl, ctypes.POINTER(_Params)]
    L.swept_run.argtypes = [vp, vp, i64, ci, vp]
    L.naive_run.argtypes = [vp, vp, i64, vp]
    L.swept_tune.argtypes = [vp, vp, ci, ctypes.POINTER(ci), vp]
    L.swept_run_host.argtypes = [vp, vp, i64, ci, ci, vp]
    L.swept_run_static.argtypes = [ci, i64, dbl, dbl, ctypes.POINTER(_Params), vp, i64, ci, vp]
    L.swept_set_option.argtypes = [vp, ci, ci]
    L.swept_get_info.argtypes = [vp, ctypes.POINTER(_Info)]
    L.swept_tile_width_ok.argtypes = [vp, ci]
    L.swept_measure_alu_peak.argtypes = [ci, ctypes.POINTER(dbl), ctypes.POINTER(dbl), vp]
    L.swept_destroy.argtypes = [vp]
    L.swept_check.argtypes = [vp]
    L.swept_plan.argtypes = [ci, ci, i64, i64, ci, ci, ci, ctypes.POINTER(_Launch), i64]
    L.swept_band_layout.argtypes = [ci, ci, ci, ctypes.POINTER(_BandLayout)]
    L.swept_band_owner.argtypes = [ctypes.POINTER(_BandLayout), ci, ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(ci)]
    L.swept_problem_info.argtypes = [ci, ctypes.POINTER(ci), ctypes.POINTER(ci), ctypes.POINTER(ci)]
    L.swept_measure_smem_peak.argtypes = [ctypes.POINTER(dbl), ctypes.POINTER(dbl), vp]
    L.swept_measure_latencies.argtypes = [ctypes.POINTER(dbl), vp]
    L.swept2d_create.argtypes = [ctypes.POINTER(vp), i64, i64, dbl, dbl, ctypes.POINTER(_Params2D)]
    L.swept2d_run.argtypes = [vp, vp, i64, ci, vp]
    L.naive2d_run.argtypes = [vp, vp, i64, vp]
    L.swept2d_run_host.argtypes = [vp, vp, i64, ci, ci, vp]
    L.swept2d_set_option.argtypes = [vp, ci, ci]
    L.swept2d_get_info.argtypes = [vp, ctypes.POINTER(_Info2D)]
    L.swept2d_destroy.argtypes = [vp]
    for name in SYMBOLS:
        getattr(L, name).restype = ci
    L.swept_plan.restype = i64
    L.swept_last_error.restype = ctypes.c_char_p
    L.swept_last_error.argtypes = []
    L.swept_version.restype = ctypes.c_char_p
    L.swept_version.argtypes = []
    _lib = L
    return L


def _check(rc: int) -> None:
    if rc != 0:
        raise SweptError(rc, lib().swept_last_error().decode("utf-8", "replace"))


def version() -> str:
    return lib().swept_version().decode()


def _stream_ptr(stream) -> int:
    import torch
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dtype_id(dtype) -> int:
    import torch
    if dtype in (F32, F64) and not isinstance(dtype, torch.dtype):
        return int(dtype)
    if dtype == torch.float64:
        return F64
    if dtype == torch.float32:
        return F32
    raise SweptError(EINVAL, f"unsupported dtype {dtype}")


class Solver:
    """One `swept_create` handle.  `u` arguments are CUDA torch tensors of shape [ncomp, nx] (or [nx] when
    ncomp == 1), contiguous, of the handle's dtype; they are advanced IN PLACE and asynchronously on `stream`."""

    def __init__(self, problem, nx: int, dx: float, dt: float, *, dtype=F64, alpha: float = 1.0, gamma: float = 1.4,
                 max_tile_width: int = 0, boundary: int = 0):
        if isinstance(problem, str):
            problem = PROBLEMS[problem]
        self._h = ctypes.c_void_p()
        self.problem, self.nx, self.dtype = int(problem), int(nx), _dtype_id(dtype)
        p = _Params(self.dtype, float(alpha), float(gamma), int(max_tile_width), int(boundary))
        _check(lib().swept_create(ctypes.byref(self._h), self.problem, self.nx, float(dx), float(dt), ctypes.byref(p)))
        import torch
        self.device = torch.cuda.current_device()      # swept_create binds the handle to the current device
        self.ncomp = self.info()["ncomp"]

    # -- marshalling ----------------------------------------------------------------------------------------
    def _ptr(self, u) -> int:
        import torch
        want = torch.float64 if self.dtype == F64 else torch.float32
        if not (isinstance(u, torch.Tensor) and u.is_cuda and u.is_contiguous() and u.dtype == want):
            raise SweptError(EINVAL, "u must be a contiguous CUDA tensor of the handle's dtype")
        if u.device.index != self.device:
            raise SweptError(EINVAL, f"u lives on cuda:{u.device.index} but the handle was created on cuda:{self.device}")
        if u.numel() != self.ncomp * self.nx:
            raise SweptError(EINVAL, f"u must hold ncomp*nx = {self.ncomp * self.nx} elements")
        return u.data_ptr()

    def swept_run(self, u, nsteps: int, tile_width: int = 0, stream=None) -> None:
        _check(lib().swept_run(self._h, self._ptr(u), int(nsteps), int(tile_width), _stream_ptr(stream)))

    def naive_run(self, u, nsteps: int, stream=None) -> None:
        _check(lib().naive_run(self._h, self._ptr(u), int(nsteps), _stream_ptr(stream)))

    def tune(self, scratch, blocks_per_sm_cap: int = 0, stream=None) -> int:
        best = ctypes.c_int(0)
        _check(lib().swept_tune(self._h, self._ptr(scratch), int(blocks_per_sm_cap), ctypes.byref(best), _stream_ptr(stream)))
        return best.value

    def run_host(self, h_u, nsteps: int, tile_width: int = 0, use_swept: bool = True, stream=None) -> None:
        """h_u: CPU torch tensor or numpy array ([ncomp, nx], contiguous, the handle's dtype; pinned is best); updated in place."""
        import numpy as np
        import torch
        if isinstance(h_u, torch.Tensor):
            if h_u.is_cuda or not h_u.is_contiguous():
                raise SweptError(EINVAL, "h_u must be a contiguous CPU tensor")
            ptr, n, es = h_u.data_ptr(), h_u.numel(), h_u.element_size()
        elif isinstance(h_u, np.ndarray) and h_u.flags["C_CONTIGUOUS"]:
            ptr, n, es = h_u.ctypes.data, h_u.size, h_u.itemsize
        else:
            raise SweptError(EINVAL, "h_u must be a contiguous CPU tensor or numpy array")
        if n != self.ncomp * self.nx or es != (8 if self.dtype == F64 else 4):
            raise SweptError(EINVAL, "h_u has the wrong size or dtype")
        _check(lib().swept_run_host(self._h, ptr, int(nsteps), int(tile_width), 1 if use_swept else 0, _stream_ptr(stream)))

    def set_option(self, key: int, value: int) -> None:
        _check(lib().swept_set_option(self._h, int(key), int(value)))

    def check(self) -> None:
        """swept_check: wait for the handle's work; raises SweptError(ECUDA) once if a launch-free sweep gave up a bounded wait."""
        _check(lib().swept_check(self._h))

    def tile_width_ok(self, tile_width: int) -> bool:
        return bool(lib().swept_tile_width_ok(self._h, int(tile_width)))

    def info(self) -> dict:
        i = _Info()
        _check(lib().swept_get_info(self._h, ctypes.byref(i)))
        return {name: getattr(i, name) for name, _ in _Info._fields_}

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().swept_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


class Solver2D:
    """One `swept2d_create` handle (include/swept2d.h): the 2-D heat equation on a periodic nx x ny grid.  `u` arguments are
    contiguous CUDA tensors of shape [ny, nx] of the handle's dtype, advanced IN PLACE and asynchronously on `stream`."""

    def __init__(self, nx: int, ny: int, dx: float, dt: float, *, dtype=F64, alpha: float = 1.0):
        self._h = ctypes.c_void_p()
        self.nx, self.ny, self.dtype = int(nx), int(ny), _dtype_id(dtype)
        p = _Params2D(self.dtype, float(alpha))
        _check(lib().swept2d_create(ctypes.byref(self._h), self.nx, self.ny, float(dx), float(dt), ctypes.byref(p)))
        import torch
        self.device = torch.cuda.current_device()

    def _ptr(self, u) -> int:
        import torch
        want = torch.float64 if self.dtype == F64 else torch.float32
        if not (isinstance(u, torch.Tensor) and u.is_cuda and u.is_contiguous() and u.dtype == want):
            raise SweptError(EINVAL, "u must be a contiguous CUDA tensor of the handle's dtype")
        if u.device.index != self.device or u.numel() != self.nx * self.ny:
            raise SweptError(EINVAL, f"u must hold ny*nx = {self.nx * self.ny} elements on cuda:{self.device}")
        return u.data_ptr()

    def swept_run(self, u, nsteps: int, tile_width: int = 0, stream=None) -> None:
        _check(lib().swept2d_run(self._h, self._ptr(u), int(nsteps), int(tile_width), _stream_ptr(stream)))

    def naive_run(self, u, nsteps: int, stream=None) -> None:
        _check(lib().naive2d_run(self._h, self._ptr(u), int(nsteps), _stream_ptr(stream)))

    def run_host(self, h_u, nsteps: int, tile_width: int = 0, use_swept: bool = True, stream=None) -> None:
        """h_u: contiguous CPU torch tensor or numpy array [ny, nx] of the handle's dtype (pinned is best); updated in place."""
        import numpy as np
        import torch
        if isinstance(h_u, torch.Tensor) and not h_u.is_cuda and h_u.is_contiguous():
            ptr, n, es = h_u.data_ptr(), h_u.numel(), h_u.element_size()
        elif isinstance(h_u, np.ndarray) and h_u.flags["C_CONTIGUOUS"]:
            ptr, n, es = h_u.ctypes.data, h_u.size, h_u.itemsize
        else:
            raise SweptError(EINVAL, "h_u must be a contiguous CPU tensor or numpy array")
        if n != self.nx * self.ny or es != (8 if self.dtype == F64 else 4):
            raise SweptError(EINVAL, "h_u has the wrong size or dtype")
        _check(lib().swept2d_run_host(self._h, ptr, int(nsteps), int(tile_width), 1 if use_swept else 0, _stream_ptr(stream)))

    def set_option(self, option: int, value: int) -> None:
        _check(lib().swept2d_set_option(self._h, int(option), int(value)))

    def info(self) -> dict:
        i = _Info2D()
        _check(lib().swept2d_get_info(self._h, ctypes.byref(i)))
        return {name: getattr(i, name) for name, _ in _Info2D._fields_}

    def close(self) -> None:
        if getattr(self, "_h", None) is not None and self._h.value:
            lib().swept2d_destroy(self._h)
            self._h = ctypes.c_void_p()

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


STATIC_SCRATCH_BYTES = 8 << 20      # SWEPT_STATIC_SCRATCH_BYTES (include/swept1d.h)


def swept_run_static(problem, u, nsteps: int, dx: float, dt: float, *, tile_width: int = 0, alpha: float = 1.0, gamma: float = 1.4,
                     stream=None) -> None:
    """`swept_run_static` (include/swept1d.h): advance `u` -- a contiguous CUDA tensor of shape [ncomp, nx] (or [nx]), float64 or
    float32 -- IN PLACE by `nsteps` timesteps with the swept rule, without a Solver and without any device allocation by the
    library.  For programs that cannot let a library call cudaMalloc: the GPU's memory belongs to their own pool, or an
    allocation's device-wide stall is not affordable where they call from.  The edge row a Solver would allocate is a fixed
    array inside the library (STATIC_SCRATCH_BYTES), so the field may hold at most that many bytes; calls on one device share the
    array and must not overlap on the GPU.  The first call per (device, problem, dtype) does a one-off set-up and belongs outside
    stream capture.  Same bits as Solver.swept_run / naive_run."""
    import torch
    if isinstance(problem, str):
        problem = PROBLEMS[problem]
    if not (isinstance(u, torch.Tensor) and u.is_cuda and u.is_contiguous() and u.dtype in (torch.float64, torch.float32)):
        raise SweptError(EINVAL, "u must be a contiguous CUDA tensor of dtype float64 or float32")
    if u.device.index != torch.cuda.current_device():
        raise SweptError(EINVAL, f"u lives on cuda:{u.device.index} but cuda:{torch.cuda.current_device()} is current")
    ncomp = problem_info(int(problem))["ncomp"]
    if u.numel() % ncomp:
        raise SweptError(EINVAL, f"u must hold ncomp = {ncomp} rows")
    p = _Params(_dtype_id(u.dtype), float(alpha), float(gamma), 0, BC_PERIODIC)
    _check(lib().swept_run_static(int(problem), u.numel() // ncomp, float(dx), float(dt), ctypes.byref(p), u.data_ptr(), int(nsteps),
                                  int(tile_width), _stream_ptr(stream)))


def measure_alu_peak(dtype=F64, stream=None) -> dict:
    """FMA-chain microbenchmark: thread-level FP instructions per second of the FP64 / FP32 pipe."""
    ips, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(lib().swept_measure_alu_peak(_dtype_id(dtype), ctypes.byref(ips), ctypes.byref(ms), _stream_ptr(stream)))
    return {"instr_per_s": ips.value, "ms": ms.value}


def measure_smem_peak(stream=None) -> dict:
    """Shared-memory read microbenchmark: bytes per second of conflict-free 16-byte loads on every SM."""
    bps, ms = ctypes.c_double(0), ctypes.c_double(0)
    _check(lib().swept_measure_smem_peak(ctypes.byref(bps), ctypes.byref(ms), _stream_ptr(stream)))
    return {"bytes_per_s": bps.value, "ms": ms.value}


def measure_latencies(stream=None) -> dict:
    """Latency probes (SM cycles per dependent operation, one warp): see swept_measure_latencies in include/swept1d.h."""
    c = (ctypes.c_double * 5)()
    _check(lib().swept_measure_latencies(c, _stream_ptr(stream)))
    names = ("dfma", "dadd_dfma", "shfl64", "lockstep_tier_2shfl_dadd_dfma", "smem_tier_1barrier_256thr")
    return dict(zip(names, (float(v) for v in c)))


def plan(problem: int, nx: int, nsteps: int, tile_width: int, *, dtype: int = F64, kernel: int = KERNEL_WAVE, chain: int = CHAIN_RING) -> list:
    """The launch list `swept_run` enqueues (swept_plan; host logic, no device needed): [(kind, W, offset, count), ...]."""
    buf = (_Launch * 64)()
    n = lib().swept_plan(int(problem), int(dtype), int(nx), int(nsteps), int(tile_width), int(kernel), int(chain), buf, 64)
    if n < 0:
        _check(int(n))
    return [(buf[i].kind, buf[i].tile_width, buf[i].offset, buf[i].count) for i in range(min(int(n), 64))]


def band_layout(ntiles: int, sm_count: int, warps_per_block: int) -> dict:
    """Grid of the streaming-band schedule (swept_band_layout; host logic, no device needed)."""
    lay = _BandLayout()
    _check(lib().swept_band_layout(int(ntiles), int(sm_count), int(warps_per_block), ctypes.byref(lay)))
    return {n: getattr(lay, n) for n, _ in _BandLayout._fields_}


def band_owner(layout: dict, band: int) -> tuple:
    """(block, warp, index in the warp's band list) that own `band` (swept_band_owner)."""
    lay = _BandLayout(**layout)
    b, w, i = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(lib().swept_band_owner(ctypes.byref(lay), int(band), ctypes.byref(b), ctypes.byref(w), ctypes.byref(i)))
    return b.value, w.value, i.value


def problem_info(problem: int) -> dict:
    """Stencil radius per sub-timestep, sub-timesteps per timestep and fields per point (swept_problem_info; no device needed)."""
    r, s, n = ctypes.c_int(), ctypes.c_int(), ctypes.c_int()
    _check(lib().swept_problem_info(int(problem), ctypes.byref(r), ctypes.byref(s), ctypes.byref(n)))
    return {"radius": r.value, "stages": s.value, "ncomp": n.value}


def steps_per_half_cycle(problem: int, tile_width: int) -> int:
    """L/S: full timesteps one half-cycle advances."""
    i = problem_info(problem)
    return tile_width // (2 * i["radius"] * i["stages"])
