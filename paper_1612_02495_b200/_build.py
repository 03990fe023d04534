"""Build libswept1d.so (hand-written CUDA for sm_100a) in-tree with nvcc.  No JIT cache, no torch headers:
the library is a plain C ABI (include/swept1d.h)."""
from __future__ import annotations

import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
OUT = os.path.join(HERE, "libswept1d.so")
SOURCES = ["api.cu", "naive.cu", "swept_smem.cu", "swept_wave.cu", "swept_wave_heat.cu", "swept_wave_ks.cu", "swept_wave_euler.cu",
           "swept_band_heat.cu", "swept_band_ks.cu", "swept_band_euler.cu", "swept_ring_heat.cu", "swept_ring_ks.cu", "swept_ring_euler.cu", "heat2d.cu", "alu_peak.cu"]
HEADERS = ["internal.h", "stencils.cuh", "swept_wave.cuh", "swept_band.cuh", "swept_ring.cuh", os.path.join("..", "..", "include", "swept1d.h"), os.path.join("..", "..", "include", "swept2d.h")]
# -fmad=false: no implicit FMA contraction -- the only fused operations are the explicit fma() calls of the
# canonical evaluation order, so classic, swept and the CPU oracle round identically.
# Default -prec-div=true -prec-sqrt=true -ftz=false are kept (IEEE division and square root, denormals).
NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo", "-fmad=false",
    "-Xcompiler", "-fPIC,-ffp-contract=off",
]
# The flags are fixed: no environment variable reaches the compiler, so a product build cannot be steered into another kernel.
# Objects built with other flags (an older checkout, a hand-run nvcc) are rebuilt: the flags are stamped beside them.
STAMP = os.path.join(OBJ, "flags.stamp")


def _nvcc() -> str:
    for c in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if c and (os.path.isabs(c) and os.path.exists(c) or not os.path.isabs(c)):
            return c
    return "nvcc"


def _stale(target: str, deps) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    hdrs = [os.path.normpath(os.path.join(CSRC, h)) for h in HEADERS] + [os.path.abspath(__file__)]
    nvcc = _nvcc()
    stamp = " ".join([nvcc, *NVCC_FLAGS])
    if not os.path.exists(STAMP) or open(STAMP).read() != stamp:
        force = True
    jobs = []
    objs = []
    for src in SOURCES:
        s = os.path.join(CSRC, src)
        o = os.path.join(OBJ, src.replace(".cu", ".o"))
        objs.append(o)
        if force or _stale(o, [s] + hdrs):
            jobs.append([nvcc, *NVCC_FLAGS, "-c", s, "-o", o])

    def run(cmd):
        if verbose:
            print(" ".join(cmd), file=sys.stderr)
        r = subprocess.run(cmd, capture_output=True, text=True)
        if r.returncode != 0:
            raise RuntimeError(f"nvcc failed: {' '.join(cmd)}\n{r.stdout}\n{r.stderr}")

    if jobs:
        with ThreadPoolExecutor(max_workers=min(8, len(jobs))) as ex:
            list(ex.map(run, jobs))
    if force or jobs or _stale(OUT, objs):
        run([nvcc, "-shared", "-o", OUT, *objs, "-gencode", "arch=compute_100a,code=sm_100a"])
    with open(STAMP, "w") as f:
        f.write(stamp)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose=True))
