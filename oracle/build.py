"""Build the CPU oracle (plain C) into oracle/liboracle.so.  Test infrastructure only."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = [os.path.join(HERE, "swept_oracle.c")]
DEPS = SRC + [os.path.join(HERE, "schemes.inc"), os.path.join(HERE, "heat2d.inc")]
OUT = os.path.join(HERE, "liboracle.so")
# -ffp-contract=off: no implicit FMA, so the only fused operations are the explicit fma() calls of
# the canonical order.  No -march flags: the .so is built on one box and run on another.
CFLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c11"]


def needs_build() -> bool:
    if not os.path.exists(OUT):
        return True
    t = os.path.getmtime(OUT)
    return any(os.path.getmtime(d) > t for d in DEPS)


def build(force: bool = False) -> str:
    if force or needs_build():
        cmd = ["gcc", *CFLAGS, "-o", OUT, *SRC, "-lm"]
        subprocess.run(cmd, check=True, cwd=HERE)
    return OUT


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
