"""The C-ABI library builds, loads and exports every symbol include/*.h declares; no compute calls (no GPU)."""
import ctypes
import os
import re

import pytest

import paper_1612_02495_b200 as sw

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADERS = [os.path.join(ROOT, "include", "swept1d.h"), os.path.join(ROOT, "include", "swept2d.h")]


def _declared_functions():
    src = "\n".join(open(h).read() for h in HEADERS)
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"^\s*(?:const\s+char\s*\*|int64_t|int)\s*\**\s*(\w+)\s*\(", src, flags=re.M)
    return sorted(set(names))


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for must in ("swept_create", "swept_run", "naive_run", "swept_tune", "swept_destroy", "swept_last_error"):
        assert must in names


def test_library_exports_every_declared_symbol():
    lib = sw.lib()
    for name in _declared_functions():
        assert hasattr(lib, name), f"libswept1d.so does not export {name}"
    assert sorted(sw.SYMBOLS) == _declared_functions()


def test_library_is_plain_c_abi_without_torch_or_oracle():
    """The product library links neither torch nor the oracle."""
    import subprocess
    out = subprocess.run(["ldd", sw.LIB_PATH], capture_output=True, text=True).stdout
    assert "torch" not in out and "oracle" not in out
    # and no source file of the product path mentions the oracle package
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_1612_02495_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "liboracle" not in txt and "from oracle" not in txt, f


def test_version_and_error_strings():
    assert "sm_100a" in sw.version()
    assert isinstance(sw.lib().swept_last_error(), bytes)


def test_argument_validation_needs_no_gpu():
    lib = sw.lib()
    h = ctypes.c_void_p()
    p = sw._Params(sw.F64, 1.0, 1.4, 0)
    assert lib.swept_create(None, sw.HEAT, 1024, 1e-3, 1e-7, ctypes.byref(p)) == sw.EINVAL
    assert lib.swept_create(ctypes.byref(h), 7, 1024, 1e-3, 1e-7, ctypes.byref(p)) == sw.EINVAL
    assert lib.swept_create(ctypes.byref(h), sw.HEAT, 1000, 1e-3, 1e-7, ctypes.byref(p)) == sw.EINVAL   # not a power of two
    assert b"power of two" in lib.swept_last_error()
    assert lib.swept_create(ctypes.byref(h), sw.HEAT, 4, 1e-3, 1e-7, ctypes.byref(p)) == sw.EINVAL
    assert lib.swept_create(ctypes.byref(h), sw.HEAT, 1024, float("nan"), 1e-7, ctypes.byref(p)) == sw.EINVAL
    assert lib.swept_create(ctypes.byref(h), sw.HEAT, 1024, 1e-3, -1.0, ctypes.byref(p)) == sw.EINVAL
    bad = sw._Params(5, 1.0, 1.4, 0)
    assert lib.swept_create(ctypes.byref(h), sw.HEAT, 1024, 1e-3, 1e-7, ctypes.byref(bad)) == sw.EINVAL
    assert lib.swept_run(None, None, 1, 0, None) == sw.EINVAL
    assert lib.naive_run(None, None, 1, None) == sw.EINVAL
    assert lib.swept_destroy(None) == sw.EINVAL
    assert lib.swept_measure_alu_peak(9, None, None, None) == sw.EINVAL


def test_no_cpu_fallback_without_a_device():
    """On a box without a GPU, creating a solver must fail loudly with ECUDA -- never compute on the CPU."""
    try:
        import torch
        has = torch.cuda.is_available()
    except Exception:
        has = False
    if has:
        pytest.skip("a CUDA device is present")
    with pytest.raises(sw.SweptError) as ei:
        sw.Solver("heat", 1024, 1.0 / 1024, 0.25 / 1024 ** 2)
    assert ei.value.code == sw.ECUDA
