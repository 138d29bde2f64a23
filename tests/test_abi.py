"""CPU-only checks of the boundary: the C-ABI library builds, loads and exports every symbol
include/spec.h declares; argument errors that need no GPU; no CPU fallback exists."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_1411_0436_b200 import build
    path = build.build()
    return ctypes.CDLL(path)


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "spec.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(spec_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol(lib):
    names = _declared_symbols()
    assert "spec_create" in names and "spec_process" in names and len(names) >= 10
    for n in names:
        assert hasattr(lib, n), f"libspec.so does not export {n}"


def test_binding_lists_the_same_symbols():
    from paper_1411_0436_b200 import spec as sp
    assert sorted(sp.SYMBOLS) == _declared_symbols()


def test_strerror_and_argument_errors_without_gpu(lib):
    lib.spec_strerror.restype = ctypes.c_char_p
    assert lib.spec_strerror(0) == b"ok"
    assert b"overrun" in lib.spec_strerror(-4)
    h = ctypes.c_void_p()
    mk = lib.spec_create
    mk.argtypes = [ctypes.POINTER(ctypes.c_void_p), ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                   ctypes.c_long, ctypes.c_int]
    assert mk(None, 1024, 8, 2, 0, 1, 1) == -1
    assert mk(ctypes.byref(h), 1000, 8, 2, 0, 1, 1) == -1      # not a power of two
    assert mk(ctypes.byref(h), 8, 8, 2, 0, 1, 1) == -1         # too small
    assert mk(ctypes.byref(h), 1 << 20, 8, 2, 0, 1, 1) == -1   # beyond the paper's 524288
    assert mk(ctypes.byref(h), 1024, 8, 3, 0, 1, 1) == -1      # npol
    assert mk(ctypes.byref(h), 1024, 0, 2, 0, 1, 1) == -1      # ntaps
    assert mk(ctypes.byref(h), 1024, 8, 2, 2, 1, 1) == -1      # mode
    assert mk(ctypes.byref(h), 1024, 8, 2, 0, 0, 1) == -1      # nacc
    assert mk(ctypes.byref(h), 1024, 8, 2, 0, 1, 7) == -1      # window
    assert not h.value


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    from paper_1411_0436_b200 import spec as sp
    with pytest.raises(sp.SpecError) as e:
        sp.Spec(1024, 8, 2, sp.MODE_PFB, 4)
    assert e.value.code == sp.ERR_CUDA


def test_product_path_does_not_touch_the_oracle():
    pkg = os.path.join(ROOT, "paper_1411_0436_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "spec_oracle" not in txt, f


def test_no_environment_switches_in_the_product_build():
    """The plan is a function of spec_create's arguments only: every getenv in csrc/ sits inside
    #ifdef SPEC_TUNING (a build flag the default build never sets) and nothing calls abort()."""
    csrc = os.path.join(ROOT, "paper_1411_0436_b200", "csrc")
    for f in sorted(os.listdir(csrc)):
        depth_tuning = 0
        stack = []
        for ln, line in enumerate(open(os.path.join(csrc, f)), 1):
            s = line.strip()
            if s.startswith("#if"):
                stack.append("SPEC_TUNING" in s and not s.startswith("#ifndef"))
            elif s.startswith("#endif") and stack:
                stack.pop()
            code = line.split("//")[0]
            if "getenv" in code:
                assert any(stack), f"{f}:{ln}: getenv outside #ifdef SPEC_TUNING"
            assert "abort(" not in code, f"{f}:{ln}: abort() in the library"
    from paper_1411_0436_b200 import build
    assert not any("SPEC_TUNING" in x for x in build.NVCC_FLAGS)


def test_build_is_reproducible_by_construction():
    """The library must come out byte-for-byte the same wherever it is built: no parallel split of the optimisation
    (a race between two code generations, profiles/r02_experiments.md row 24) and no absolute path on the command line."""
    from paper_1411_0436_b200 import build
    assert "-split-compile" not in build.NVCC_FLAGS
    assert "-lineinfo" in build.NVCC_FLAGS and "arch=compute_100a,code=sm_100a" in build.NVCC_FLAGS
    src = open(build.__file__).read()
    assert "os.path.relpath(p, CSRC)" in src
