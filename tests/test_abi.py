"""CPU-only checks of the boundary: libwl.so builds for sm_100a, loads, and exports every symbol include/wl.h declares;
argument validation that needs no GPU.  No compute calls here."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    from paper_2304_08159_b200 import build, binding
    build.build_cuda()
    return binding.load()


def test_every_declared_symbol_is_exported(lib):
    from paper_2304_08159_b200 import binding
    hdr = open(os.path.join(ROOT, "include", "wl.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wl_[a-z_0-9]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    assert declared == set(binding.SIGNATURES), declared ^ set(binding.SIGNATURES)
    for name in declared:
        assert getattr(lib, name) is not None


def test_library_is_sm100a_and_has_no_oracle_code(lib):
    import subprocess
    from paper_2304_08159_b200 import binding
    out = subprocess.run(["cuobjdump", "-lelf", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "sm_100a" in out
    syms = subprocess.run(["nm", "-D", "--defined-only", binding.LIB_PATH], capture_output=True, text=True).stdout
    assert "orc_" not in syms  # the oracle shares nothing with the product


def test_create_rejects_bad_arguments_without_a_gpu(lib):
    from paper_2304_08159_b200 import binding as wl
    out = ctypes.c_void_p()
    d2 = (ctypes.c_int64 * 3)(8, 8, 8)
    assert lib.wl_create(1, d2, 0, ctypes.byref(out)) == wl.WL_EDIMS
    assert lib.wl_create(4, d2, 0, ctypes.byref(out)) == wl.WL_EDIMS
    d3 = (ctypes.c_int64 * 3)(8, 3, 8)
    assert lib.wl_create(3, d3, 0, ctypes.byref(out)) == wl.WL_EDIMS
    assert lib.wl_create(3, d2, 7, ctypes.byref(out)) == wl.WL_EINVAL
    assert lib.wl_create(3, None, 0, ctypes.byref(out)) == wl.WL_EINVAL
    assert not out.value
    assert b"wl_create" in lib.wl_last_error(None)
    # null contexts are rejected, never dereferenced
    assert lib.wl_set_coeff(None, None) == wl.WL_EINVAL
    assert lib.wl_num_levels(None) == wl.WL_EINVAL
    lib.wl_destroy(None)


def test_no_cpu_fallback():
    """Without a GPU the product path must fail loudly (no oracle, no CPU path behind the binding)."""
    import torch
    from paper_2304_08159_b200 import binding as wl
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises((RuntimeError, wl.WlError)):
        wl.Projector((8, 8), "float32")
    with pytest.raises(wl.WlError) as ei:
        wl.wl_create((8, 8), "float32")
    assert ei.value.code == wl.WL_ECUDA
    src = open(os.path.join(ROOT, "paper_2304_08159_b200", "binding.py")).read()
    assert "import oracle" not in src and "from oracle" not in src
