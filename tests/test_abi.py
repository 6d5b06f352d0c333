"""CPU-side checks of the boundary: libwz.so builds, loads, and exports every symbol
include/wz.h declares; argument validation that needs no device.  No compute calls."""
import ctypes
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def wzmod():
    from paper_1005_3276_b200 import build, wz

    build.build()
    return wz


def test_header_symbols_exported(wzmod):
    hdr = open(os.path.join(ROOT, "include", "wz.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(wz_[a-z0-9_A-Z]+)\s*\(", hdr))
    assert declared, "no declarations parsed"
    lib = ctypes.CDLL(wzmod.LIB_PATH)
    for name in sorted(declared):
        assert hasattr(lib, name), name
    assert declared == set(wzmod.EXPORTS)


def test_status_strings_and_version(wzmod):
    L = wzmod.lib()
    assert L.wz_version().decode() == "0.1"
    texts = {L.wz_status_string(i).decode() for i in range(6)}
    assert len(texts) == 6 and "ok" in texts


def test_supported_lattices(wzmod):
    for dims in [(4, 4, 4, 4), (8, 8, 8, 8), (16, 16, 16, 16), (32, 32, 32, 32), (48, 24, 24, 24), (64, 64, 64, 64),
                 (32, 8, 8, 8), (32, 16, 16, 16), (64, 32, 32, 32)]:  # the last three: the paper's L^3 x T lattices
        assert wzmod.supported(dims, "c64") and wzmod.supported(dims, "c128"), dims
    assert not wzmod.supported((5, 4, 4, 4), "c128")   # T odd
    assert not wzmod.supported((10, 4, 4, 4), "c128")  # prime factor 5


def test_plan_create_argument_errors(wzmod):
    L = wzmod.lib()
    h = ctypes.c_void_p()
    assert L.wz_plan_create(ctypes.byref(h), 5, 4, 4, 4, 1, 1, None) == wzmod.WZ_EINVAL
    assert L.wz_plan_create(ctypes.byref(h), 4, 4, 4, 1, 1, 1, None) == wzmod.WZ_EINVAL
    assert L.wz_plan_create(ctypes.byref(h), 4, 4, 4, 4, 1, 0, None) == wzmod.WZ_EINVAL
    assert L.wz_plan_create(ctypes.byref(h), 4, 4, 4, 4, 7, 1, None) == wzmod.WZ_EINVAL
    assert L.wz_plan_create(ctypes.byref(h), 10, 4, 4, 4, 1, 1, None) == wzmod.WZ_EUNSUPPORTED
    assert L.wz_plan_create(None, 4, 4, 4, 4, 1, 1, None) == wzmod.WZ_EINVAL
    assert L.wz_plan_destroy(None) == wzmod.WZ_EINVAL


def test_no_cpu_fallback(wzmod):
    import torch

    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(wzmod.WZError):
        wzmod.Plan((4, 4, 4, 4), "c128", 1)
