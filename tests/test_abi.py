"""CPU-side checks of the C-ABI boundary (include/bfxcorr.h): the library builds, loads without a
GPU, exports every symbol the header declares, and fails loudly (no CPU fallback) when there is no
sm_100 device.  No compute calls are made here."""
import ctypes
import os
import re

import pytest

import paper_1708_00720_b200 as bfx

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADERS = [os.path.join(ROOT, "include", n) for n in sorted(os.listdir(os.path.join(ROOT, "include"))) if n.endswith(".h")]


def _declared_functions():
    names = set()
    for header in HEADERS:
        src = open(header).read()
        src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
        names.update(re.findall(r"\b(bf(?:Xcorr|Beamform)[A-Z]\w*)\s*\(", src))
    return sorted(names)


def test_header_declares_the_north_star_entry_points():
    names = _declared_functions()
    for must in ("bfXcorrCreate", "bfXcorrExecute", "bfXcorrDestroy", "bfBeamformCreate", "bfBeamformExecute"):
        assert must in names


def test_library_builds_and_exports_every_declared_symbol():
    lib = ctypes.CDLL(bfx.build())
    for name in _declared_functions():
        assert hasattr(lib, name), name


def test_binding_mirrors_the_header_one_to_one():
    assert sorted(bfx.SIGNATURES) == _declared_functions()
    for name in bfx.SIGNATURES:
        assert callable(getattr(bfx, name)), name


def test_status_strings():
    assert bfx.bfXcorrGetStatusString(0) == "BF_XCORR_OK"
    assert bfx.bfXcorrGetStatusString(6) == "BF_XCORR_UNSUPPORTED_DEVICE"
    assert bfx.bfXcorrGetStatusString(1234) == "BF_XCORR_UNKNOWN_STATUS"


def test_argument_errors_need_no_device():
    lib = bfx.lib()
    plan = ctypes.c_void_p()
    assert lib.bfXcorrCreate(None, 16, 4, 256, 8) == 1                       # INVALID_POINTER
    assert lib.bfXcorrCreate(ctypes.byref(plan), 0, 4, 256, 8) == 3          # INVALID_ARGUMENT
    assert lib.bfXcorrCreate(ctypes.byref(plan), 16, 4, 70000, 8) == 3       # ntime > 65535
    assert lib.bfXcorrCreate(ctypes.byref(plan), 16, 4, 256, 5) == 4         # INVALID_DTYPE
    assert lib.bfXcorrCreate(ctypes.byref(plan), 3, 1, 3, 8) == 5            # UNSUPPORTED_SHAPE (6-byte rows)
    assert lib.bfXcorrCreate(ctypes.byref(plan), 8, 1, 3, 4) == 5            # UNSUPPORTED_SHAPE (8-byte rows)
    assert lib.bfXcorrDestroy(None) == 2                                     # INVALID_HANDLE
    assert lib.bfXcorrExecute(None, None, None, 0, None) == 2
    assert lib.bfBeamformCreate(None, 16, 4, 256, 2, 8) == 1
    assert lib.bfBeamformCreate(ctypes.byref(plan), 16, 4, 256, 0, 8) == 3   # nbeam <= 0
    assert lib.bfBeamformCreate(ctypes.byref(plan), 16, 4, 256, 2, 5) == 4
    assert lib.bfBeamformCreate(ctypes.byref(plan), 16, 4, 256, 129, 8) == 5  # nbeam > 128
    assert lib.bfBeamformCreate(ctypes.byref(plan), 8, 1, 3, 1, 4) == 5      # 8-byte rows
    assert lib.bfBeamformExecute(None, None, None, None) == 2


def test_no_cpu_fallback_without_a_device():
    import torch
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    with pytest.raises(bfx.BfXcorrError) as e:
        bfx.bfXcorrCreate(16, 4, 256, 8)
    assert e.value.status == 6  # BF_XCORR_UNSUPPORTED_DEVICE


def test_product_does_not_import_the_oracle():
    pkg = os.path.join(ROOT, "paper_1708_00720_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt, f
                assert "xcorr_oracle" not in txt, f
