"""`-m gpu`: the build that follows the PTX memory model to the letter, against the product build.

Two cross-CTA hand-offs of the pair kernels use plain remote mbarrier arrivals where the memory model asks for a
cluster-scope release (the slot release of the tile-index ring, and the ci4 pair kernel's relay "the
peer's stage is written"); the product keeps them because nothing is published through those arrivals that the arriving
thread has not already observed complete, and the release costs 6-8 % on cfg2.  This test compiles the library with
-DBFX_RING_ARRIVE=2 (every such arrival a `mbarrier.arrive.release.cluster`) into a temporary directory, loads it beside
the product library and requires identical bytes on the shapes that exercise those hand-offs -- repeatedly for the
shape that exposed the one real ordering bug of round 1 (the slot READ overtaken by the arrival, fixed in PrRing::get).
"""
import ctypes
import os
import subprocess

import pytest
import torch

import paper_1708_00720_b200 as bfx
from paper_1708_00720_b200 import _build

pytestmark = pytest.mark.gpu

# (ninputs, nchan, ntime, dtype, repeats)
SHAPES = [
    (512, 8, 600, 4, 1),        # ci4 pair kernel in place (relay + tile ring)
    (1152, 920, 130, 4, 6),     # ci4 pair kernel through the packed S1 ring: the shape of round 1's lost tiles
    (512, 6, 1024, 8, 1),       # ci8 stripe kernel in place
    (1152, 460, 130, 8, 3),     # ci8 stripe kernel through the S1 ring
    (192, 5, 1100, 8, 1),       # ci8 pair kernel through the S1 ring
]


@pytest.fixture(scope="module")
def conformant(tmp_path_factory):
    out = str(tmp_path_factory.mktemp("conformant") / "libbfxcorr_conformant.so")
    cmd = [_build._nvcc()] + _build.NVCC_FLAGS + ["-DBFX_RING_ARRIVE=2", "-I", _build.INCLUDE, "-o", out,
                                                 os.path.join(_build.CSRC, "bfxcorr.cu"), os.path.join(_build.CSRC, "bfbeamform.cu")]
    res = subprocess.run(cmd, capture_output=True, text=True)
    assert res.returncode == 0, res.stderr
    handle = ctypes.CDLL(out)
    for name, (restype, argtypes) in bfx.SIGNATURES.items():
        fn = getattr(handle, name)
        fn.restype = restype
        fn.argtypes = argtypes
    return handle


def _run(handle, shape, spans, stream):
    N, C, T, dt, _ = shape
    vp = ctypes.c_void_p
    out = torch.full((C, N * (N + 1) // 2, 2), 0x5A5A5A5A, dtype=torch.int32, device=spans[0].device)
    plan = vp()
    assert handle.bfXcorrCreate(ctypes.byref(plan), N, C, T, dt) == 0
    try:
        for s, x in enumerate(spans):
            assert handle.bfXcorrExecute(plan, vp(x.data_ptr()), vp(out.data_ptr()), 1 if s > 0 else 0, vp(stream)) == 0
        torch.cuda.synchronize()
    finally:
        assert handle.bfXcorrDestroy(plan) == 0
    return out


@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "N%d_C%d_T%d_ci%d_x%d" % s)
def test_conformant_build_gives_the_same_bytes(conformant, shape):
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    N, C, T, dt, repeats = shape
    g = torch.Generator(device=dev)
    g.manual_seed(N * 7 + C * 3 + T + dt)
    spans = [torch.randint(0, 256, (T * C * N * (1 if dt == 4 else 2),), dtype=torch.uint8, device=dev, generator=g) for _ in range(3)]
    want = _run(bfx.lib(), shape, spans, stream)
    for _ in range(repeats):
        assert torch.equal(_run(conformant, shape, spans, stream), want)
        assert torch.equal(_run(bfx.lib(), shape, spans, stream), want)
