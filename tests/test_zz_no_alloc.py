"""`-m gpu`: bfXcorrExecuteNoAlloc (include/bfxcorr.h) -- one span with no plan and no device allocation, every kernel's
scratch in the library's static device array -- against the existing path (bfXcorrCreate / bfXcorrExecute), bit for bit
(the path is integer-only: the suite's tolerance is equality), on two calls in a row that accumulate into one buffer.

Collected last on purpose (the name sorts after every other test file): the suite runs with pytest -x.
Passes alone in a fresh process (the first call does the device's one-time set-up) and after the other tests.
"""
import pytest
import torch

import paper_1708_00720_b200 as bfx

pytestmark = pytest.mark.gpu

# (ninputs, nchan, ntime, dtype): which kernel, and whether its scratch is more than the scheduler words
SHAPES = [
    (16, 4, 256, 8),        # BASELINE.json configs[0]: few-input kernel, span read in place
    (64, 40, 300, 4),       # few-input kernel, ci4
    (512, 6, 1024, 8),      # stripe kernel in place (register-direct epilogue, then the L2-reduce epilogue)
    (512, 5, 520, 4),       # ci4 pair kernel in place
    (192, 5, 1100, 8),      # more than 1024 samples: pair kernel through the S1 ring (ring + ready / done flags)
    (1152, 460, 130, 8),    # 9 row blocks, samples 1.06 MB apart: stripe kernel through the S1 ring
    (1152, 920, 130, 4),    # the same for ci4: pair4 kernel through the packed S1 ring
]


def _spans(shape, dev, n=2):
    N, C, T, dt = shape
    g = torch.Generator(device=dev)
    g.manual_seed(1000 * N + 10 * C + T + dt)
    return [torch.randint(0, 256, (T * C * N * (1 if dt == 4 else 2),), dtype=torch.uint8, device=dev, generator=g) for _ in range(n)]


def _plan_path(shape, spans, dev, stream):
    N, C, T, dt = shape
    out = torch.full((C, N * (N + 1) // 2, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
    plan = bfx.bfXcorrCreate(N, C, T, dt)
    try:
        for s, x in enumerate(spans):
            bfx.bfXcorrExecute(plan, x.data_ptr(), out.data_ptr(), s > 0, stream)
        torch.cuda.synchronize()
    finally:
        bfx.bfXcorrDestroy(plan)
    return out


def _no_alloc_path(shape, spans, dev, stream):
    N, C, T, dt = shape
    out = torch.full((C, N * (N + 1) // 2, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
    for s, x in enumerate(spans):
        bfx.bfXcorrExecuteNoAlloc(x.data_ptr(), out.data_ptr(), N, C, T, dt, s > 0, stream)
    torch.cuda.synchronize()
    return out


@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "N%d_C%d_T%d_ci%d" % s)
def test_two_calls_in_a_row_match_the_plan_path(shape):
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    spans = _spans(shape, dev)
    want = _plan_path(shape, spans, dev, stream)
    got = _no_alloc_path(shape, spans, dev, stream)
    assert torch.equal(got, want)
    # and once more: the static array now holds this shape's own leftovers
    again = _no_alloc_path(shape, spans, dev, stream)
    assert torch.equal(again, want)


def test_shapes_interleaved_on_one_stream_and_nothing_allocated():
    """The array is shared by every call and keeps the last call's contents: ring shapes and in-place shapes in turn, each
    checked against the plan path; over all of these calls the device's free memory does not move."""
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    order = [SHAPES[5], SHAPES[0], SHAPES[4], SHAPES[6], SHAPES[2], SHAPES[5], SHAPES[3], SHAPES[4]]
    spans = {sh: _spans(sh, dev) for sh in set(order)}
    want = {sh: _plan_path(sh, spans[sh], dev, stream) for sh in set(order)}
    outs = [torch.empty_like(want[sh]) for sh in order]
    # the device's one-time set-up (no allocation either, but module loading may move the numbers) happens here
    bfx.bfXcorrExecuteNoAlloc(spans[order[0]][0].data_ptr(), outs[0].data_ptr(), *order[0], False, stream)
    torch.cuda.synchronize()
    free_before, _ = torch.cuda.mem_get_info()
    for sh, out in zip(order, outs):
        for s, x in enumerate(spans[sh]):
            bfx.bfXcorrExecuteNoAlloc(x.data_ptr(), out.data_ptr(), *sh, s > 0, stream)
    torch.cuda.synchronize()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after == free_before
    for sh, out in zip(order, outs):
        assert torch.equal(out, want[sh]), sh


def test_limits_and_argument_errors():
    dev = torch.device("cuda:0")
    x = torch.zeros(1024, dtype=torch.uint8, device=dev)
    out = torch.zeros(1024, dtype=torch.int32, device=dev)

    def status(*args):
        with pytest.raises(bfx.BfXcorrError) as e:
            bfx.bfXcorrExecuteNoAlloc(*args)
        return e.value.status

    # 8192 inputs x 4096 samples of ci8: one ring slab is 64 MiB, the smallest ring is 6 of them
    assert status(x.data_ptr(), out.data_ptr(), 8192, 8, 4096, 8, False, 0) == bfx.BF_XCORR_SCRATCH_LIMIT
    assert "SCRATCH_LIMIT" in bfx.bfXcorrGetStatusString(bfx.BF_XCORR_SCRATCH_LIMIT)
    # a ring shape with more channels than the flag area holds
    assert status(x.data_ptr(), out.data_ptr(), 192, 65537, 1100, 8, False, 0) == bfx.BF_XCORR_SCRATCH_LIMIT
    # the same number of channels read in place is no limit case (rejected here only for the NULL pointer)
    assert status(0, out.data_ptr(), 64, 65537, 8, 4, False, 0) == 1          # BF_XCORR_INVALID_POINTER
    assert status(x.data_ptr() + 4, out.data_ptr(), 16, 4, 8, 8, False, 0) == 1  # misaligned
    assert status(x.data_ptr(), out.data_ptr(), 0, 4, 8, 8, False, 0) == 3      # BF_XCORR_INVALID_ARGUMENT
    assert status(x.data_ptr(), out.data_ptr(), 16, 4, 8, 5, False, 0) == 4     # BF_XCORR_INVALID_DTYPE
    assert status(x.data_ptr(), out.data_ptr(), 12, 4, 8, 4, False, 0) == 5     # BF_XCORR_UNSUPPORTED_SHAPE (row not 16-byte)
    # nothing above launched anything or disturbed the device
    torch.cuda.synchronize()
    assert int(out.abs().sum()) == 0


def test_full_size_config_through_the_static_ring():
    """BASELINE.json configs[3] (2048 inputs, 1024 channels): the one config that uses the S1 ring -- 16 slabs of 4 MiB, the
    whole 64 MiB -- against the plan path, whole output."""
    from xcorr_inputs import CONFIGS, generate_span

    cfg = CONFIGS["cfg4"]
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info()
    if free < 2 * cfg.out_bytes + cfg.span_bytes + (4 << 30):
        pytest.skip("needs %.1f GB of device memory" % ((2 * cfg.out_bytes + cfg.span_bytes) / 1e9))
    stream = torch.cuda.current_stream().cuda_stream
    x = generate_span(cfg, 0, device=dev)
    shape = (cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
    want = _plan_path(shape, [x], dev, stream)
    got = _no_alloc_path(shape, [x], dev, stream)
    assert torch.equal(got, want)
