"""`-m gpu`: bfXcorrDump (integration dump) against the oracle, bit for bit (float32 results of a
fixed IEEE sequence: int32 -> float32 round-to-nearest-even, one float32 multiply)."""
import numpy as np
import pytest
import torch

import oracle
import paper_1708_00720_b200 as bfx

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("shape", [(16, 3), (24, 1), (192, 5), (520, 2)], ids=lambda s: "n%dc%d" % s)
@pytest.mark.parametrize("zero", [False, True])
def test_dump_matches_oracle(shape, zero):
    N, C = shape
    nb = N * (N + 1) // 2
    rng = np.random.default_rng(N + C)
    acc = rng.integers(-2 ** 31, 2 ** 31, size=(C, nb, 2), dtype=np.int64).astype(np.int32)
    acc.reshape(-1)[:6] = [0, 2 ** 24 + 1, 2 ** 24 + 3, -(2 ** 31), 2 ** 31 - 1, -1]   # ties and extremes
    dev = torch.device("cuda:0")
    plan = bfx.bfXcorrCreate(N, C, 64, 8)
    try:
        for scale in (1.0, 1.0 / 4096, 2.5e-4):
            a = torch.from_numpy(acc.copy()).to(dev)
            o = torch.full((C, nb, 2), float("nan"), dtype=torch.float32, device=dev)
            bfx.bfXcorrDump(plan, a.data_ptr(), o.data_ptr(), scale, zero, torch.cuda.current_stream().cuda_stream)
            assert bfx.bfXcorrGetLaunchCount(plan) == 1
            torch.cuda.synchronize()
            ref_acc = acc.copy()
            exp = oracle.dump(ref_acc, scale, zero_acc=zero)
            np.testing.assert_array_equal(o.cpu().numpy().view(np.uint32), exp.view(np.uint32))
            np.testing.assert_array_equal(a.cpu().numpy(), ref_acc)
    finally:
        bfx.bfXcorrDestroy(plan)


def test_dump_after_integration_then_next_integration_accumulates_from_zero():
    """Two integrations of two spans each through one buffer: dump-and-clear between them."""
    N, C, T = 136, 3, 90
    rng = np.random.default_rng(8)
    spans = [rng.integers(0, 256, size=(T, C, 2 * N), dtype=np.uint8) for _ in range(4)]
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    nb = N * (N + 1) // 2
    plan = bfx.bfXcorrCreate(N, C, T, 8)
    try:
        acc = torch.zeros((C, nb, 2), dtype=torch.int32, device=dev)
        outs = []
        for k, x in enumerate(spans):
            xd = torch.from_numpy(x).to(dev)
            bfx.bfXcorrExecute(plan, xd.data_ptr(), acc.data_ptr(), True, stream)   # always accumulate: buffer starts cleared
            if k % 2 == 1:
                o = torch.empty((C, nb, 2), dtype=torch.float32, device=dev)
                bfx.bfXcorrDump(plan, acc.data_ptr(), o.data_ptr(), 0.5, True, stream)
                torch.cuda.synchronize()
                outs.append(o.cpu().numpy())
        for k in range(2):
            v = oracle.xcorr(spans[2 * k], N, C, T, 8)
            oracle.xcorr(spans[2 * k + 1], N, C, T, 8, out=v, accumulate=True)
            np.testing.assert_array_equal(outs[k], oracle.dump(v, 0.5))
        assert int(acc.abs().max()) == 0
    finally:
        bfx.bfXcorrDestroy(plan)


def test_dump_full_size_cfg3_buffer_matches_float32_cast():
    """At BASELINE.json configs[2]'s buffer size (3.2 GB): every component equals the IEEE float32 conversion, checked
    on the device against torch's int32 -> float32 cast and multiply (same rounding rules as the oracle's C)."""
    from xcorr_inputs import CONFIGS
    cfg = CONFIGS["cfg3"]
    dev = torch.device("cuda:0")
    if torch.cuda.mem_get_info()[0] < 4 * cfg.out_bytes:
        pytest.skip("not enough device memory")
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    acc = torch.randint(-2 ** 31, 2 ** 31 - 1, (cfg.nchan, cfg.nbaselines, 2), dtype=torch.int32, device=dev, generator=g)
    out = torch.empty(acc.shape, dtype=torch.float32, device=dev)
    plan = bfx.bfXcorrCreate(cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
    try:
        bfx.bfXcorrDump(plan, acc.data_ptr(), out.data_ptr(), 1.0 / 2048, False, torch.cuda.current_stream().cuda_stream)
        torch.cuda.synchronize()
    finally:
        bfx.bfXcorrDestroy(plan)
    step = cfg.nchan // 8
    for c0 in range(0, cfg.nchan, step):
        exp = acc[c0:c0 + step].to(torch.float32) * (1.0 / 2048)
        assert torch.equal(out[c0:c0 + step], exp)


@pytest.mark.parametrize("shape", [(16, 3), (24, 1), (40, 70), (192, 5), (520, 2), (1040, 1)], ids=lambda s: "n%dc%d" % s)
@pytest.mark.parametrize("zero", [False, True])
def test_dump_matrix_matches_oracle(shape, zero):
    """bfXcorrDumpMatrix (reorder to the full Hermitian matrix): float32 bit patterns against the oracle, every element
    written (the output starts as NaN), the accumulator cleared or untouched."""
    N, C = shape
    nb = N * (N + 1) // 2
    rng = np.random.default_rng(7 * N + C)
    acc = rng.integers(-2 ** 31, 2 ** 31, size=(C, nb, 2), dtype=np.int64).astype(np.int32)
    acc.reshape(-1)[:6] = [0, 2 ** 24 + 1, 2 ** 24 + 3, -(2 ** 31), 2 ** 31 - 1, -1]
    dev = torch.device("cuda:0")
    plan = bfx.bfXcorrCreate(N, C, 64, 8)
    try:
        for scale in (1.0, 2.5e-4):
            a = torch.from_numpy(acc.copy()).to(dev)
            o = torch.full((C, N, N, 2), float("nan"), dtype=torch.float32, device=dev)
            bfx.bfXcorrDumpMatrix(plan, a.data_ptr(), o.data_ptr(), scale, zero, torch.cuda.current_stream().cuda_stream)
            assert bfx.bfXcorrGetLaunchCount(plan) == 1
            torch.cuda.synchronize()
            ref_acc = acc.copy()
            exp = oracle.dump_matrix(ref_acc, N, scale, zero_acc=zero)
            np.testing.assert_array_equal(o.cpu().numpy().view(np.uint32), exp.view(np.uint32))
            np.testing.assert_array_equal(a.cpu().numpy(), ref_acc)
    finally:
        bfx.bfXcorrDestroy(plan)


def test_dump_matrix_full_size_cfg3_is_hermitian_and_matches_the_packed_dump():
    """cfg3's 3.2 GB accumulator -> 6.4 GB of matrices: the lower triangle equals bfXcorrDump's output, the upper is its
    conjugate (properties that hold at any size), and sampled channels equal the oracle bit for bit."""
    N, C = 512, 3072
    nb = N * (N + 1) // 2
    dev = torch.device("cuda:0")
    if torch.cuda.mem_get_info()[0] < 16 * 2 ** 30:
        pytest.skip("needs 16 GiB of device memory")
    g = torch.Generator(device=dev)
    g.manual_seed(5)
    acc = torch.randint(-2 ** 31, 2 ** 31, (C, nb, 2), dtype=torch.int64, device=dev, generator=g).to(torch.int32)
    d = torch.arange(N, device=dev)
    acc[:, d * (d + 1) // 2 + d, 1] = 0        # autocorrelations are real, as in any accumulator the X-engine produced
    flat = torch.empty((C, nb, 2), dtype=torch.float32, device=dev)
    mat = torch.full((C, N, N, 2), float("nan"), dtype=torch.float32, device=dev)
    plan = bfx.bfXcorrCreate(N, C, 1024, 8)
    try:
        s = torch.cuda.current_stream().cuda_stream
        bfx.bfXcorrDump(plan, acc.data_ptr(), flat.data_ptr(), 0.125, False, s)
        bfx.bfXcorrDumpMatrix(plan, acc.data_ptr(), mat.data_ptr(), 0.125, False, s)
        torch.cuda.synchronize()
    finally:
        bfx.bfXcorrDestroy(plan)
    ii, jj = torch.tril_indices(N, N, device=dev)
    for c0 in range(0, C, 256):
        m = mat[c0:c0 + 256]
        assert torch.equal(m[:, ii, jj], flat[c0:c0 + 256])
        assert torch.equal(m[..., 0], m[..., 0].transpose(1, 2))
        assert torch.equal(m[..., 1], -m[..., 1].transpose(1, 2))
    for c in (0, 1777, C - 1):
        exp = oracle.dump_matrix(acc[c:c + 1].cpu().numpy().copy(), N, 0.125)
        np.testing.assert_array_equal(mat[c:c + 1].cpu().numpy().view(np.uint32), exp.view(np.uint32))
