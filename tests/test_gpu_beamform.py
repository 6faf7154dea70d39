"""`-m gpu`: the beamformer kernel (include/bfbeamform.h) against oracle.beamform, bit for bit
(exact integer arithmetic), through the C ABI."""
import numpy as np
import pytest
import torch

import oracle
import paper_1708_00720_b200 as bfx
from xcorr_inputs import CONFIGS, generate_channel_slab, generate_span, generate_weights

pytestmark = pytest.mark.gpu
DEV = "cuda:0"


def run_beamform(x, w, N, C, T, K, dtype, poison=True):
    plan = bfx.bfBeamformCreate(N, C, T, K, dtype)
    try:
        xd = torch.as_tensor(np.ascontiguousarray(x)).to(DEV).view(torch.uint8).reshape(-1)
        wd = torch.as_tensor(np.ascontiguousarray(w)).to(DEV).view(torch.uint8).reshape(-1)
        assert xd.numel() == bfx.bfBeamformGetInputBytes(plan)
        assert wd.numel() == bfx.bfBeamformGetWeightBytes(plan)
        assert bfx.bfBeamformGetOutputBytes(plan) == T * C * K * 8
        out = torch.empty((T, C, K, 2), dtype=torch.int32, device=DEV)
        if poison:
            out.fill_(0x5A5A5A5A)
        stream = torch.cuda.current_stream().cuda_stream
        bfx.bfBeamformSetWeights(plan, wd.data_ptr(), stream)
        bfx.bfBeamformExecute(plan, xd.data_ptr(), out.data_ptr(), stream)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        bfx.bfBeamformDestroy(plan)


def _random_case(rng, N, C, T, K, dtype, extreme=False):
    x = rng.integers(0, 256, size=(T, C, N * (1 if dtype == 4 else 2)), dtype=np.uint8)   # every code, -8 / -128 too
    wr = rng.integers(-128, 128, size=(C, K, N))
    wi = rng.integers(-128, 128, size=(C, K, N))   # the whole int8 range for both parts (reading B4)
    if extreme:
        wr[:], wi[:] = -128, -128 if extreme == "neg" else 127
        x[:] = 0x88 if dtype == 4 else 0x80
    w = np.stack((wr & 0xFF, wi & 0xFF), axis=-1).astype(np.uint8).reshape(C, K, 2 * N)
    return x, w


SHAPES = [
    # N, C, T, K
    (16, 4, 256, 1),      # cfg1 shape, one beam (odd: 8-byte stores)
    (16, 3, 130, 8),      # ragged sample block
    (64, 5, 200, 16),
    (80, 7, 129, 3),      # rows that are no multiple of 128 bytes, odd beam count
    (512, 3, 300, 32),    # station shape: several K stages, ragged tail
    (528, 2, 128, 5),
    (128, 2, 257, 127),   # maximum beam count (2 * 127 + 2 = 256 accumulator columns)
    (256, 170, 64, 4),    # more units than SMs with a single short sample block (ci8: two-piece span boxes, 5-d map)
    (512, 3, 296, 32),    # ci8: two-piece span boxes, four K stages, a sample count that is a multiple of 8 but not of 128
    (256, 6, 1000, 16),   # the same with eight sample blocks
    (1024, 2, 136, 40),   # wider weight tiles beside the two-piece boxes
    (384, 4, 264, 9),     # rows of three pieces: no whole number of two-piece boxes, so the 3-d map
    (512, 3, 264, 127),   # ci8: the largest weight tiles -- only two two-piece stages fit
]


@pytest.mark.parametrize("dtype", [4, 8])
@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "n%dc%dt%dk%d" % s)
def test_matches_oracle(shape, dtype):
    N, C, T, K = shape
    if dtype == 4 and N % 16:
        pytest.skip("ci4 rows must be multiples of 16 bytes")
    rng = np.random.default_rng(hash(shape) % (2 ** 31) + dtype)
    x, w = _random_case(rng, N, C, T, K, dtype)
    got = run_beamform(x, w, N, C, T, K, dtype)
    exp = oracle.beamform(x, w, N, C, T, K, dtype)
    np.testing.assert_array_equal(got, exp)


@pytest.mark.parametrize("extreme", ["neg", "mixed"])
@pytest.mark.parametrize("dtype", [4, 8])
def test_extreme_codes(dtype, extreme):
    """Every sample at the most negative code and every weight -128 - 128j ("neg") or -128 + 127j ("mixed")."""
    N, C, T, K = 512, 2, 140, 8
    x, w = _random_case(np.random.default_rng(0), N, C, T, K, dtype, extreme=extreme)
    np.testing.assert_array_equal(run_beamform(x, w, N, C, T, K, dtype), oracle.beamform(x, w, N, C, T, K, dtype))


def test_no_weights_and_limits():
    """Execute without weights is refused; every weight code (-128 in either part) is accepted; 128 beams are not."""
    N, C, T, K = 16, 1, 8, 1
    plan = bfx.bfBeamformCreate(N, C, T, K, 8)
    try:
        w = torch.zeros(C * K * N * 2, dtype=torch.uint8, device=DEV)
        x = torch.zeros(T * C * N * 2, dtype=torch.uint8, device=DEV)
        out = torch.zeros((T, C, K, 2), dtype=torch.int32, device=DEV)
        with pytest.raises(bfx.BfXcorrError) as e:     # no weights yet
            bfx.bfBeamformExecute(plan, x.data_ptr(), out.data_ptr(), 0)
        assert e.value.status == 3
        w[4] = 0x80
        w[5] = 0x80                                    # -128 - 128j
        bfx.bfBeamformSetWeights(plan, w.data_ptr(), 0)
        bfx.bfBeamformExecute(plan, x.data_ptr(), out.data_ptr(), 0)
        torch.cuda.synchronize()
    finally:
        bfx.bfBeamformDestroy(plan)
    with pytest.raises(bfx.BfXcorrError) as e:
        bfx.bfBeamformCreate(N, C, T, 128, 8)
    assert e.value.status == 5


@pytest.mark.parametrize("name,nbeam", [("cfg2", 32), ("cfg3", 16), ("cfg4", 16), ("cfg5", 8), ("cfg2", 127), ("cfg2", 7)])
def test_full_config_sampled_channels(name, nbeam):
    """BASELINE.json's station-shaped spans at full size, in the launch configuration bench.py times: sampled
    channels (all samples, all beams) against the oracle."""
    cfg = CONFIGS[name]
    N, C, T = cfg.ninputs, cfg.nchan, cfg.ntime
    x = generate_span(cfg, 0, device=DEV)
    w = generate_weights(cfg.seed, C, nbeam, N, device=DEV)
    plan = bfx.bfBeamformCreate(N, C, T, nbeam, cfg.dtype)
    try:
        out = torch.full((T, C, nbeam, 2), 0x5A5A5A5A, dtype=torch.int32, device=DEV)
        stream = torch.cuda.current_stream().cuda_stream
        bfx.bfBeamformSetWeights(plan, w.data_ptr(), stream)
        bfx.bfBeamformExecute(plan, x.data_ptr(), out.data_ptr(), stream)
        torch.cuda.synchronize()
        chans = sorted({0, 1, C // 2 - 1, C // 2, C - 2, C - 1, 147, 148, (C * 3) // 7})
        xs = generate_channel_slab(cfg, 0, chans).numpy()
        ws = generate_weights(cfg.seed, C, nbeam, N, channels=chans).numpy()
        exp = oracle.beamform(xs, ws, N, len(chans), T, nbeam, cfg.dtype)
        got = out[:, chans].cpu().numpy()
        np.testing.assert_array_equal(got, exp)
        # nothing left unwritten anywhere (the poison value is not reachable: |b| < 2^30)
        assert int((out == 0x5A5A5A5A).sum().item()) == 0
    finally:
        bfx.bfBeamformDestroy(plan)
