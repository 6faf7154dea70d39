"""`-m gpu` parity of the three-multiplication ci4 variant (bfXcorrSetAlgo(BF_XCORR_ALGO_TCGEN05_GAUSS3); SURVEY.md section
8(f) N3, xcorr_gauss4.cuh).  It computes the same visibilities as the default path, so it is held to the same bar: bit
for bit against the oracle on the whole ci4 suite -- ragged shapes, few and many inputs, the extreme code -8 - 8j (where
re + im reaches -16 and 8 (re + im) = -128 must still fit the int8 operand), accumulation laws -- and on full-size cfg2."""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1708_00720_b200 as bfx
from gpu_harness import run_spans
from helpers import pack, read_golden, tri_index
from xcorr_inputs import CONFIGS, generate_channel_slab, generate_span

pytestmark = pytest.mark.gpu
G3 = bfx.BF_XCORR_ALGO_TCGEN05_GAUSS3


def rand4(rng, T, C, N):
    return pack(4, rng.integers(-8, 8, size=(T, C, N)), rng.integers(-8, 8, size=(T, C, N)))


SHAPES = [(16, 3, 40), (64, 4, 129), (96, 2, 64), (128, 3, 31), (208, 2, 70), (256, 1, 128), (512, 1, 96), (144, 2, 1),
          (400, 3, 333), (1040, 1, 65)]


@pytest.mark.parametrize("shape", SHAPES, ids=lambda s: "n%dc%dt%d" % s)
def test_random_ci4_bit_exact(shape):
    N, C, T = shape
    x = rand4(np.random.default_rng(3000 + N + T), T, C, N)
    np.testing.assert_array_equal(run_spans([x], N, C, T, 4, G3), oracle.xcorr(x, N, C, T, 4))


@pytest.mark.parametrize("name", ["worked_example_n3.txt", "worked_example_n2.txt"])
def test_worked_examples_embedded(name):
    g = read_golden(name)
    T = 1 + max(t for t, _, _, _ in g["x"])
    N = 16
    re = np.zeros((T, 1, N), dtype=np.int64)
    im = np.zeros((T, 1, N), dtype=np.int64)
    for t, i, r, m in g["x"]:
        re[t, 0, i], im[t, 0, i] = r, m
    got = run_spans([pack(4, re, im)], N, 1, T, 4, G3)
    exp = np.zeros_like(got)
    n_small = 1 + max(i for _, i, _, _ in g["x"])
    k = 0
    for i in range(n_small):
        for j in range(i + 1):
            _, vr, vi = g["v"][k]
            exp[0, tri_index(i, j)] = (vr, vi)
            k += 1
    np.testing.assert_array_equal(got, exp)


def test_extreme_code_fits_the_operand():
    """Every sample -8 - 8j: the sum planes hold 8 (-8 + -8) = -128, the smallest int8; V = 2 * 64 * T real, 0 imaginary.
    And a span mixing -8 and +7 in every combination of parts (all four sign patterns of re +- im)."""
    N, C, T = 144, 2, 100
    re = np.full((T, C, N), -8, dtype=np.int64)
    got = run_spans([pack(4, re, re)], N, C, T, 4, G3)
    assert (got[..., 0] == 2 * 64 * T).all() and (got[..., 1] == 0).all()
    rng = np.random.default_rng(4)
    re = rng.choice([-8, 7], size=(T, C, N))
    im = rng.choice([-8, 7], size=(T, C, N))
    x = pack(4, re, im)
    np.testing.assert_array_equal(run_spans([x], N, C, T, 4, G3), oracle.xcorr(x, N, C, T, 4))


def test_accumulation_laws_and_wraparound():
    N, C, T = 192, 3, 70
    rng = np.random.default_rng(81)
    xs = [rand4(rng, T, C, N) for _ in range(3)]
    exp = oracle.xcorr(xs[0], N, C, T, 4)
    for x in xs[1:]:
        oracle.xcorr(x, N, C, T, 4, out=exp, accumulate=True)
    np.testing.assert_array_equal(run_spans(xs, N, C, T, 4, G3), exp)
    one = run_spans([np.concatenate(xs[:2], axis=0)], N, C, 2 * T, 4, G3)
    np.testing.assert_array_equal(one, run_spans(xs[:2], N, C, T, 4, G3))
    nb = N * (N + 1) // 2
    init = torch.full((C, nb, 2), 2**31 - 5, dtype=torch.int32)
    got = run_spans([xs[0]], N, C, T, 4, G3, first_accumulate=True, init=init)
    exp = init.numpy().copy()
    oracle.xcorr(xs[0], N, C, T, 4, out=exp, accumulate=True)
    np.testing.assert_array_equal(got, exp)


def test_longest_span_and_ci8_is_refused():
    N, C, T = 64, 2, 65535
    x = rand4(np.random.default_rng(6), T, C, N)
    np.testing.assert_array_equal(run_spans([x], N, C, T, 4, G3), oracle.xcorr(x, N, C, T, 4))
    plan = bfx.bfXcorrCreate(64, 2, 16, 8)
    try:
        with pytest.raises(bfx.BfXcorrError) as e:
            bfx.bfXcorrSetAlgo(plan, G3)
        assert e.value.status == 3
    finally:
        bfx.bfXcorrDestroy(plan)


def test_cfg2_full_size_whole_output():
    """BASELINE.json configs[1] as bench.py runs it (4 accumulated spans): the whole output against the default
    tensor-core path on the device, and 64 evenly spaced channels against the oracle."""
    cfg = CONFIGS["cfg2"]
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    outs = []
    for algo in (G3, bfx.BF_XCORR_ALGO_TCGEN05):
        plan = bfx.bfXcorrCreate(cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
        bfx.bfXcorrSetAlgo(plan, algo)
        out = torch.full((cfg.nchan, cfg.nbaselines, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
        for s in range(cfg.nspans):
            x = generate_span(cfg, s, device=dev)
            bfx.bfXcorrExecute(plan, x.data_ptr(), out.data_ptr(), s > 0, stream)
            torch.cuda.synchronize()
        bfx.bfXcorrDestroy(plan)
        outs.append(out)
    assert torch.equal(outs[0], outs[1])
    chans = sorted(set(int(round(k * (cfg.nchan - 1) / 63)) for k in range(64)))
    slabs = [generate_channel_slab(cfg, s, chans, device=dev).cpu().numpy() for s in range(cfg.nspans)]
    exp = oracle.xcorr(slabs[0], cfg.ninputs, len(chans), cfg.ntime, cfg.dtype)
    for sl in slabs[1:]:
        oracle.xcorr(sl, cfg.ninputs, len(chans), cfg.ntime, cfg.dtype, out=exp, accumulate=True)
    np.testing.assert_array_equal(outs[0][torch.tensor(chans, device=dev)].cpu().numpy(), exp)
