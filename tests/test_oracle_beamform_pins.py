"""Pins of oracle.beamform against things other than itself.

Each test fixes the oracle to a fact that a plausible slip (a conjugated weight, re/im swapped, a wrong sign in the
complex product, the weight index order [c][k][i] transposed, nibbles swapped) would break.
"""
from __future__ import annotations

import numpy as np
import pytest

import oracle
from helpers import pack, tri_index


def _w(wr, wi):
    """int arrays [C][K][N] -> ci8 weight bytes [C][K][2N]."""
    wr = np.asarray(wr, dtype=np.int64)
    wi = np.asarray(wi, dtype=np.int64)
    return np.stack((wr & 0xFF, wi & 0xFF), axis=-1).astype(np.uint8).reshape(*wr.shape[:-1], -1)


def _rand(rng, dtype, shape):
    lim = 7 if dtype == 4 else 127
    return rng.integers(-lim - 1, lim + 1, size=shape), rng.integers(-lim - 1, lim + 1, size=shape)


def test_hand_worked_two_inputs():
    # x0 = 1+2i, x1 = 3-4i; w0 = 2+i, w1 = -1+3i:
    #   w0 x0 = (2-2) + (4+1)i = 0+5i;  w1 x1 = (-3+12) + (4+9)i = 9+13i;  b = 9+18i       (worked by hand)
    for dtype in (4, 8):
        x = pack(dtype, [[[1, 3]]], [[[2, -4]]])
        b = oracle.beamform(x, _w([[[2, -1]]], [[[1, 3]]]), 2, 1, 1, 1, dtype)
        assert b.tolist() == [[[[9, 18]]]]


def test_multiplying_by_i_rotates_a_quarter_turn():
    # w = i on one input: b = i (xr + i xi) = -xi + i xr -- fails if the weight were conjugated or re/im swapped
    rng = np.random.default_rng(1)
    for dtype in (4, 8):
        xr, xi = _rand(rng, dtype, (5, 3, 4))
        wr = np.zeros((3, 1, 4), dtype=np.int64)
        wi = np.zeros((3, 1, 4), dtype=np.int64)
        wi[:, 0, 2] = 1
        b = oracle.beamform(pack(dtype, xr, xi), _w(wr, wi), 4, 3, 5, 1, dtype)
        assert np.array_equal(b[:, :, 0, 0], -xi[:, :, 2])
        assert np.array_equal(b[:, :, 0, 1], xr[:, :, 2])


def test_selector_weights_pick_one_input_per_channel_and_beam():
    # w[c][k][i] = 1 iff i == (c + 2k) % N: pins the [c][k][i] index order of the weights and [t][c][k] of the output
    rng = np.random.default_rng(2)
    T, C, N, K = 4, 5, 6, 3
    xr, xi = _rand(rng, 8, (T, C, N))
    wr = np.zeros((C, K, N), dtype=np.int64)
    for c in range(C):
        for k in range(K):
            wr[c, k, (c + 2 * k) % N] = 1
    b = oracle.beamform(pack(8, xr, xi), _w(wr, np.zeros_like(wr)), N, C, T, K, 8)
    for c in range(C):
        for k in range(K):
            assert np.array_equal(b[:, c, k, 0], xr[:, c, (c + 2 * k) % N])
            assert np.array_equal(b[:, c, k, 1], xi[:, c, (c + 2 * k) % N])


def test_coherent_sum_closed_form():
    # every input carries a + bi, every weight is p + qi: b = N (p + qi)(a + bi)
    N, a, b_, p, q = 12, 5, -3, -7, 4
    x = pack(8, np.full((2, 1, N), a), np.full((2, 1, N), b_))
    out = oracle.beamform(x, _w(np.full((1, 1, N), p), np.full((1, 1, N), q)), N, 1, 2, 1, 8)
    assert out[0, 0, 0].tolist() == [N * (p * a - q * b_), N * (p * b_ + q * a)]


@pytest.mark.parametrize("dtype", [4, 8])
def test_numpy_complex_matmul(dtype):
    # special case that is a library routine: per channel, b = x_c (T x N) @ w_c^T (N x K) in complex128 (exact here)
    rng = np.random.default_rng(3 + dtype)
    T, C, N, K = 7, 3, 10, 4
    xr, xi = _rand(rng, dtype, (T, C, N))
    wr = rng.integers(-128, 128, size=(C, K, N))
    wi = rng.integers(-128, 128, size=(C, K, N))
    b = oracle.beamform(pack(dtype, xr, xi), _w(wr, wi), N, C, T, K, dtype)
    xc = xr + 1j * xi
    wc = wr + 1j * wi
    for c in range(C):
        ref = xc[:, c, :] @ wc[c].T
        assert np.array_equal(b[:, c, :, 0], np.rint(ref.real).astype(np.int64))
        assert np.array_equal(b[:, c, :, 1], np.rint(ref.imag).astype(np.int64))


def test_linear_in_the_weights_and_in_the_voltages():
    rng = np.random.default_rng(5)
    T, C, N, K = 3, 2, 8, 2
    xr, xi = rng.integers(-60, 60, size=(2, T, C, N)), rng.integers(-60, 60, size=(2, T, C, N))
    wr, wi = rng.integers(-60, 60, size=(2, C, K, N)), rng.integers(-60, 60, size=(2, C, K, N))
    f = lambda a, b_, c, d: oracle.beamform(pack(8, a, b_), _w(c, d), N, C, T, K, 8).astype(np.int64)
    assert np.array_equal(f(xr[0], xi[0], wr[0] + wr[1], wi[0] + wi[1]),
                          f(xr[0], xi[0], wr[0], wi[0]) + f(xr[0], xi[0], wr[1], wi[1]))
    assert np.array_equal(f(xr[0] + xr[1], xi[0] + xi[1], wr[0], wi[0]),
                          f(xr[0], xi[0], wr[0], wi[0]) + f(xr[1], xi[1], wr[0], wi[0]))


def test_beam_power_equals_the_quadratic_form_of_the_visibilities():
    # sum_t |b_k|^2 = sum_ij w_i conj(w_j) V_ij with V from the X-engine oracle (full Hermitian matrix from the
    # lower triangle): ties the two definitions together through an identity neither of them uses
    rng = np.random.default_rng(6)
    T, N, K = 9, 5, 2
    xr, xi = _rand(rng, 4, (T, 1, N))
    wr, wi = rng.integers(-20, 20, size=(1, K, N)), rng.integers(-20, 20, size=(1, K, N))
    x = pack(4, xr, xi)
    b = oracle.beamform(x, _w(wr, wi), N, 1, T, K, 4).astype(np.int64)
    v = oracle.xcorr(x, N, 1, T, 4)[0].astype(np.int64)
    for k in range(K):
        w = [complex(int(wr[0, k, i]), int(wi[0, k, i])) for i in range(N)]
        q = 0
        for i in range(N):
            for j in range(N):
                vij = complex(*v[tri_index(i, j)]) if i >= j else complex(*v[tri_index(j, i)]).conjugate()
                q += w[i] * w[j].conjugate() * vij
        assert abs(q.imag) < 1e-6
        assert int(round(q.real)) == int((b[:, 0, k, 0] ** 2 + b[:, 0, k, 1] ** 2).sum())


def test_extreme_codes_whole_weight_range():
    # x = -128 - 128i on 3 inputs, w = -128 + 127i: (-128)(-128) - 127(-128) = 32640; (-128)(-128) + 127(-128) = 128
    x = pack(8, np.full((1, 1, 3), -128), np.full((1, 1, 3), -128))
    b, nwrap = oracle.beamform(x, _w(np.full((1, 1, 3), -128), np.full((1, 1, 3), 127)), 3, 1, 1, 1, 8,
                               return_nwrap=True)
    assert b[0, 0, 0].tolist() == [3 * 32640, 3 * 128] and nwrap == 0
    # every weight code is legal (reading B4).  w = -128 - 128i on the same x, worked by hand:
    # (-128 - 128i)(-128 - 128i) = 128^2 (1 + i)^2 = 32768 i   ->   re 0, im 32768 per input
    b = oracle.beamform(x, _w(np.full((1, 1, 3), -128), np.full((1, 1, 3), -128)), 3, 1, 1, 1, 8)
    assert b[0, 0, 0].tolist() == [0, 3 * 32768]
    # w = 0 - 128i, x = 1 + 0i: -128 i;  x = 0 + 1i: (-128 i)(i) = +128
    b = oracle.beamform(pack(8, np.array([[[1, 0]]]), np.array([[[0, 1]]])),
                        _w(np.zeros((1, 1, 2)), np.full((1, 1, 2), -128)), 2, 1, 1, 1, 8)
    assert b[0, 0, 0].tolist() == [128, -128]


def test_ci4_equals_ci8_on_the_same_values():
    rng = np.random.default_rng(8)
    T, C, N, K = 4, 2, 16, 3
    xr, xi = _rand(rng, 4, (T, C, N))
    w = _w(rng.integers(-128, 128, size=(C, K, N)), rng.integers(-128, 128, size=(C, K, N)))
    assert np.array_equal(oracle.beamform(pack(4, xr, xi), w, N, C, T, K, 4),
                          oracle.beamform(pack(8, xr, xi), w, N, C, T, K, 8))
