"""Pins for oracle/xcorr_oracle.c against what the definition and the mathematics fix
(pins P1..P12).  CPU only.

Each pin is chosen so that one plausible mistake in the oracle (conjugate on the wrong
factor, swapped nibbles, wrong triangle index, dropped term, off-by-one at i == j or
i == N-1, accumulate ignored) fails it.  None of them re-types the oracle's loop:
they use hand-worked values, closed forms, O(NT) identities, numpy complex128 matmul
and a sample-by-sample Python complex evaluation.
"""
import numpy as np
import pytest

import oracle
from helpers import pack, pack_ci4, pack_ci8, read_golden, tri_index


def rand_span(rng, T, C, N, dtype, extremes=True):
    lo, hi = (-8, 7) if dtype == 4 else (-128, 127)
    if not extremes:
        lo += 1
    re = rng.integers(lo, hi + 1, size=(T, C, N))
    im = rng.integers(lo, hi + 1, size=(T, C, N))
    return re, im


# ---------------------------------------------------------------- P1 hand-worked examples
@pytest.mark.parametrize("name", ["worked_example_n3.txt", "worked_example_n2.txt"])
@pytest.mark.parametrize("dtype", [4, 8])
def test_p1_worked_example(name, dtype):
    g = read_golden(name)
    T = 1 + max(t for t, _, _, _ in g["x"])
    N = 1 + max(i for _, i, _, _ in g["x"])
    re = np.zeros((T, 1, N), dtype=np.int64)
    im = np.zeros((T, 1, N), dtype=np.int64)
    for t, i, r, m in g["x"]:
        re[t, 0, i], im[t, 0, i] = r, m
    x = pack(dtype, re, im)
    key = "ci4" if dtype == 4 else "ci8"
    for t, row in g[key].items():           # the byte formats themselves are part of the fixture
        assert x[t, 0].tobytes() == row
    out = oracle.xcorr(x, N, 1, T, dtype)
    assert out.shape == (1, N * (N + 1) // 2, 2)
    for k, vr, vi in g["v"]:
        assert (int(out[0, k, 0]), int(out[0, k, 1])) == (vr, vi), k


# ---------------------------------------------------------------- P2 two constant inputs
@pytest.mark.parametrize("dtype", [4, 8])
def test_p2_two_constant_inputs_closed_form(dtype):
    N, C, T = 7, 2, 5
    p, q = 5, 2
    a, b, c, d = 3, -2, -1, 4                       # x_p = 3-2j, x_q = -1+4j
    re = np.zeros((T, C, N), dtype=np.int64)
    im = np.zeros((T, C, N), dtype=np.int64)
    re[:, :, p], im[:, :, p] = a, b
    re[:, :, q], im[:, :, q] = c, d
    out = oracle.xcorr(pack(dtype, re, im), N, C, T, dtype)
    exp = np.zeros_like(out)
    exp[:, tri_index(p, q)] = (T * (a * c + b * d), T * (b * c - a * d))      # (-55, -50)
    exp[:, tri_index(p, p)] = (T * (a * a + b * b), 0)
    exp[:, tri_index(q, q)] = (T * (c * c + d * d), 0)
    assert (exp[0, tri_index(p, q)] == (-55, -50)).all()
    np.testing.assert_array_equal(out, exp)


def test_p2_unit_imag_sign():
    # x_i = j, x_j = 1  =>  V_ij = j * conj(1) = +j per sample (reading A1: Im = +T)
    N, T = 2, 9
    re = np.zeros((T, 1, N), dtype=np.int64)
    im = np.zeros((T, 1, N), dtype=np.int64)
    re[:, 0, 0] = 1        # x_0 = 1
    im[:, 0, 1] = 1        # x_1 = j
    out = oracle.xcorr(pack_ci8(re, im), N, 1, T, 8)
    assert tuple(out[0, tri_index(1, 0)]) == (0, T)


def test_p2_single_impulse():
    N, C, T = 6, 3, 4
    re = np.zeros((T, C, N), dtype=np.int64)
    im = np.zeros((T, C, N), dtype=np.int64)
    re[2, 1, 4], im[2, 1, 4] = -7, 5              # one non-zero sample in the whole span
    out = oracle.xcorr(pack_ci8(re, im), N, C, T, 8)
    exp = np.zeros_like(out)
    exp[1, tri_index(4, 4)] = (49 + 25, 0)
    np.testing.assert_array_equal(out, exp)


# ---------------------------------------------------------------- P3 Hermitian symmetry, P4 autos
@pytest.mark.parametrize("dtype", [4, 8])
def test_p3_p4_hermitian_and_autos(dtype):
    rng = np.random.default_rng(3)
    N, C, T = 9, 2, 33
    re, im = rand_span(rng, T, C, N, dtype)
    x = pack(dtype, re, im)
    cc, ii, jj = np.meshgrid(np.arange(C), np.arange(N), np.arange(N), indexing="ij")
    full = oracle.xcorr_entries(x, N, C, T, dtype, cc.ravel(), ii.ravel(), jj.ravel()).reshape(C, N, N, 2)
    np.testing.assert_array_equal(full[..., 0], full[..., 0].transpose(0, 2, 1))      # Re symmetric
    np.testing.assert_array_equal(full[..., 1], -full[..., 1].transpose(0, 2, 1))     # Im antisymmetric
    d = np.arange(N)
    assert (full[:, d, d, 1] == 0).all()
    np.testing.assert_array_equal(full[:, d, d, 0], (re.astype(np.int64) ** 2 + im ** 2).sum(axis=0))
    assert (full[:, d, d, 0] >= 0).all()
    # the packed triangle is the i >= j part of that matrix
    out = oracle.xcorr(x, N, C, T, dtype)
    for i in range(N):
        for j in range(i + 1):
            np.testing.assert_array_equal(out[:, tri_index(i, j)], full[:, i, j])


# ---------------------------------------------------------------- P5 O(NT) identities
def beam_power_check(out, re, im, w):
    """sum_i |w_i|^2 V_ii + 2 Re sum_{i>j} w_i conj(w_j) V_ij  ==  sum_t |sum_i w_i x_i|^2 (per channel)."""
    T, C, N = re.shape
    x = re.astype(np.complex128) + 1j * im
    rhs = (np.abs((x * w[None, None, :]).sum(axis=2)) ** 2).sum(axis=0)          # [C], exact (< 2^53)
    V = out[..., 0].astype(np.complex128) + 1j * out[..., 1]
    lhs = np.zeros(C)
    for i in range(N):
        lhs += (abs(w[i]) ** 2) * V[:, tri_index(i, i)].real
        for j in range(i):
            lhs += 2.0 * (w[i] * np.conj(w[j]) * V[:, tri_index(i, j)]).real
    np.testing.assert_array_equal(lhs, rhs)


@pytest.mark.parametrize("dtype", [4, 8])
def test_p5_trace_and_beam_power(dtype):
    rng = np.random.default_rng(5)
    N, C, T = 12, 3, 50
    re, im = rand_span(rng, T, C, N, dtype)
    out = oracle.xcorr(pack(dtype, re, im), N, C, T, dtype)
    tr = sum(out[:, tri_index(i, i), 0].astype(np.int64) for i in range(N))
    np.testing.assert_array_equal(tr, (re ** 2 + im ** 2).sum(axis=(0, 2)))
    beam_power_check(out, re, im, np.ones(N, dtype=np.complex128))                # sees Re only
    beam_power_check(out, re, im, (1j) ** np.arange(N))                           # sees Im and its sign


# ---------------------------------------------------------------- P6 accumulation laws
@pytest.mark.parametrize("dtype", [4, 8])
def test_p6_accumulation(dtype):
    rng = np.random.default_rng(6)
    N, C, T = 5, 2, 24
    re, im = rand_span(rng, T, C, N, dtype)
    x = pack(dtype, re, im)
    one = oracle.xcorr(x, N, C, T, dtype)
    # accumulate=0 ignores whatever is in out
    garbage = rng.integers(-2**31, 2**31 - 1, size=one.shape, dtype=np.int64).astype(np.int32)
    np.testing.assert_array_equal(oracle.xcorr(x, N, C, T, dtype, out=garbage.copy()), one)
    # twice with accumulate -> exactly 2x
    acc = one.copy()
    oracle.xcorr(x, N, C, T, dtype, out=acc, accumulate=True)
    np.testing.assert_array_equal(acc, 2 * one)
    # one span of T == two spans of T/2 accumulated
    h = T // 2
    halves = oracle.xcorr(x[:h], N, C, h, dtype)
    oracle.xcorr(x[h:], N, C, T - h, dtype, out=halves, accumulate=True)
    np.testing.assert_array_equal(halves, one)


def test_p6_wraps_mod_2_32():
    # reading A7: the int32 accumulator wraps; the oracle reports how many sums did not fit
    N, T = 1, 4
    x = pack_ci8(np.full((T, 1, N), -128), np.full((T, 1, N), -128))
    out = np.full((1, 1, 2), 2**31 - 1, dtype=np.int32)
    out, nwrap = oracle.xcorr(x, N, 1, T, 8, out=out, accumulate=True, return_nwrap=True)
    assert nwrap == 0                                   # the span's own sum fits
    assert int(out[0, 0, 0]) == ((2**31 - 1 + 4 * 32768 + 2**31) % 2**32) - 2**31


# ---------------------------------------------------------------- P7 invariances
def test_p7_invariances():
    rng = np.random.default_rng(7)
    N, C, T = 6, 3, 20
    re, im = rand_span(rng, T, C, N, 8, extremes=False)          # avoid -128 so that *j stays in range
    base = oracle.xcorr(pack_ci8(re, im), N, C, T, 8)
    # permuting time samples
    pt = rng.permutation(T)
    np.testing.assert_array_equal(oracle.xcorr(pack_ci8(re[pt], im[pt]), N, C, T, 8), base)
    # permuting channels
    pc = rng.permutation(C)
    np.testing.assert_array_equal(oracle.xcorr(pack_ci8(re[:, pc], im[:, pc]), N, C, T, 8), base[pc])
    # multiplying every sample by j: (re, im) -> (-im, re)
    np.testing.assert_array_equal(oracle.xcorr(pack_ci8(-im, re), N, C, T, 8), base)
    # multiplying only input k by j: row k times j, column k times -j
    k = 2
    re2, im2 = re.copy(), im.copy()
    re2[:, :, k], im2[:, :, k] = -im[:, :, k], re[:, :, k]
    got = oracle.xcorr(pack_ci8(re2, im2), N, C, T, 8)
    exp = base.copy()
    for i in range(N):
        for j in range(i + 1):
            v = base[:, tri_index(i, j)].astype(np.int64)
            if i == k and j != k:
                exp[:, tri_index(i, j)] = np.stack((-v[:, 1], v[:, 0]), axis=-1)      # * j
            elif j == k and i != k:
                exp[:, tri_index(i, j)] = np.stack((v[:, 1], -v[:, 0]), axis=-1)      # * -j
    np.testing.assert_array_equal(got, exp)
    # permuting inputs permutes the (full, Hermitian) matrix
    pi = rng.permutation(N)
    got = oracle.xcorr(pack_ci8(re[:, :, pi], im[:, :, pi]), N, C, T, 8)
    for i in range(N):
        for j in range(i + 1):
            a, b = pi[i], pi[j]
            v = base[:, tri_index(max(a, b), min(a, b))].astype(np.int64)
            if a < b:
                v = np.stack((v[:, 0], -v[:, 1]), axis=-1)                            # conj
            np.testing.assert_array_equal(got[:, tri_index(i, j)], v)


# ---------------------------------------------------------------- P8 numpy complex128 HERK
@pytest.mark.parametrize("dtype,N,C,T", [(8, 40, 3, 300), (4, 33, 2, 513), (8, 64, 2, 128)])
def test_p8_numpy_herk(dtype, N, C, T):
    rng = np.random.default_rng(8)
    re, im = rand_span(rng, T, C, N, dtype)
    out = oracle.xcorr(pack(dtype, re, im), N, C, T, dtype)
    x = re.astype(np.complex128) + 1j * im                     # [T][C][N]; all sums < 2^53: exact
    for c in range(C):
        X = x[:, c, :]                                         # [T][N]
        V = X.T @ X.conj()                                     # V[i][j] = sum_t x_i conj(x_j)
        ii, jj = np.tril_indices(N)
        np.testing.assert_array_equal(out[c, :, 0], np.rint(V[ii, jj].real).astype(np.int64))
        np.testing.assert_array_equal(out[c, :, 1], np.rint(V[ii, jj].imag).astype(np.int64))


# ---------------------------------------------------------------- P9 ci4 == ci8
def test_p9_ci4_equals_widened_ci8():
    rng = np.random.default_rng(9)
    N, C, T = 10, 4, 64
    re, im = rand_span(rng, T, C, N, 4)
    np.testing.assert_array_equal(oracle.xcorr(pack_ci4(re, im), N, C, T, 4),
                                  oracle.xcorr(pack_ci8(re, im), N, C, T, 8))


# ---------------------------------------------------------------- P10 extreme codes
def test_p10_extremes():
    N, C, T = 4, 2, 4
    nb = N * (N + 1) // 2
    x8 = np.full((T, C, 2 * N), 0x80, dtype=np.uint8)             # -128-128j everywhere
    out = oracle.xcorr(x8, N, C, T, 8)
    assert (out[..., 0] == 4 * 32768).all() and (out[..., 1] == 0).all() and out.shape == (C, nb, 2)
    x4 = np.full((T, C, N), 0x88, dtype=np.uint8)                 # -8-8j everywhere
    out = oracle.xcorr(x4, N, C, T, 4)
    assert (out[..., 0] == 4 * 128).all() and (out[..., 1] == 0).all()


# ---------------------------------------------------------------- P12 brute force, tiny random
def brute_force(x_bytes, N, C, T, dtype):
    """Differently written: decode with Python ints, full N x N matrix by complex arithmetic
    sample by sample, then take the lower triangle and pack."""
    raw = x_bytes.reshape(T, C, -1)
    out = np.zeros((C, N * (N + 1) // 2, 2), dtype=np.int64)
    for c in range(C):
        M = [[0j] * N for _ in range(N)]
        for t in range(T):
            xs = []
            for i in range(N):
                if dtype == 8:
                    r, m = int(raw[t, c, 2 * i]), int(raw[t, c, 2 * i + 1])
                    r, m = (r - 256 if r > 127 else r), (m - 256 if m > 127 else m)
                else:
                    byte = int(raw[t, c, i])
                    r, m = byte // 16, byte % 16
                    r, m = (r - 16 if r > 7 else r), (m - 16 if m > 7 else m)
                xs.append(complex(r, m))
            for i in range(N):
                for j in range(N):
                    M[i][j] += xs[i] * xs[j].conjugate()
        k = 0
        for i in range(N):
            for j in range(i + 1):
                out[c, k] = (int(M[i][j].real), int(M[i][j].imag))
                k += 1
    return out


@pytest.mark.parametrize("seed", range(6))
@pytest.mark.parametrize("dtype", [4, 8])
def test_p12_brute_force(seed, dtype):
    rng = np.random.default_rng(100 + seed)
    N = int(rng.integers(1, 9))
    C = int(rng.integers(1, 4))
    T = int(rng.integers(1, 17))
    re, im = rand_span(rng, T, C, N, dtype)
    x = pack(dtype, re, im)
    np.testing.assert_array_equal(oracle.xcorr(x, N, C, T, dtype), brute_force(x, N, C, T, dtype))


# ---------------------------------------------------------------- argument checking
def test_bad_arguments():
    x = np.zeros(16, dtype=np.uint8)
    with pytest.raises(ValueError):
        oracle.xcorr(x, 4, 1, 3, 8)            # wrong byte count
    with pytest.raises(ValueError):
        oracle.xcorr(x, 8, 1, 1, 8, accumulate=True)
    assert oracle.threads() >= 1


# ---- integration dump: int32 accumulators -> float32, pinned against what IEEE-754 fixes ----
def test_dump_exact_values_and_zeroing():
    """Integers up to 2^24 in magnitude are exactly representable in float32: the dump of such values with scale 1
    must reproduce them digit for digit, and power-of-two scales only change the exponent."""
    acc = np.array([[[0, 1], [-1, 2 ** 24]], [[-(2 ** 24), 12345678], [7, -8]]], dtype=np.int32)
    keep = acc.copy()
    out = oracle.dump(acc, 1.0)
    assert out.dtype == np.float32 and out.shape == acc.shape
    assert [float(v) for v in out.reshape(-1)] == [0.0, 1.0, -1.0, 16777216.0, -16777216.0, 12345678.0, 7.0, -8.0]
    np.testing.assert_array_equal(acc, keep)                      # zero_acc = 0 leaves the accumulator alone
    half = oracle.dump(acc, 0.5)
    assert [float(v) for v in half.reshape(-1)] == [0.0, 0.5, -0.5, 8388608.0, -8388608.0, 6172839.0, 3.5, -4.0]
    out2 = oracle.dump(acc, 1.0, zero_acc=True)
    np.testing.assert_array_equal(out2, out)
    assert not acc.any()                                          # cleared for the next integration


def test_dump_rounds_to_nearest_even_beyond_2_24():
    """Worked by hand: float32 has a 24-bit significand, so above 2^24 integers are spaced 2 apart (4 above 2^25) and
    ties go to the even significand: 2^24+1 -> 2^24, 2^24+3 -> 2^24+4, 2^25+2 -> 2^25, 2^25+6 -> 2^25+8; INT32_MAX -> 2^31."""
    acc = np.array([2 ** 24 + 1, 2 ** 24 + 2, 2 ** 24 + 3, 2 ** 25 + 2, 2 ** 25 + 6, -(2 ** 24) - 1, 2 ** 31 - 1, -(2 ** 31)],
                   dtype=np.int32)
    out = oracle.dump(acc, 1.0)
    assert [float(v) for v in out] == [16777216.0, 16777218.0, 16777220.0, 33554432.0, 33554440.0, -16777216.0,
                                       2147483648.0, -2147483648.0]


def test_dump_agrees_with_numpy_float32_arithmetic():
    """Library special case: numpy's int32 -> float32 cast and float32 multiply follow the same IEEE rules."""
    rng = np.random.default_rng(3)
    acc = rng.integers(-2 ** 31, 2 ** 31, size=(5, 33, 2), dtype=np.int64).astype(np.int32)
    for scale in (1.0, 1.0 / 1024, 3.0e-5):
        exp = acc.astype(np.float32) * np.float32(scale)
        np.testing.assert_array_equal(oracle.dump(acc, scale), exp)


# ---- integration dump with reorder (optional part): packed triangle -> full Hermitian float32 matrix ----
def test_dump_matrix_worked_example_and_hermitian():
    """The hand-worked N = 3 visibilities of tests/golden/worked_example_n3.txt as a full matrix, written out by hand:
    row i, column j holds V_ij below / on the diagonal and conj(V_ji) above it."""
    g = read_golden("worked_example_n3.txt")
    acc = np.array([[(r, m) for _, r, m in g["v"]]], dtype=np.int32)       # [1][6][2]: (17,0) (-9,22) (46,0) (1,0) (-15,3) (34,0)
    m = oracle.dump_matrix(acc, 3, 1.0)
    z = m[0, ..., 0] + 1j * m[0, ..., 1]
    exp = np.array([[17, -9 - 22j, 1 - 0j], [-9 + 22j, 46, -15 - 3j], [1 + 0j, -15 + 3j, 34]])
    assert np.array_equal(z, exp)
    assert np.array_equal(z, z.conj().T)                                    # Hermitian
    assert np.signbit(m[0, 0, 2, 1]) and not np.signbit(m[0, 2, 0, 1])      # conj of a zero imaginary part is -0.0
    half = oracle.dump_matrix(acc, 3, 0.5)
    assert np.array_equal(half, m * np.float32(0.5))


def test_dump_matrix_agrees_with_dump_and_numpy_indexing():
    """Independent construction: oracle.dump's floats scattered into a matrix with numpy's tril indices; zeroing."""
    rng = np.random.default_rng(21)
    N, C = 11, 3
    nb = N * (N + 1) // 2
    acc = rng.integers(-2**31, 2**31, size=(C, nb, 2), dtype=np.int64).astype(np.int32)
    scale = 0.37
    flat = oracle.dump(acc.copy(), scale)
    exp = np.zeros((C, N, N, 2), dtype=np.float32)
    ii, jj = np.tril_indices(N)                                             # row-major lower triangle = the packed order
    exp[:, ii, jj] = flat
    exp[:, jj, ii, 0] = flat[..., 0]
    off = ii != jj
    exp[:, jj[off], ii[off], 1] = -flat[:, off, 1]
    work = acc.copy()
    got = oracle.dump_matrix(work, N, scale, zero_acc=True)
    assert np.array_equal(got.view(np.uint32)[:, ii, jj], exp.view(np.uint32)[:, ii, jj])
    assert np.array_equal(got, exp) and not work.any()
    assert np.array_equal(oracle.dump_matrix(acc.copy(), N, scale), got)    # zero_acc does not change the output
