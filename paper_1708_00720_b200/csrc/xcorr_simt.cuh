// xcorr_simt.cuh -- plain CUDA-core X-engine kernel (BF_XCORR_ALGO_SIMT).
//
// Not the product path: an on-device cross-check of the tcgen05 kernel at sizes the CPU oracle cannot
// reach in test time (include/bfxcorr.h, bfXcorrAlgo).  It shares nothing with the tensor-core kernels: own
// decode, own tiling, own triangle indexing.
//
// One CTA = one channel x one 32x32 block of input pairs (I-block >= J-block); 256 threads, each
// owning a 2x2 patch of pairs; the span is walked in chunks of SIMT_TT samples staged in shared
// memory as (re, im) int16 pairs.  V = sum_t x_i conj(x_j)  (include/bfxcorr.h).
#pragma once
#include <cstdint>

namespace bfx {

constexpr int SIMT_TILE = 32;  // inputs per tile edge
constexpr int SIMT_TT = 64;    // samples staged per chunk

__device__ __forceinline__ short2 simt_decode(const uint8_t* __restrict__ in, int dtype, long long sample)
{
    if (dtype == 8) {
        const char2 v = *reinterpret_cast<const char2*>(in + 2 * sample);
        return make_short2(v.x, v.y);
    }
    const uint8_t b = in[sample];
    const int re = static_cast<int>(static_cast<int8_t>(b & 0xF0)) >> 4;
    const int im = static_cast<int>(static_cast<int8_t>(static_cast<uint8_t>(b << 4))) >> 4;
    return make_short2(static_cast<short>(re), static_cast<short>(im));
}

// grid = (ntile_pairs, min(nchan, 65535)); tile pair p -> (bi >= bj) by row-major triangle enumeration.
__global__ void __launch_bounds__(256)
xcorr_simt_kernel(const uint8_t* __restrict__ in, int32_t* __restrict__ out, int N, int C, int T, int dtype,
                  int accumulate)
{
    __shared__ short2 sa[SIMT_TT][SIMT_TILE];
    __shared__ short2 sb[SIMT_TT][SIMT_TILE];

    // invert p = bi*(bi+1)/2 + bj
    int p = blockIdx.x;
    int bi = static_cast<int>((sqrtf(8.0f * p + 1.0f) - 1.0f) * 0.5f);
    while ((bi + 1) * (bi + 2) / 2 <= p) ++bi;
    while (bi * (bi + 1) / 2 > p) --bi;
    const int bj = p - bi * (bi + 1) / 2;
    const int i0 = bi * SIMT_TILE, j0 = bj * SIMT_TILE;
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;  // 16 x 16 threads, 2x2 pairs each

  for (int c = blockIdx.y; c < C; c += gridDim.y) {
    int re[2][2] = {{0, 0}, {0, 0}}, im[2][2] = {{0, 0}, {0, 0}};

    for (int t0 = 0; t0 < T; t0 += SIMT_TT) {
        __syncthreads();
        for (int e = threadIdx.x; e < SIMT_TT * SIMT_TILE; e += 256) {
            const int tt = e / SIMT_TILE, k = e % SIMT_TILE;
            const int t = t0 + tt;
            short2 a = make_short2(0, 0), b = make_short2(0, 0);
            if (t < T) {
                const long long row = (static_cast<long long>(t) * C + c) * N;
                if (i0 + k < N) a = simt_decode(in, dtype, row + i0 + k);
                if (j0 + k < N) b = simt_decode(in, dtype, row + j0 + k);
            }
            sa[tt][k] = a;
            sb[tt][k] = b;
        }
        __syncthreads();
#pragma unroll 8
        for (int tt = 0; tt < SIMT_TT; ++tt) {
            short2 a[2], b[2];
            a[0] = sa[tt][2 * ty];
            a[1] = sa[tt][2 * ty + 1];
            b[0] = sb[tt][2 * tx];
            b[1] = sb[tt][2 * tx + 1];
#pragma unroll
            for (int u = 0; u < 2; ++u)
#pragma unroll
                for (int v = 0; v < 2; ++v) {
                    re[u][v] += a[u].x * b[v].x + a[u].y * b[v].y;
                    im[u][v] += a[u].y * b[v].x - a[u].x * b[v].y;
                }
        }
    }

    const long long B = static_cast<long long>(N) * (N + 1) / 2;
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int v = 0; v < 2; ++v) {
            const int i = i0 + 2 * ty + u, j = j0 + 2 * tx + v;
            if (i < N && j <= i) {
                int32_t* dst = out + 2 * (static_cast<long long>(c) * B + static_cast<long long>(i) * (i + 1) / 2 + j);
                int2 acc = make_int2(re[u][v], im[u][v]);
                if (accumulate) {
                    const int2 old = *reinterpret_cast<const int2*>(dst);
                    acc.x = static_cast<int>(static_cast<unsigned>(acc.x) + static_cast<unsigned>(old.x));
                    acc.y = static_cast<int>(static_cast<unsigned>(acc.y) + static_cast<unsigned>(old.y));
                }
                *reinterpret_cast<int2*>(dst) = acc;
            }
        }
  }  // channel loop
}

}  // namespace bfx
