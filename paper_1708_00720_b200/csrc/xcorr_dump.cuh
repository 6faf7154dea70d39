// xcorr_dump.cuh -- integration dump: the step after the hot path.  When an
// integration is complete ("accumulate") the packed int32 visibilities are handed on as floats
// (the deployed pipelines convert integer data to floating point for the stages that follow):
//        out[k] = (float) acc[k] * scale        (cvt.rn.f32.s32, then one float32 multiply)
// over the same [nchan][B][2] order, and the accumulator is cleared in the same pass if asked, so that the next
// integration can run with accumulate = 1 from its first span.
//
// Pure streaming: 8 B read + 8 B written (+ 8 B written when clearing) per visibility, 16-byte vectors, a grid
// of a few CTAs per SM walking the buffer with a grid stride.  Bound by HBM.
#pragma once
#include <cstdint>

namespace bfx {

constexpr int DUMP_THREADS = 256;

__global__ void __launch_bounds__(DUMP_THREADS)
xcorr_dump_kernel(int32_t* __restrict__ acc, float* __restrict__ out, long long ncomp, float scale, int zero_acc)
{
    const long long nvec = ncomp >> 2;  // the buffers are 16-byte aligned and ncomp is even; the tail is < 4 components
    const long long stride = static_cast<long long>(gridDim.x) * DUMP_THREADS;
    int4* const a4 = reinterpret_cast<int4*>(acc);
    float4* const o4 = reinterpret_cast<float4*>(out);
    for (long long v = static_cast<long long>(blockIdx.x) * DUMP_THREADS + threadIdx.x; v < nvec; v += stride) {
        const int4 a = __ldcs(a4 + v);
        float4 f;
        f.x = __fmul_rn(__int2float_rn(a.x), scale);
        f.y = __fmul_rn(__int2float_rn(a.y), scale);
        f.z = __fmul_rn(__int2float_rn(a.z), scale);
        f.w = __fmul_rn(__int2float_rn(a.w), scale);
        __stcs(o4 + v, f);
        if (zero_acc) __stcs(a4 + v, make_int4(0, 0, 0, 0));
    }
    if (blockIdx.x == 0 && threadIdx.x < (ncomp & 3)) {
        const long long k = (nvec << 2) + threadIdx.x;
        out[k] = __fmul_rn(__int2float_rn(acc[k]), scale);
        if (zero_acc) acc[k] = 0;
    }
}

// Integration dump with reorder (the optional part of N4; the paper's back end has "efficient data reordering",
// PAPER.md:147): packed lower triangle -> the FULL Hermitian matrix out[c][i][j] in float32, the upper
// triangle being the conjugate of the mirrored lower entry.  One CTA per 32 x 32 tile of the lower triangle of one
// channel: the tile's rows are read as contiguous 256-byte segments of the packed rows, written once as they are and
// once transposed and conjugated through a padded shared-memory tile, so both writes are coalesced too.
constexpr int DM_TILE = 32;

__global__ void __launch_bounds__(256)
xcorr_dump_matrix_kernel(int32_t* __restrict__ acc, float2* __restrict__ out, int ninputs, int nchan, float scale, int zero_acc)
{
    __shared__ float2 tile[DM_TILE][DM_TILE + 1];
    const int tx = threadIdx.x & 31, ty = threadIdx.x >> 5;   // 32 x 8 threads
    // tile index -> (row block R, column block Cb <= R) of the lower triangle of 32 x 32 blocks
    const int q = blockIdx.x;
    int R = static_cast<int>((sqrtf(8.0f * static_cast<float>(q) + 1.0f) - 1.0f) * 0.5f);
    while (R * (R + 1) / 2 > q) --R;
    while ((R + 1) * (R + 2) / 2 <= q) ++R;
    const int Cb = q - R * (R + 1) / 2;
    const long long nbl = static_cast<long long>(ninputs) * (ninputs + 1) / 2;
    for (int c = blockIdx.y; c < nchan; c += gridDim.y) {
        int2* const a = reinterpret_cast<int2*>(acc) + static_cast<long long>(c) * nbl;
        float2* const o = out + static_cast<long long>(c) * ninputs * ninputs;
#pragma unroll
        for (int r = ty; r < DM_TILE; r += 8) {
            const int i = DM_TILE * R + r, j = DM_TILE * Cb + tx;
            if (i < ninputs && j <= i) {
                const long long k = static_cast<long long>(i) * (i + 1) / 2 + j;
                const int2 v = a[k];
                const float2 f = make_float2(__fmul_rn(__int2float_rn(v.x), scale), __fmul_rn(__int2float_rn(v.y), scale));
                o[static_cast<long long>(i) * ninputs + j] = f;
                tile[r][tx] = f;
                if (zero_acc) a[k] = make_int2(0, 0);
            }
        }
        __syncthreads();
#pragma unroll
        for (int r = ty; r < DM_TILE; r += 8) {
            // row j' of the output, column i': the conjugate of V[i'][j'] (strictly above the diagonal only)
            const int jo = DM_TILE * Cb + r, io = DM_TILE * R + tx;
            if (io < ninputs && jo < io) {
                const float2 f = tile[tx][r];
                o[static_cast<long long>(jo) * ninputs + io] = make_float2(f.x, -f.y);
            }
        }
        __syncthreads();
    }
}

}  // namespace bfx
