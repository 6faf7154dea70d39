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

}  // namespace bfx
