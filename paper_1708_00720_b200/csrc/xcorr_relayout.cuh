// xcorr_relayout.cuh -- S1, the unpack-and-transpose stage.
//
// A span arrives as x[t][c][i] (include/bfxcorr.h): the samples of one channel lie nchan*row bytes
// apart, one piece per time sample.  The tensor-core kernel re-reads every 64-input piece of a channel
// once per tile that uses it (6x at 512 inputs, 17x at 2048), and fetched straight from the span each
// of those reads is a 64..128-byte access to a different 2 MiB page: measured on B200, the TMA unit
// then spends its time on address translation and the contraction runs at a quarter of the tensor peak
// (profiles/round1.md).  So the span is first rewritten, once, channel-major:
//
//     z[c][t][2 i + part]   int8,  part 0 = re, 1 = im          (the "real-embedded complex layout")
//
// ci8 bytes are copied as they are; ci4 bytes are widened to two sign-extended int8.  Every (t, c) row is
// read with coalesced 16-byte loads, exactly once, and written as coalesced 16-byte stores; a channel's
// slab z[c] is contiguous, so the operand boxes of xcorr_tcgen05.cuh touch one or two pages per tile.
#pragma once
#include <cstdint>

namespace bfx {

constexpr int RL_TB = 32;        // samples per CTA
constexpr int RL_THREADS = 256;

__device__ __forceinline__ uint4 rl_ld16(const uint8_t* p)
{
    uint4 v;
    asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0, %1, %2, %3}, [%4];"
                 : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                 : "l"(p));
    return v;
}

__device__ __forceinline__ void rl_st16(uint8_t* p, uint4 v)
{
    asm volatile("st.global.L1::no_allocate.v4.u32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(v.x), "r"(v.y), "r"(v.z), "r"(v.w)
                 : "memory");
}

// four ci4 bytes (re = high nibble, im = low nibble, two's complement: include/bfxcorr.h) ->
// eight int8: re0 im0 re1 im1 | re2 im2 re3 im3
__device__ __forceinline__ void rl_widen(uint32_t w, uint32_t& o0, uint32_t& o1)
{
    const uint32_t ure = (w >> 4) & 0x0F0F0F0Fu, uim = w & 0x0F0F0F0Fu;
    // sign-extend each nibble inside its byte: bit 3 set -> OR in 0xF0 (bit3 * 0x1E = bits 4..7)
    const uint32_t sre = ure | ((ure & 0x08080808u) * 0x1Eu);
    const uint32_t sim = uim | ((uim & 0x08080808u) * 0x1Eu);
    o0 = __byte_perm(sre, sim, 0x5140);
    o1 = __byte_perm(sre, sim, 0x7362);
}

// grid = (ceil(ntime / RL_TB), nchan).  row_in = ninputs * (1 | 2) bytes, a multiple of 16.
template <bool CI4>
__global__ void __launch_bounds__(RL_THREADS)
xcorr_relayout_kernel(const uint8_t* __restrict__ in, uint8_t* __restrict__ z, int row_in, int nchan, int ntime)
{
    const int c = blockIdx.y;
    const int t0 = blockIdx.x * RL_TB;
    const int nt = min(RL_TB, ntime - t0);
    const int vec = row_in >> 4;        // 16-byte vectors per input row
    const int total = nt * vec;
    const long long row_out = CI4 ? 2ll * row_in : row_in;
    const uint8_t* src = in + (static_cast<long long>(t0) * nchan + c) * row_in;
    uint8_t* dst = z + (static_cast<long long>(c) * ntime + t0) * row_out;
    const long long src_pitch = static_cast<long long>(nchan) * row_in;
    constexpr int U = 4;
    for (int base = threadIdx.x; base < total; base += U * RL_THREADS) {
        uint4 v[U];
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int idx = base + u * RL_THREADS;
            if (idx < total) v[u] = rl_ld16(src + (idx / vec) * src_pitch + (idx % vec) * 16);
        }
#pragma unroll
        for (int u = 0; u < U; ++u) {
            const int idx = base + u * RL_THREADS;
            if (idx < total) {
                uint8_t* d = dst + (idx / vec) * row_out + (idx % vec) * (CI4 ? 32 : 16);
                if (CI4) {
                    uint4 a, b;
                    rl_widen(v[u].x, a.x, a.y);
                    rl_widen(v[u].y, a.z, a.w);
                    rl_widen(v[u].z, b.x, b.y);
                    rl_widen(v[u].w, b.z, b.w);
                    rl_st16(d, a);
                    rl_st16(d + 16, b);
                } else {
                    rl_st16(d, v[u]);
                }
            }
        }
    }
}

}  // namespace bfx
