// mem_probe.cuh -- a no-math streaming kernel with the X-engine's HBM access mix ("measure a
// same-mix streaming kernel ... as the true HBM ceiling"): every 16-byte vector of `in` is read once, every 16-byte
// vector of `out` is written once (accumulate = 0) or read, incremented and written back (accumulate != 0), the two
// streams interleaved in proportion, all accesses coalesced and contiguous.  It is what the path's algorithmic bytes
// cost when nothing but the memory system is in the way; bench.py times it beside the real kernel and reports it as
// roofline.same_mix_peak.  Measurement aid only: it computes nothing of the method.
#pragma once
#include <cstdint>
#include "ptx_sm100.cuh"

namespace bfx {

constexpr int MP_THREADS = 512;

// One chunk = 4 vectors per thread.  The `in` chunks and the `out` chunks are dealt to the blocks round-robin and
// interleaved in proportion, so at any moment the whole grid works on one neighbourhood of each stream (as a copy
// kernel's blocks do) with loads and stores in flight together.
constexpr int MP_CHUNK = 4 * MP_THREADS;

__global__ void __launch_bounds__(MP_THREADS) mem_probe_kernel(const uint4* __restrict__ in, long long nin, uint4* __restrict__ out,
                                                               long long nout, int accumulate, unsigned int* sink)
{
    uint32_t acc = 0;
    const unsigned long long nci = (nin + MP_CHUNK - 1) / MP_CHUNK, nco = (nout + MP_CHUNK - 1) / MP_CHUNK;
    const unsigned long long nc = nci > nco ? nci : nco;
    // chunk of stream s handled at step k: floor(k * ncs / nc), taken when it differs from step k - 1's (32.32 fixed point)
    const unsigned long long ri = nc ? (nci << 32) / nc : 0, ro = nc ? (nco << 32) / nc : 0;
    for (unsigned long long k = blockIdx.x; k < nc; k += gridDim.x) {
        uint4 v[4];
        const unsigned long long ci = nci == nc ? k : (k * ri) >> 32, co = nco == nc ? k : (k * ro) >> 32;
        const bool do_in = nci == nc || k == 0 || ((k - 1) * ri) >> 32 != ci;
        const bool do_out = nco == nc || k == 0 || ((k - 1) * ro) >> 32 != co;
        const long long ib = static_cast<long long>(ci) * MP_CHUNK + threadIdx.x, ob = static_cast<long long>(co) * MP_CHUNK + threadIdx.x;
        if (do_in && ci < nci) {
#pragma unroll
            for (int q = 0; q < 4; ++q)
                if (ib + q * MP_THREADS < nin) {
                    v[q] = ptx::ld_global_stream_v4(reinterpret_cast<const uint8_t*>(in + ib + q * MP_THREADS));
                    acc ^= v[q].x ^ v[q].y ^ v[q].z ^ v[q].w;
                }
        }
        if (do_out && co < nco) {
            if (accumulate) {
                uint4 w[4];
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (ob + q * MP_THREADS < nout) w[q] = out[ob + q * MP_THREADS];
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (ob + q * MP_THREADS < nout) {
                        w[q].x += 1u; w[q].y += 1u; w[q].z += 1u; w[q].w += 1u;
                        out[ob + q * MP_THREADS] = w[q];
                    }
            } else {
                const uint4 w = make_uint4(static_cast<uint32_t>(k), 1u, 2u, 3u);
#pragma unroll
                for (int q = 0; q < 4; ++q)
                    if (ob + q * MP_THREADS < nout) out[ob + q * MP_THREADS] = w;
            }
        }
    }
    if (acc == 0x9E3779B9u && sink) atomicAdd(sink, 1u);   // keeps the loads alive; practically never taken
}

}  // namespace bfx
