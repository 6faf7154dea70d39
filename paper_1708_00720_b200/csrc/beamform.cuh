// beamform.cuh -- phase-and-sum beamformer on the span x[t][c][i] (include/bfbeamform.h).
//
// Per channel c it is the dense contraction  b[t][k] = sum_i w[c][k][i] x[t][c][i]  over the INPUT axis, so, unlike
// the X-engine, the span rows are already the K-major operand: a row x[t][c][0..N) of ci8 samples is, byte for byte,
// the int8 row a[t][0..2N) with a[2i] = re_i, a[2i+1] = im_i.  Re b needs -wi, kind::i8 cannot negate an operand, and
// -(-128) is no int8: so the weight operand is UNSIGNED 8-bit (the instruction descriptor gives A and B their own
// formats) and holds every weight with an offset; per channel, two rows per beam and two rows of selectors:
//     W[2k  ][2i] = wr + 128   W[2k  ][2i+1] = 127 - wi    ->  D[t][2k]   = Re b[t][k] + 128 Sr[t] + 127 Si[t]
//     W[2k+1][2i] = wi + 128   W[2k+1][2i+1] = wr + 128    ->  D[t][2k+1] = Im b[t][k] + 128 Sr[t] + 128 Si[t]
//     W[2K  ][2i] = 1          W[2K  ][2i+1] = 0           ->  D[t][2K]   = Sr[t] = sum_i re_i
//     W[2K+1][2i] = 0          W[2K+1][2i+1] = 1           ->  D[t][2K+1] = Si[t] = sum_i im_i
// (bfBeamformSetWeights); the epilogue subtracts the offsets, exactly (int32, wrapping), so every weight code
// including -128 - 128j is legal (reading B4).  ci4 rows are widened
// on chip as in xcorr_pair4.cuh: each 32-bit word of 4 samples becomes the 4 re bytes (<< 4) then the 4 im bytes
// (<< 4), the weight rows are stored in the same grouped order, and the factor 16 is shifted out exactly in the
// epilogue.  Every sample is used once, so the span is consumed in place: no ring, no relayout.
//
// Work unit: 128 samples x 1 channel (MMA M = 128 samples, N = 2 nbeam rounded up to 16, K = the input axis in
// stages of 128 span bytes).  Units are dealt round-robin in groups of `group` adjacent channels x all sample blocks,
// so the CTAs of one wave read adjacent channels of the same samples (whole DRAM pages) and a group's weights stay
// in the L2 while its sample blocks go by.
//
// Roles (512 threads, one CTA per SM): warp 0 span producer (TMA boxes of 128 span bytes x 128 samples of one channel:
// ci8 lands 128B-swizzled straight in the operand stage -- two adjacent 128-byte pieces per box through a 5-d view of
// the span where the shape allows it (rows a multiple of 256 bytes, samples a multiple of 8, two stages fit), which
// the memory system serves much faster when a channel's samples lie pages apart: 76 -> 92 % of the HBM copy peak on
// BASELINE.json configs[2], 70 -> 102 % on configs[3] (profiles/round2.md) --, ci4 lands raw in a ring), warp 3 weight producer (ci4 only; for
// ci8 warp 0 loads both), warp 1 MMA issuer, warp 2 TMEM allocator, warps 4..7 epilogue (TMEM -> registers -> shared
// staging -> global, eight lanes per 128-byte row piece), warps 8..15 (ci4 only) widen raw rows into the 128B-swizzled K-major int8 layout the
// UMMA descriptor expects.  TMA keeps every free stage in flight (up to 128 KB per SM), which register-staged loads
// could not (profiles/round1.md).
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ptx_sm100.cuh"

namespace bfx {

constexpr int BM_MT = 128;             // samples per unit
constexpr int BM_LOAD_WARPS = 8;
constexpr int BM_THREADS = 256 + 32 * BM_LOAD_WARPS;
constexpr int BM_MAX_STAGES = 8;
constexpr int BM_MAX_RAW = 4;          // raw ci4 stages (16 KB each)
constexpr int BM_STG_PITCH = 144;      // epilogue staging: 32 rows x 128 bytes, pitch 144 -> conflict-free 16-byte accesses
constexpr int BM_STG_WARP = 32 * BM_STG_PITCH;
constexpr int BM_STG_BYTES = 4 * BM_STG_WARP;
constexpr int BM_SMEM_MAX = 232448 - 1024;

struct BmParams {
    const uint8_t* x;
    int32_t* out;
    int ninputs, nchan, ntime, nbeam;
    int row_in;      // bytes of one (t, c) row of the span
    int nb2;         // MMA N: 2 * nbeam rounded up to a multiple of 16
    int nks;         // K stages: ceil(row_in / 128)
    int ntb;         // sample blocks: ceil(ntime / 128)
    int group;       // adjacent channels per scheduling group
    int stages;      // operand stages
    int raw_stages;  // raw ci4 stages (0 for ci8)
    int pw;          // ci8: 128-byte row pieces per K stage and span box (1, or 2 with the 5-d span map: see the producer)
    long long nunits;
};

// the (sample block, channel) of unit u: groups of `group` channels, sample blocks inside a group, channels fastest
struct BmUnit {
    int c, t0;
};
__device__ __forceinline__ BmUnit bm_decode(const BmParams& p, long long u)
{
    const long long per = static_cast<long long>(p.group) * p.ntb;
    const int cg = static_cast<int>(u / per);
    const int r = static_cast<int>(u - cg * per);
    int gl = p.nchan - cg * p.group;
    gl = gl > p.group ? p.group : gl;
    const int tb = r / gl;
    return BmUnit{cg * p.group + (r - tb * gl), tb * BM_MT};
}

// UMMA shared-memory descriptor, K-major, SWIZZLE_128B: rows of 128 bytes, 8-row atoms `sbo` bytes apart (1024: a dense tile)
__device__ __forceinline__ uint64_t bm_smem_desc(uint32_t saddr, uint32_t sbo = 1024u)
{
    uint64_t d = 0;
    d |= static_cast<uint64_t>((saddr >> 4) & 0x3FFF);
    d |= static_cast<uint64_t>(1) << 16;
    d |= static_cast<uint64_t>((sbo >> 4) & 0x3FFF) << 32;
    d |= static_cast<uint64_t>(1) << 46;
    d |= static_cast<uint64_t>(2) << 61;
    return d;
}

// UMMA instruction descriptor: dense, D = S32, A = signed int8 (voltages), B = UNSIGNED int8 (offset weights), both K-major
__host__ __device__ constexpr uint32_t bm_instr_desc(int m, int n)
{
    return (2u << 4) | (1u << 7) | (0u << 10) | (static_cast<uint32_t>(n >> 3) << 17) | (static_cast<uint32_t>(m >> 4) << 24);
}

template <bool CI4>
__global__ void __launch_bounds__(BM_THREADS, 1)
beamform_kernel(const __grid_constant__ CUtensorMap xmap, const __grid_constant__ CUtensorMap wmap, const BmParams p)
{
    constexpr int KS = CI4 ? 256 : 128;        // int8 K bytes per stage (128 span bytes)
    constexpr int KH = KS / 128;               // 128-byte K tiles per stage
    constexpr int A_TILE = BM_MT * 128;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t w_tile = static_cast<uint32_t>(p.nb2) * 128u;
    const int kh = CI4 ? KH : p.pw;             // 128-byte K tiles per stage
    const uint32_t stage_bytes = kh * (A_TILE + w_tile);
    const int S = p.stages;
    const int R = p.raw_stages;
    const uint32_t raw_base = smem_base + S * stage_bytes;      // [R] raw ci4 tiles [128 samples][128 bytes]
    const uint32_t stg_base = raw_base + R * A_TILE;            // epilogue staging, one buffer per warp
    const uint32_t bar_base = stg_base + BM_STG_BYTES;
    const uint32_t bar_full = bar_base;                          // [S] span tile written + weight boxes landed
    const uint32_t bar_empty = bar_full + 8 * BM_MAX_STAGES;     // [S] MMAs reading the stage have completed
    const uint32_t bar_tfull = bar_empty + 8 * BM_MAX_STAGES;    // [2] accumulator complete
    const uint32_t bar_tempty = bar_tfull + 16;                  // [2] accumulator drained
    const uint32_t bar_rfull = bar_tempty + 16;                  // [R] raw bytes landed
    const uint32_t bar_rempty = bar_rfull + 8 * BM_MAX_RAW;      // [R] raw bytes consumed by the widening warps
    const uint32_t tmem_slot = bar_rempty + 8 * BM_MAX_RAW;

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&xmap);
        ptx::prefetch_tensormap(&wmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, CI4 ? BM_LOAD_WARPS + 1 : 1);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int s = 0; s < R; ++s) {
            ptx::mbar_init(bar_rfull + 8 * s, 1);
            ptx::mbar_init(bar_rempty + 8 * s, BM_LOAD_WARPS);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(bar_tfull + 8 * b, 1);
            ptx::mbar_init(bar_tempty + 8 * b, 4);
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<1>(tmem_slot, 512);
        ptx::tmem_relinquish<1>();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const long long u0 = blockIdx.x, ustep = gridDim.x;

    if (warp == 0) {
        // ===================== span producer (converged warp, lane 0 issues); ci8: the weights too =====================
        // the span is read once (evict first); a group's weights are re-read by every sample block (evict last)
        const uint64_t pol_first = ptx::policy_evict_first(), pol_last = ptx::policy_evict_last();
        uint32_t stage = 0, phase = 0;
        const uint32_t nst = CI4 ? static_cast<uint32_t>(R) : static_cast<uint32_t>(S);
        for (long long u = u0; u < p.nunits; u += ustep) {
            const BmUnit un = bm_decode(p, u);
            for (int ks = 0; ks < p.nks; ++ks) {
                if (CI4) {
                    ptx::mbar_wait(bar_rempty + 8 * stage, phase ^ 1);
                    if (lane == 0) {
                        ptx::mbar_expect_tx(bar_rfull + 8 * stage, A_TILE);
                        ptx::tma_load_3d_hint(raw_base + stage * A_TILE, &xmap, bar_rfull + 8 * stage, ks * 128, un.c, un.t0, pol_first);
                    }
                } else {
                    ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    if (lane == 0) {
                        const uint32_t dst = smem_base + stage * stage_bytes;
                        ptx::mbar_expect_tx(bar_full + 8 * stage, kh * (A_TILE + w_tile));
                        if (p.pw == 1) {
                            ptx::tma_load_3d_hint(dst, &xmap, bar_full + 8 * stage, ks * 128, un.c, un.t0, pol_first);
                        } else {
                            // 5-d view of the span {128 B, 8 samples, row pieces, channels, 8-sample groups}, box {128, 8, pw, 1, 16}:
                            // the requests of one 8-sample group walk the SAME eight pages once per piece, which the memory
                            // system serves faster than a new page per request (profiles/round2.md: 650 against 842 cycles per
                            // 16 KiB with every SM loading).  In shared memory piece h is the canonical K-major tile with its
                            // 8-row atoms pw KiB apart.
                            ptx::tma_load_5d_hint(dst, &xmap, bar_full + 8 * stage, 0, 0, ks * p.pw, un.c, un.t0 >> 3, pol_first);
                        }
                        for (int h = 0; h < kh; ++h)
                            ptx::tma_load_2d_hint(dst + kh * A_TILE + h * w_tile, &wmap, bar_full + 8 * stage, (ks * kh + h) * 128, un.c * p.nb2, pol_last);
                    }
                }
                __syncwarp();
                if (++stage == nst) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 3) {
        // ===================== weight producer, ci4 (converged warp, lane 0 issues) =====================
        if (CI4) {
            const uint64_t pol_last = ptx::policy_evict_last();
            uint32_t stage = 0, phase = 0;
            for (long long u = u0; u < p.nunits; u += ustep) {
                const BmUnit un = bm_decode(p, u);
                for (int ks = 0; ks < p.nks; ++ks) {
                    ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    if (lane == 0) {
                        const uint32_t dst = smem_base + stage * stage_bytes + KH * A_TILE;
                        ptx::mbar_expect_tx(bar_full + 8 * stage, KH * w_tile);
#pragma unroll
                        for (int h = 0; h < KH; ++h)
                            ptx::tma_load_2d_hint(dst + h * w_tile, &wmap, bar_full + 8 * stage, ks * KS + h * 128, un.c * p.nb2, pol_last);
                    }
                    __syncwarp();
                    if (++stage == static_cast<uint32_t>(S)) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (converged warp, lane 0 issues) =====================
        uint32_t stage = 0, phase = 0, it = 0;
        const uint32_t idesc = bm_instr_desc(BM_MT, p.nb2);
        for (long long u = u0; u < p.nunits; u += ustep, ++it) {
            const uint32_t b = it & 1;
            ptx::mbar_wait(bar_tempty + 8 * b, ((it >> 1) & 1) ^ 1);
            ptx::tc_fence_after();
            for (int ks = 0; ks < p.nks; ++ks) {
                ptx::mbar_wait(bar_full + 8 * stage, phase);
                ptx::tc_fence_after();
                if (lane == 0) {
                    const uint32_t abase = smem_base + stage * stage_bytes;
                    const uint32_t wbase = abase + kh * A_TILE;
                    for (int h = 0; h < kh; ++h) {
                        // ci4: dense tiles one after the other; ci8: piece h of the span box (atoms kh KiB apart; kh = 1: dense)
                        const uint64_t adesc = CI4 ? bm_smem_desc(abase + h * A_TILE) : bm_smem_desc(abase + h * 1024u, kh * 1024u);
                        const uint64_t bdesc = bm_smem_desc(wbase + h * w_tile);
#pragma unroll
                        for (int k = 0; k < 4; ++k)
                            ptx::mma_i8<1>(tmem_base + 256 * b, adesc + 2u * k, bdesc + 2u * k, idesc, (ks | h | k) != 0 ? 1u : 0u);
                    }
                    ptx::mma_commit(bar_empty + 8 * stage);
                }
                __syncwarp();
                if (++stage == static_cast<uint32_t>(S)) { stage = 0; phase ^= 1; }
            }
            if (lane == 0) ptx::mma_commit(bar_tfull + 8 * b);
            __syncwarp();
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue: one sample row per thread =====================
        const int wq = warp - 4;
        uint32_t it = 0;
        const bool vec4 = (p.nbeam & 1) == 0;
        const uint32_t stg_warp = stg_base + wq * BM_STG_WARP;
        for (long long u = u0; u < p.nunits; u += ustep, ++it) {
            const BmUnit un = bm_decode(p, u);
            const uint32_t b = it & 1;
            ptx::mbar_wait(bar_tfull + 8 * b, (it >> 1) & 1);
            ptx::tc_fence_after();
            const int t = un.t0 + 32 * wq + static_cast<int>(lane);
            int32_t* const orow = p.out + 2 * ((static_cast<long long>(t) * p.nchan + un.c) * p.nbeam);
            const int nrows = p.ntime - (un.t0 + 32 * wq);   // rows of this warp that exist
            // this sample's Sr, Si (columns 2 nbeam, 2 nbeam + 1): the offsets carried by every beam column
            uint32_t sr, si;
            ptx::tmem_ld_32x32b_x2(tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + 256 * b + 2 * p.nbeam, sr, si);
            ptx::tmem_ld_wait();
            const uint32_t off_re = 128u * sr + 127u * si, off_im = 128u * (sr + si);
            for (int col = 0; col < 2 * p.nbeam; col += 32) {
                uint32_t r[32];
                ptx::tmem_ld_32x32b_x32(tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + 256 * b + col, r);
                ptx::tmem_ld_wait();
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    r[j] -= (j & 1) ? off_im : off_re;   // exact in wrapping int32: the true beam fits (|b| < 2^31)
                    if (CI4) r[j] = static_cast<uint32_t>(static_cast<int32_t>(r[j]) >> 4);   // x was widened as 16 x
                }
                {
                    if (vec4) {
                        // through shared memory so that eight lanes write one row's 128 contiguous bytes
                        const uint32_t srow = stg_warp + lane * BM_STG_PITCH;
#pragma unroll
                        for (int j = 0; j < 32; j += 4)
                            asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(srow + 4 * j), "r"(r[j]), "r"(r[j + 1]),
                                         "r"(r[j + 2]), "r"(r[j + 3])
                                         : "memory");
                        __syncwarp();
                        const int piece = static_cast<int>(lane) & 7, npiece = (2 * p.nbeam - col + 3) >> 2;
                        int32_t* const obase = p.out + 2 * ((static_cast<long long>(un.t0 + 32 * wq) * p.nchan + un.c) * p.nbeam) + col + 4 * piece;
                        const long long rstride = 2ll * p.nchan * p.nbeam;
#pragma unroll
                        for (int i = 0; i < 8; ++i) {
                            const int row = 4 * i + (static_cast<int>(lane) >> 3);
                            if (row < nrows && piece < npiece) {
                                uint4 v;
                                asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                             : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w)
                                             : "r"(stg_warp + row * BM_STG_PITCH + piece * 16));
                                ptx::st_global_v4(reinterpret_cast<uint8_t*>(obase + row * rstride), v);
                            }
                        }
                        __syncwarp();
                    } else if (static_cast<int>(lane) < nrows) {
#pragma unroll
                        for (int j = 0; j < 32; j += 2)
                            if (col + j < 2 * p.nbeam)
                                ptx::st_global_v2(orow + col + j, make_int2(static_cast<int>(r[j]), static_cast<int>(r[j + 1])));
                    }
                }
            }
            ptx::tc_fence_before();
            __syncwarp();
            if (lane == 0) ptx::mbar_arrive(bar_tempty + 8 * b);
        }
    } else if (warp >= 8) {
        // ===================== ci4: raw rows -> swizzled K-major int8 tiles =====================
        // vector v = i * 256 + tid of a stage: sample row v >> 3, 16-byte chunk v & 7 of the row's 128 raw bytes (16
        // samples), widened to chunks 2 * chunk and 2 * chunk + 1 of the row's 256 int8 bytes
        if (CI4) {
            const int tid = static_cast<int>(threadIdx.x) - 256;
            const int chunk = tid & 7;
            uint32_t rstage = 0, rphase = 0, stage = 0, phase = 0;
            for (long long u = u0; u < p.nunits; u += ustep) {
                for (int ks = 0; ks < p.nks; ++ks) {
                    ptx::mbar_wait(bar_rfull + 8 * rstage, rphase);
                    ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                    const uint32_t rsrc = raw_base + rstage * A_TILE;
                    const uint32_t abase = smem_base + stage * stage_bytes;
#pragma unroll
                    for (int i = 0; i < 4; ++i) {
                        const int rowi = i * 32 + (tid >> 3);
                        uint4 w;
                        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                     : "=r"(w.x), "=r"(w.y), "=r"(w.z), "=r"(w.w)
                                     : "r"(rsrc + rowi * 128 + chunk * 16));
                        const uint32_t tile = abase + rowi * 128 + (chunk >> 2) * A_TILE;
                        const uint32_t j0 = static_cast<uint32_t>(2 * chunk) & 7u;
                        const uint32_t a0 = tile + ((j0 ^ (rowi & 7)) << 4), a1 = tile + (((j0 + 1) ^ (rowi & 7)) << 4);
                        // chunks c and c + 4 of a row fall on the same banks (different K tiles): the upper four lanes of
                        // a row write their odd chunk first, so every store covers all 32 banks once
                        const bool hi = (chunk & 4) != 0;
                        const uint32_t e0 = w.x & 0xF0F0F0F0u, e1 = (w.x << 4) & 0xF0F0F0F0u, e2 = w.y & 0xF0F0F0F0u, e3 = (w.y << 4) & 0xF0F0F0F0u;
                        const uint32_t o0 = w.z & 0xF0F0F0F0u, o1 = (w.z << 4) & 0xF0F0F0F0u, o2 = w.w & 0xF0F0F0F0u, o3 = (w.w << 4) & 0xF0F0F0F0u;
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(hi ? a1 : a0), "r"(hi ? o0 : e0), "r"(hi ? o1 : e1),
                                     "r"(hi ? o2 : e2), "r"(hi ? o3 : e3)
                                     : "memory");
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(hi ? a0 : a1), "r"(hi ? e0 : o0), "r"(hi ? e1 : o1),
                                     "r"(hi ? e2 : o2), "r"(hi ? e3 : o3)
                                     : "memory");
                    }
                    ptx::fence_proxy_async_smem();  // generic-proxy stores -> visible to the tensor core (async proxy)
                    __syncwarp();
                    if (lane == 0) {
                        ptx::mbar_arrive(bar_rempty + 8 * rstage);
                        ptx::mbar_arrive(bar_full + 8 * stage);
                    }
                    if (++rstage == static_cast<uint32_t>(R)) { rstage = 0; rphase ^= 1; }
                    if (++stage == static_cast<uint32_t>(S)) { stage = 0; phase ^= 1; }
                }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, 512);
}

// bfBeamformSetWeights: w[c][k][i] (ci8) -> W[c][n][kk] uint8, n = 2k + part of b for the beams, n = 2 nbeam, 2 nbeam + 1
// the selector rows, kk in the order the loaders write the span bytes (header comment); the other rows, and the columns
// beyond the inputs, are zero (the span reads as zero there too).
template <bool CI4>
__global__ void beamform_weights_kernel(const int8_t* __restrict__ w, uint8_t* __restrict__ wp, int ninputs, int nchan, int nbeam,
                                        int nb2, int kp)
{
    const long long total = static_cast<long long>(nchan) * nb2 * kp;
    for (long long q = blockIdx.x * static_cast<long long>(blockDim.x) + threadIdx.x; q < total;
         q += static_cast<long long>(gridDim.x) * blockDim.x) {
        const int kk = static_cast<int>(q % kp);
        const long long cn = q / kp;
        const int n = static_cast<int>(cn % nb2), c = static_cast<int>(cn / nb2);
        const int k = n >> 1, bpart = n & 1;
        int i, xpart;
        if (CI4) {
            i = 4 * (kk >> 3) + (kk & 3);
            xpart = (kk >> 2) & 1;
        } else {
            i = kk >> 1;
            xpart = kk & 1;
        }
        int v = 0;
        if (i < ninputs) {
            if (k < nbeam) {
                const int8_t* s = w + 2 * ((static_cast<long long>(c) * nbeam + k) * ninputs + i);
                const int wr = s[0], wi = s[1];
                v = bpart == 0 ? (xpart == 0 ? wr + 128 : 127 - wi) : (xpart == 0 ? wi + 128 : wr + 128);
            } else if (k == nbeam) {
                v = bpart == xpart ? 1 : 0;   // row 2 nbeam selects the re components, row 2 nbeam + 1 the im components
            }
        }
        wp[q] = static_cast<uint8_t>(v);
    }
}

}  // namespace bfx
