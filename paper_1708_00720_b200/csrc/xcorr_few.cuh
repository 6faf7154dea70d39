// xcorr_few.cuh -- few-input spans (ninputs <= 64: one 64 x 64-input tile per channel), the bandwidth-bound case
// of BASELINE.json configs[4].  Every sample is used by exactly one tile, so there is no re-read to save and the
// span is consumed in place; what limits a per-channel kernel is address translation and DRAM locality: a
// channel's samples are 64..128-byte pieces lying nchan*row bytes (1 MiB on cfg5) apart, and the TMA unit
// delivered 6.5 B/clk/SM on them (profiles/round1.md).  Here one CTA contracts FW_NC = 4 ADJACENT channels at
// once, so each TMA box row is a contiguous run of 4 rows and the translations per byte drop fourfold; the four
// 128-lane x 128-column accumulators fill the CTA's 512 TMEM columns.
//
// Roles (512 threads): warp 0 TMA producer (raw bytes, box {row bytes, 4 channels, FW_KT samples}), warp 1 MMA
// issuer (per channel: A = B = the channel's int8 tile, M = 128, N = 128), warp 2 TMEM allocator, warps 4..7
// epilogue (tc_epilogue_chunk, one 64-visibility chunk per channel), warps 8..15 unpack: raw [t][c][row] bytes ->
// per-channel 128B-swizzled int8 tiles (ci4: nibble << 4, the 16 x 16 scale is shifted out exactly in the
// epilogue; ci8: a swizzling copy).
#pragma once
#include "xcorr_common.cuh"

namespace bfx {

constexpr int FW_NC = 4;     // channels per CTA tile
constexpr int FW_KT = 64;    // samples per stage
constexpr int FW_OP_TILE_BYTES = FW_KT * 128;             // one channel: [t][128 B] swizzled
constexpr int FW_OP_STAGE_BYTES = FW_NC * FW_OP_TILE_BYTES;
constexpr int FW_UNPACK_WARPS = 8;
#ifndef BFX_FW_STG_BUFS
#define BFX_FW_STG_BUFS 1
#endif
constexpr int FW_STG_BUFS = BFX_FW_STG_BUFS;          // epilogue staging buffers per warp (1: more room for span stages)
constexpr int FW_STG_BYTES = 4 * FW_STG_BUFS * TC_STG_BUF_BYTES;
constexpr int FW_THREADS = 256 + 32 * FW_UNPACK_WARPS;

template <bool CI4>
struct FwCfg {
    static constexpr int kRawRow = CI4 ? 64 : 128;                     // bytes of a 64-input raw row
    static constexpr int kRawStageBytes = FW_KT * FW_NC * kRawRow;     // [t][c][<= kRawRow]
#ifndef BFX_FW_RAW4
#define BFX_FW_RAW4 4
#endif
#ifndef BFX_FW_OP4
#define BFX_FW_OP4 4
#endif
    static constexpr int kRawStages = CI4 ? BFX_FW_RAW4 : 2, kOpStages = CI4 ? BFX_FW_OP4 : 2;
    static constexpr int kSmemBytes = 1024 + kRawStages * kRawStageBytes + kOpStages * FW_OP_STAGE_BYTES + FW_STG_BYTES + 512;
};

template <bool CI4>
__global__ void __launch_bounds__(FW_THREADS, 1)
xcorr_few_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int R = FwCfg<CI4>::kRawStages, S = FwCfg<CI4>::kOpStages;
    constexpr int FW_RAW_STAGE_BYTES = FwCfg<CI4>::kRawStageBytes;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t op_base = smem_base;
    const uint32_t raw_base = op_base + S * FW_OP_STAGE_BYTES;
    const uint32_t stg_base = raw_base + R * FW_RAW_STAGE_BYTES;
    const uint32_t bar_base = stg_base + FW_STG_BYTES;
    const uint32_t bar_full = bar_base;               // [S] int8 tiles written by the unpack warps
    const uint32_t bar_empty = bar_full + 8 * S;      // [S] MMAs reading the stage have completed
    const uint32_t bar_rfull = bar_empty + 8 * S;     // [R] raw bytes landed
    const uint32_t bar_rempty = bar_rfull + 8 * R;    // [R] raw bytes consumed by the unpack warps
    const uint32_t bar_tfull = bar_rempty + 8 * R;    // accumulators complete
    const uint32_t bar_tempty = bar_tfull + 8;        // accumulators drained by the 4 epilogue warps
    const uint32_t tmem_slot = bar_tempty + 8;
    const uint32_t bar_sfull = tmem_slot + 8;
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING;
    const uint32_t ring_base = bar_sempty + 8 * TC_RING;

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();
    const int row = p.row_in;  // bytes per (t, c): ninputs (ci4) or 2 * ninputs (ci8), a multiple of 16

    // the int8 tiles are 128 bytes wide; with fewer than 64 inputs the unpack warps never touch the right part
    for (uint32_t o = threadIdx.x * 16; o < S * FW_OP_STAGE_BYTES; o += FW_THREADS * 16)
        asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(op_base + o), "r"(0) : "memory");
    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, FW_UNPACK_WARPS);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int s = 0; s < R; ++s) {
            ptx::mbar_init(bar_rfull + 8 * s, 1);
            ptx::mbar_init(bar_rempty + 8 * s, FW_UNPACK_WARPS);
        }
        ptx::mbar_init(bar_tfull, 1);
        ptx::mbar_init(bar_tempty, 4);
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            ptx::mbar_init(bar_sempty + 8 * s, 5 + FW_UNPACK_WARPS);  // MMA issuer + 4 epilogue warps + unpack warps
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<1>(tmem_slot, TC_TMEM_COLS);
        ptx::tmem_relinquish<1>();
    }
    ptx::fence_proxy_async_smem();  // the zero fill above is read by the tensor core
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const int nkb = (p.ntime + FW_KT - 1) / FW_KT;
    const TcRing ring{bar_sfull, bar_sempty, ring_base};

    if (warp == 0) {
        // ===================== TMA producer + tile scheduler (converged warp, lane 0 issues) =====================
        uint32_t stage = 0, phase = 0;
        unsigned long long w_next = 0;
        if (lane == 0) w_next = atomicAdd(p.sched, 1ull);
        w_next = __shfl_sync(0xffffffffu, w_next, 0);
        const uint32_t stage_tx = static_cast<uint32_t>(FW_KT * FW_NC * row);
        for (uint32_t n = 0;; ++n) {
            ring.wait_free(n);
            long long w = static_cast<long long>(w_next);
            if (w >= p.ntiles) w = -1;
            if (lane == 0) {
                if (w >= 0) w_next = atomicAdd(p.sched, 1ull);
                ring.publish(n, w);
            }
            w_next = __shfl_sync(0xffffffffu, w_next, 0);
            if (w < 0) break;
            const int c0 = static_cast<int>(w) * FW_NC;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rempty + 8 * stage, phase ^ 1);
                if (lane == 0) {
                    ptx::mbar_expect_tx(bar_rfull + 8 * stage, stage_tx);
                    ptx::tma_load_3d(raw_base + stage * FW_RAW_STAGE_BYTES, &tmap, bar_rfull + 8 * stage, 0, c0, kb * FW_KT);
                }
                __syncwarp();
                if (++stage == R) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (converged warp, lane 0 issues) =====================
        uint32_t stage = 0, phase = 0;
        const uint32_t idesc = tc_instr_desc(128, 128);
        for (uint32_t it = 0;; ++it) {
            const long long w = __shfl_sync(0xffffffffu, ring.get<true>(it, lane), 0);
            if (w < 0) break;
            ptx::mbar_wait(bar_tempty, (it & 1) ^ 1);
            ptx::tc_fence_after();
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_full + 8 * stage, phase);
                ptx::tc_fence_after();
                const uint32_t sbase = op_base + stage * FW_OP_STAGE_BYTES;
                const int trem = p.ntime - kb * FW_KT;
                const int nk = trem >= FW_KT ? FW_KT / 32 : (trem + 31) / 32;
                if (lane == 0) {
#pragma unroll
                    for (int ch = 0; ch < FW_NC; ++ch) {
                        // V[c] = x x^H: both operands are the channel's own tile
                        const uint64_t desc = tc_smem_desc(sbase + ch * FW_OP_TILE_BYTES, FW_OP_TILE_BYTES);
                        for (int k = 0; k < nk; ++k)
                            ptx::mma_i8<1>(tmem_base + 128 * ch, desc + 256u * k, desc + 256u * k, idesc, (kb | k) != 0 ? 1u : 0u);
                    }
                    ptx::mma_commit(bar_empty + 8 * stage);
                }
                __syncwarp();
                if (++stage == S) { stage = 0; phase ^= 1; }
            }
            if (lane == 0) ptx::mma_commit(bar_tfull);
            __syncwarp();
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue (S4): one 64-visibility chunk per channel =====================
        const int wq = warp - 4;
        const uint32_t stg_warp = stg_base + wq * FW_STG_BUFS * TC_STG_BUF_BYTES;
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        uint32_t nchunks_done = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const int c0 = static_cast<int>(w) * FW_NC;
            ptx::mbar_wait(bar_tfull, it & 1);
            ptx::tc_fence_after();
            // rows of this warp that exist at all (ninputs may be < 64); TMEM must be released either way
            const bool any = 16 * wq < p.ninputs;
            int nch = p.nchan - c0;
            nch = nch > FW_NC ? FW_NC : nch;
            if (!any) nch = 0;
            for (int ch = 0; ch < nch; ++ch, ++nchunks_done) {
                const uint32_t stg_buf = stg_warp + (nchunks_done % FW_STG_BUFS) * TC_STG_BUF_BYTES;
                const uint32_t tcol = tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + 128 * ch;
                int32_t* const out_c = p.out + 2 * (static_cast<long long>(c0 + ch) * nbl);
                tc_epilogue_chunk<CI4, false, FW_STG_BUFS - 1, CI4>(p, lane, tcol, stg_buf, out_c, 16 * wq, 0, ch == nch - 1 ? bar_tempty : 0u);
            }
            if (nch == 0) {
                ptx::tc_fence_before();
                __syncwarp();
                if (lane == 0) ptx::mbar_arrive(bar_tempty);
            }
        }
        if (lane < 16) ptx::bulk_wait_read<0>();  // shared memory must outlive the bulk reads
    } else if (warp >= 8) {
        // ===================== unpack warps (S1): raw [t][c][row] nibble bytes -> per-channel int8 tiles =====================
        // int8 tile: [t][128 B], 16-byte chunks XOR-swizzled by (t & 7) exactly as TMA SWIZZLE_128B would have written
        // them.  ci8: byte 2i = re_i, byte 2i+1 = im_i.  ci4: bytes 8g..8g+3 = re of inputs 4g..4g+3 (<< 4), bytes
        // 8g+4..8g+7 = their im (<< 4).
        // lane -> (row t, 16-byte chunk qc) of one channel; a quarter-warp writes whole swizzled rows, which touches
        // every bank once; no divisions on the way.  ci4: 4 chunks of 16 samples per row, each widened to two int8
        // chunks; ci8: 8 chunks per row, copied to their swizzled place.
        constexpr int QPR = CI4 ? 4 : 8;   // raw chunks per full row
        constexpr int RPW = 32 / QPR;      // rows per warp pass
        const int uw = warp - 8, tl = static_cast<int>(lane) / QPR, qc = static_cast<int>(lane) % QPR;
        const int qn = row >> 4;           // 16-byte chunks this span's rows really have
        uint32_t rstage = 0, rphase = 0, ostage = 0, ophase = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rfull + 8 * rstage, rphase);
                ptx::mbar_wait(bar_empty + 8 * ostage, ophase ^ 1);
                const uint32_t rsrc = raw_base + rstage * FW_RAW_STAGE_BYTES;
                const uint32_t odst = op_base + ostage * FW_OP_STAGE_BYTES;
#pragma unroll
                for (int ch = 0; ch < FW_NC; ++ch) {
#pragma unroll
                    for (int t = uw * RPW + tl; t < FW_KT; t += RPW * FW_UNPACK_WARPS) {
                        if (qc < qn) {
                            uint32_t wv[4];
                            asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                         : "=r"(wv[0]), "=r"(wv[1]), "=r"(wv[2]), "=r"(wv[3])
                                         : "r"(rsrc + (t * FW_NC + ch) * row + qc * 16));
                            const uint32_t rowa = odst + ch * FW_OP_TILE_BYTES + t * 128;
                            if (CI4) {
                                // grouped real embedding: the four re bytes of a word, then its four im bytes -- no byte
                                // permutes; tc_epilogue_chunk<..., GROUPED> pairs lanes and columns 4 apart
                                uint32_t o[8];
#pragma unroll
                                for (int u = 0; u < 4; ++u) {
                                    o[2 * u] = wv[u] & 0xF0F0F0F0u;                   // re0..re3, each << 4
                                    o[2 * u + 1] = (wv[u] << 4) & 0xF0F0F0F0u;        // im0..im3, each << 4
                                }
                                const uint32_t a0 = rowa + static_cast<uint32_t>((2 * qc) ^ (t & 7)) * 16;
                                const uint32_t a1 = rowa + static_cast<uint32_t>((2 * qc + 1) ^ (t & 7)) * 16;
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a0), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a1), "r"(o[4]), "r"(o[5]), "r"(o[6]), "r"(o[7]) : "memory");
                            } else {
                                const uint32_t a0 = rowa + static_cast<uint32_t>(qc ^ (t & 7)) * 16;
                                asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a0), "r"(wv[0]), "r"(wv[1]), "r"(wv[2]), "r"(wv[3]) : "memory");
                            }
                        }
                    }
                }
                ptx::fence_proxy_async_smem();  // generic-proxy stores -> visible to the tensor core (async proxy)
                __syncwarp();
                if (lane == 0) {
                    ptx::mbar_arrive(bar_rempty + 8 * rstage);
                    ptx::mbar_arrive(bar_full + 8 * ostage);
                }
                if (++rstage == R) { rstage = 0; rphase ^= 1; }
                if (++ostage == S) { ostage = 0; ophase ^= 1; }
            }
        }
    }

    ptx::tc_fence_before();
    __syncthreads();
    if (warp == 2) ptx::tmem_dealloc<1>(tmem_base, TC_TMEM_COLS);
    if (threadIdx.x == 0 && atomicAdd(p.sched + 1, 1ull) == gridDim.x - 1) {
        p.sched[0] = 0;
        p.sched[1] = 0;
        p.sched[2] = 0;
    }
}

}  // namespace bfx
