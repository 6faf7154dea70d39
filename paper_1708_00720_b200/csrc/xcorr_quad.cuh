// xcorr_quad.cuh -- the CTA-pair contraction of xcorr_pair.cuh run in clusters of FOUR CTAs (two pairs) that work
// on two tiles of the same 128-input row block at once, so that the row block's operand (the A-halves) is read
// from the L2 once and delivered to both pairs by TMA multicast.  The pair kernel is bound by L2 throughput
// (profiles/round1.md); per two tiles this moves 6 boxes through the L2 instead of 8.
//
// A job = two tiles.  "Shared" jobs: tiles (R, 2j) on pair 0 and (R, 2j + 1) on pair 1; CTA r of pair 0 loads
// A-half(R, r) with a multicast to CTA r of both pairs, every CTA loads its own B-half (none on a diagonal tile,
// where B-half = A-half).  Rows with an even R have one tile left over, the diagonal one; two such tiles (rows
// 4m and 4m + 2) form an "unshared" job in which every CTA loads just its own A-half.  A lone leftover leaves
// pair 1 idle for one job.  Both pairs walk the same shared-memory stages in lockstep: every CTA's "stage free"
// barrier collects the MMA commits of BOTH pair leaders, because a multicast load writes into both pairs.
//
// Everything else (S1 relayout ring and flags, TMEM double buffering, epilogue) is as in xcorr_pair.cuh.
#pragma once
#include "xcorr_pair.cuh"

namespace bfx {

struct QdJob {
    int c;          // channel
    int active;     // this pair has a tile in the job
    int shared;     // the two tiles share their row block (A multicast)
    int R, Cb;      // this pair's tile
};

// jobs of a channel: first the shared ones, row-major (row R has (R + 1) / 2 of them), then the unshared ones
__device__ __forceinline__ QdJob qd_decode(long long w, const TcParams& p, int pair)
{
    const uint32_t wu = static_cast<uint32_t>(w), jpc = static_cast<uint32_t>(p.qd_jobs_per_chan);
    const uint32_t c = wu / jpc;
    int q = static_cast<int>(wu - c * jpc);
    QdJob jb;
    jb.c = static_cast<int>(c);
    if (q < p.qd_nshared) {
        int R = 1;
        while (q >= (R + 1) / 2) { q -= (R + 1) / 2; ++R; }
        jb.active = 1;
        jb.shared = 1;
        jb.R = R;
        jb.Cb = 2 * q + pair;
    } else {
        const int R = 4 * (q - p.qd_nshared) + 2 * pair;  // leftover diagonal tiles of the even rows
        jb.active = R < p.qd_nb ? 1 : 0;
        jb.shared = 0;
        jb.R = R;
        jb.Cb = R;
    }
    return jb;
}

__device__ __forceinline__ void qd_tma_load_mc(uint32_t dst, const CUtensorMap* m, uint32_t bar, int x, int y, int z, uint16_t mask,
                                               uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.multicast::cluster.cta_group::2"
        ".L2::cache_hint [%0], [%1, {%3, %4, %5}], [%2], %6, %7;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(x), "r"(y), "r"(z), "h"(mask), "l"(pol)
        : "memory");
}

__global__ void __launch_bounds__(PR_THREADS, 1)
xcorr_quad_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int S = PR_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t op_base = smem_base;                         // S stages of (A-half, B-half)
    const uint32_t stg_base = op_base + S * PR_STAGE_BYTES;     // epilogue staging
    const uint32_t bar_base = stg_base + TC_STG_BYTES;
    const uint32_t bar_full = bar_base;                  // [S]  pair leader: all operand boxes of the pair have landed
    const uint32_t bar_empty = bar_full + 8 * S;         // [S]  every CTA: BOTH pair leaders' MMAs on the stage are done
    const uint32_t bar_tfull = bar_empty + 8 * S;        // [2]  accumulator complete (own pair)
    const uint32_t bar_tempty = bar_tfull + 16;          // [2]  pair leader: drained by the 8 epilogue warps of the pair
    const uint32_t tmem_slot = bar_tempty + 16;
    const uint32_t bar_sfull = tmem_slot + 8;            // [TC_RING] job index published
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING; // [TC_RING] cluster leader: all consumer roles of the 4 CTAs read it
    const uint32_t ring_base = bar_sempty + 8 * TC_RING;

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();
    const uint32_t rank = ptx::cluster_ctarank();        // 0..3
    const int pr = static_cast<int>(rank & 1);           // CTA within its pair (0 = pair leader)
    const int pair = static_cast<int>(rank >> 1);
    const bool leader = pr == 0;
    const bool cleader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, 1);
            ptx::mbar_init(bar_empty + 8 * s, 2);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(bar_tfull + 8 * b, 1);
            ptx::mbar_init(bar_tempty + 8 * b, 8);
        }
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            // rank 0: MMA + 4 epilogue; rank 1: producer + 4; rank 2: producer + MMA + 4; rank 3: producer + 4
            ptx::mbar_init(bar_sempty + 8 * s, 21);
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<2>(tmem_slot, TC_TMEM_COLS);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const int nkb = (p.ntime + TC_KT - 1) / TC_KT;
    const PrRing ring{bar_sfull, ring_base, ptx::mapa(bar_sempty, 0)};
    const uint32_t lead_full = ptx::mapa(bar_full, rank & ~1u);
    const uint32_t lead_tempty = ptx::mapa(bar_tempty, rank & ~1u);
    const uint16_t pair_mask = static_cast<uint16_t>(3u << (2 * pair));

    if (warp == 0) {
        // ===================== TMA producer (+ job scheduler in the cluster leader) =====================
        uint32_t stage = 0, phase = 0;
        int ready_chan = -1;
        const uint64_t pol_last = ptx::policy_evict_last();
        unsigned long long w_next = 0;
        if (cleader) {
            if (lane == 0) w_next = atomicAdd(p.sched, 1ull);
            w_next = __shfl_sync(0xffffffffu, w_next, 0);
        }
        for (uint32_t n = 0;; ++n) {
            long long w;
            if (cleader) {
                const uint32_t slot = n % TC_RING;
                ptx::mbar_wait(bar_sempty + 8 * slot, ((n / TC_RING) & 1) ^ 1);
                w = static_cast<long long>(w_next);
                if (w >= p.ntiles) w = -1;
                if (lane == 0) {
                    if (w >= 0) w_next = atomicAdd(p.sched, 1ull);
                    asm volatile("st.shared.s64 [%0], %1;" ::"r"(ring_base + 8 * slot), "l"(w) : "memory");
                    ptx::mbar_arrive(bar_sfull + 8 * slot);
                    for (uint32_t d = 1; d < 4; ++d) {
                        asm volatile("st.shared::cluster.s64 [%0], %1;" ::"r"(ptx::mapa(ring_base + 8 * slot, d)), "l"(w) : "memory");
                        ptx::mbar_arrive_cluster(bar_sfull + 8 * slot, d);
                    }
                }
                w_next = __shfl_sync(0xffffffffu, w_next, 0);
            } else {
                w = __shfl_sync(0xffffffffu, ring.get<true>(n, lane), 0);
            }
            if (w < 0) break;
            const QdJob jb = qd_decode(w, p, pair);
            const int c = jb.c;
            if (c != ready_chan) {
                if (lane == 0) {
                    const unsigned long long want = p.epoch * static_cast<unsigned long long>(p.rl_units);
                    uint32_t spins = 0;
                    while (ptx::ld_acquire_u64(p.ready + c) < want)
                        if (++spins > (1u << 26)) __trap();
                    ptx::fence_proxy_async_global();
                }
                __syncwarp();
                ready_chan = c;
            }
            const int cs = c % p.ring_w;
            const bool diag = jb.R == jb.Cb;
            const int xa = 256 * jb.R + 128 * pr;
            const int xb = 256 * jb.Cb + 128 * pr;
            // bytes landing in this pair's two CTAs per stage: the A-halves (own loads or pair 0's multicast) and the
            // B-halves unless the tile is diagonal
            const uint32_t pair_bytes = jb.active ? (diag ? 2u : 4u) * TC_BOX_BYTES : 0u;
            const bool load_a = jb.active && (!jb.shared || pair == 0);
            const bool load_b = jb.active && !diag;
            const uint16_t a_mask = jb.shared ? static_cast<uint16_t>(5u << pr) : static_cast<uint16_t>(1u << rank);
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                if (lane == 0) {
                    if (leader && jb.active) ptx::mbar_expect_tx(bar_full + 8 * stage, pair_bytes);
                    const uint32_t dst = op_base + stage * PR_STAGE_BYTES;
                    const uint32_t fullb = lead_full + 8 * stage;
                    const int t0 = kb * TC_KT;
                    if (load_a) qd_tma_load_mc(dst, &tmap, fullb, xa, cs, t0, a_mask, pol_last);
                    if (load_b) ptx::tma_load_3d_cg2_hint(dst + TC_BOX_BYTES, &tmap, fullb, xb, cs, t0, pol_last);
                }
                __syncwarp();
                if (++stage == S) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (S3), pair leaders =====================
        if (leader) {
            uint32_t stage = 0, phase = 0, it = 0;
            const uint32_t idesc = tc_instr_desc(256, 256);
            for (uint32_t n = 0;; ++n) {
                const long long w = __shfl_sync(0xffffffffu, ring.get<true>(n, lane), 0);
                if (w < 0) break;
                const QdJob jb = qd_decode(w, p, pair);
                if (!jb.active) {
                    // idle pair: keep the lockstep -- release every stage once per use, as an MMA commit would
                    for (int kb = 0; kb < nkb; ++kb) {
                        ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                        if (lane == 0) ptx::mma_commit_cg2(bar_empty + 8 * stage, 0xF);
                        __syncwarp();
                        if (++stage == S) { stage = 0; phase ^= 1; }
                    }
                    continue;
                }
                const bool diag = jb.R == jb.Cb;
                const uint32_t buf = it & 1, bphase = (it >> 1) & 1;
                const uint32_t d_tmem = tmem_base + buf * 256;
                ptx::mbar_wait(bar_tempty + 8 * buf, bphase ^ 1);
                ptx::tc_fence_after();
                for (int kb = 0; kb < nkb; ++kb) {
                    ptx::mbar_wait(bar_full + 8 * stage, phase);
                    ptx::tc_fence_after();
                    const uint32_t sbase = op_base + stage * PR_STAGE_BYTES;
                    const uint64_t adesc = tc_smem_desc(sbase, TC_BOX_BYTES);
                    const uint64_t bdesc = tc_smem_desc(diag ? sbase : sbase + TC_BOX_BYTES, TC_BOX_BYTES);
                    const int trem = p.ntime - kb * TC_KT;
                    const int nk = trem >= TC_KT ? TC_KT / 32 : (trem + 31) / 32;
                    if (lane == 0) {
                        for (int k = 0; k < nk; ++k)
                            ptx::mma_i8<2>(d_tmem, adesc + 256u * k, bdesc + 256u * k, idesc, (kb | k) != 0 ? 1u : 0u);
                        ptx::mma_commit_cg2(bar_empty + 8 * stage, 0xF);  // frees the stage in all four CTAs
                    }
                    __syncwarp();
                    if (++stage == S) { stage = 0; phase ^= 1; }
                }
                if (lane == 0) {
                    ptx::mma_commit_cg2(bar_tfull + 8 * buf, pair_mask);
                    ptx::red_relaxed_add_u64(p.done + jb.c, 1ull);
                }
                __syncwarp();
                ++it;
            }
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue (S4), all CTAs =====================
        const int wq = warp - 4;
        const uint32_t stg_warp = stg_base + wq * TC_STG_WARP_BYTES;
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        uint32_t nchunks_done = 0, it = 0;
        for (uint32_t n = 0;; ++n) {
            const long long w = ring.get<true>(n, lane);
            if (w < 0) break;
            const QdJob jb = qd_decode(w, p, pair);
            if (!jb.active) continue;
            const int c = jb.c;
            const uint32_t buf = it & 1, bphase = (it >> 1) & 1;
            ++it;
            const int i0 = PR_BLK * jb.R + 64 * pr + 16 * wq;  // first input row of this warp
            const int j0 = PR_BLK * jb.Cb;
            int nchunk = (i0 + 15 - j0) / TC_CJ + 1;
            nchunk = nchunk > 2 ? 2 : nchunk;
            int32_t* const out_c = p.out + 2 * (static_cast<long long>(c) * nbl);
            if (p.accumulate && lane < 16) {
                const int i_own = i0 + static_cast<int>(lane);
                int nn = i_own + 1 - j0;
                nn = nn > PR_BLK ? PR_BLK : nn;
                if (i_own < p.ninputs && nn > 0) {
                    const long long e0 = static_cast<long long>(i_own) * (i_own + 1) / 2 + j0;
                    const long long ea = e0 & ~1ll, eb = (e0 + nn + 1) & ~1ll;
                    ptx::bulk_prefetch_l2(out_c + 2 * ea, static_cast<uint32_t>(8 * (eb - ea)));
                }
            }
            ptx::mbar_wait(bar_tfull + 8 * buf, bphase);
            ptx::tc_fence_after();
            for (int jc = 0; jc < nchunk; ++jc, ++nchunks_done) {
                const uint32_t stg_buf = stg_warp + (nchunks_done & 1) * TC_STG_BUF_BYTES;
                const uint32_t tcol = tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + buf * 256 + jc * 128;
                tc_epilogue_chunk<false, true>(p, lane, tcol, stg_buf, out_c, i0, j0 + jc * TC_CJ,
                                               jc == nchunk - 1 ? lead_tempty + 8 * buf : 0u);
            }
        }
        if (lane < 16) ptx::bulk_wait_read<0>();
    } else if (warp >= 8) {
        tc_relayout_role(p, lane);
    }

    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();
    if (warp == 2) ptx::tmem_dealloc<2>(tmem_base, TC_TMEM_COLS);
    if (threadIdx.x == 0 && atomicAdd(p.sched + 1, 1ull) == gridDim.x - 1) {
        p.sched[0] = 0;
        p.sched[1] = 0;
        p.sched[2] = 0;
    }
}

}  // namespace bfx
