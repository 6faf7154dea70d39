// xcorr_pair.cuh -- the X-engine contraction on CTA pairs (tcgen05 cta_group::2), the product path for
// ninputs > 64.  Same method as xcorr_common.cuh (real Gram embedding, accumulators in TMEM for the whole
// span, S1 relayout warps feeding an L2-resident ring, S4 bulk store / L2 reduce-add epilogue); what changes
// is the tile: two CTAs of a cluster share one 128-input x 128-input tile,
//
//     CTA r (r = 0, 1) owns rows   [128 R + 64 r, +64)  -> its TMEM holds 128 lanes x 256 columns
//     and loads         A-half  =  inputs [128 R  + 64 r, +64)   (128 bytes per sample)
//                       B-half  =  inputs [128 Cb + 64 r, +64)   (the MMA reads N/2 columns from each CTA)
//
// so every CTA pulls two 8 KiB boxes per 64-sample stage from the L2 instead of three for the same MMA time
// (one box on diagonal tiles, where A-half == B-half), which is what bounds the 1-CTA kernel once S1 has
// removed the address-translation stall (profiles/round1.md).  One `tcgen05.mma.cta_group::2` of M = 256,
// N = 256, K = 32 is issued by the leader CTA (rank 0) per 32 samples; `tcgen05.commit ... multicast` frees the
// stage / publishes the accumulator in both CTAs.
//
// Warp roles (both CTAs unless noted): 0 TMA producer (the leader's also draws the tile index from the global
// counter and publishes it to both CTAs' rings), 1 MMA issuer (leader only), 2 TMEM allocator, 4..7 epilogue,
// 8..15 relayout (tc_relayout_role).
#pragma once
#include "xcorr_common.cuh"

namespace bfx {

constexpr int PR_BLK = 128;                         // inputs per tile edge
#ifndef BFX_PR_STAGES
#define BFX_PR_STAGES (8 * 64 / BFX_KT)
#endif
constexpr int PR_STAGES = BFX_PR_STAGES;
constexpr int PR_STAGE_BYTES = 2 * TC_BOX_BYTES;    // A-half, B-half
constexpr int PR_THREADS = 512;
constexpr int PR_SMEM_BYTES = 1024 + PR_STAGES * PR_STAGE_BYTES + TC_STG_BYTES + 512;

// S2 decode without touching memory: tile index w -> (channel c, row block R, column block Cb <= R), tiles of a
// channel enumerated row-major over the lower triangle of 128-input blocks: q = R (R + 1) / 2 + Cb.
struct PrWhere {
    int c, R, Cb;
};
__device__ __forceinline__ PrWhere pr_decode(long long w, int tiles_per_chan)
{
    const uint32_t wu = static_cast<uint32_t>(w), tpc = static_cast<uint32_t>(tiles_per_chan);  // ntiles < 2^32 (host-checked)
    const uint32_t c = wu / tpc, q = wu - c * tpc;
    int R = static_cast<int>((sqrtf(8.0f * static_cast<float>(q) + 1.0f) - 1.0f) * 0.5f);
    while (R * (R + 1) / 2 > static_cast<int>(q)) --R;
    while ((R + 1) * (R + 2) / 2 <= static_cast<int>(q)) ++R;
    return PrWhere{static_cast<int>(c), R, static_cast<int>(q) - R * (R + 1) / 2};
}

// wait with cluster-scope acquire: the data guarded by the barrier was written by the peer CTA
__device__ __forceinline__ void pr_mbar_wait_cluster(uint32_t bar, uint32_t parity)
{
    uint32_t spins = 0, ok = 0;
    while (!ok) {
        asm volatile(
            "{\n\t"
            ".reg .pred p;\n\t"
            "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%1], %2;\n\t"
            "selp.u32 %0, 1, 0, p;\n\t"
            "}"
            : "=r"(ok)
            : "r"(bar), "r"(parity)
            : "memory");
        if (!ok && ++spins > (1u << 28)) __trap();
    }
}

// The tile ring of a pair: the leader's producer draws an index and writes it into slot n of BOTH CTAs' rings;
// every consumer role of either CTA reads its local slot and then arrives on the LEADER's "slot free" barrier.
// Arrival on the leader's sempty after reading a slot.  0 (default): a plain arrival issued AFTER the shuffle that
// broadcasts the loaded index, i.e. after the load has returned -- a value already in a register cannot be changed by
// the rewrite that the arrival allows.  2: cluster-scope release from every consumer, 1: from the peer CTA's consumers
// only -- what the PTX memory model asks for in the letter; measured cost on cfg2 6 - 8 % (2031 / 2070 vs 2204 TOPS),
// on cfg3 1 - 3 %, with the same 0 wrong runs of 40 as 0 (profiles/round1.md).
#ifndef BFX_RING_ARRIVE
#define BFX_RING_ARRIVE 0
#endif
struct PrRing {
    uint32_t bar_sfull, ring_base;  // local shared addresses
    uint32_t lead_sempty;           // shared::cluster address of the leader's bar_sempty[0]

    // The slot is rewritten by the leader CTA (a remote store for the peer's copy) as soon as every consumer has
    // arrived on sempty, so the READ of the slot must be complete before the arrival leaves: lane 0 reads, and the
    // shuffle that broadcasts the value cannot issue before the load has returned.  (Before: every lane loaded, then
    // __syncwarp, then lane 0's remote arrival -- which does not wait for the load.  In xcorr_pair4_kernel, whose
    // unpack warps keep the shared-memory pipe busy, a peer epilogue warp that was the last to arrive now and then
    // got the index published TC_RING iterations later and added its tile there: profiles/round1.md.)
    template <bool WARP>
    __device__ __forceinline__ long long get(uint32_t n, uint32_t lane) const
    {
        const uint32_t slot = n % TC_RING;
        pr_mbar_wait_cluster(bar_sfull + 8 * slot, (n / TC_RING) & 1);
        long long w = 0;
        if (!WARP || lane == 0)
            asm volatile("ld.shared.s64 %0, [%1];" : "=l"(w) : "r"(ring_base + 8 * slot) : "memory");
        if (WARP) w = __shfl_sync(0xffffffffu, w, 0);
        if (!WARP || lane == 0) {
#if BFX_RING_ARRIVE == 2
            ptx::mbar_arrive_release_cluster_addr(lead_sempty + 8 * slot);
#elif BFX_RING_ARRIVE == 1
            if (ptx::cluster_ctarank() != 0) ptx::mbar_arrive_release_cluster_addr(lead_sempty + 8 * slot);
            else ptx::mbar_arrive_cluster_addr(lead_sempty + 8 * slot);   // the leader's own barrier: CTA scope is enough
#else
            ptx::mbar_arrive_cluster_addr(lead_sempty + 8 * slot);
#endif
        }
        return w;
    }
};

__global__ void __launch_bounds__(PR_THREADS, 1)
xcorr_pair_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int S = PR_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t op_base = smem_base;                         // S stages of (A-half, B-half)
    const uint32_t stg_base = op_base + S * PR_STAGE_BYTES;     // epilogue staging
    const uint32_t bar_base = stg_base + TC_STG_BYTES;
    const uint32_t bar_full = bar_base;                  // [S]  leader: both CTAs' operand boxes have landed
    const uint32_t bar_empty = bar_full + 8 * S;         // [S]  both: the MMAs reading the stage have completed
    const uint32_t bar_tfull = bar_empty + 8 * S;        // [2]  both: accumulator complete
    const uint32_t bar_tempty = bar_tfull + 16;          // [2]  leader: drained by the 8 epilogue warps of the pair
    const uint32_t tmem_slot = bar_tempty + 16;          // TMEM base address
    const uint32_t bar_sfull = tmem_slot + 8;            // [TC_RING] both: tile index published
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING; // [TC_RING] leader: all consumer roles of the pair have read it
    const uint32_t ring_base = bar_sempty + 8 * TC_RING; // [TC_RING] int64 tile index, -1 = no more work

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();
    const uint32_t rank = ptx::cluster_ctarank();        // 0 = leader
    const bool leader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, 1);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(bar_tfull + 8 * b, 1);
            ptx::mbar_init(bar_tempty + 8 * b, 8);
        }
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            // leader: MMA issuer + 4 epilogue warps; peer: producer + 4 epilogue warps
            ptx::mbar_init(bar_sempty + 8 * s, 10);
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<2>(tmem_slot, TC_TMEM_COLS);
        ptx::tmem_relinquish<2>();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();  // the peer's barriers are initialised before anything arrives on them remotely
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const int nkb = (p.ntime + TC_KT - 1) / TC_KT;
    const PrRing ring{bar_sfull, ring_base, ptx::mapa(bar_sempty, 0)};
    const uint32_t lead_full = ptx::mapa(bar_full, 0);
    const uint32_t lead_tempty = ptx::mapa(bar_tempty, 0);

    // The producer and MMA-issuer loops are run by whole, converged warps with only the asynchronous instructions
    // predicated on lane 0: all addresses, descriptors and coordinates are then warp-uniform, so the compiler keeps
    // them in uniform registers and a UTMALDG / UTCIMMA issue costs a few cycles instead of ~80 (measured:
    // four MMAs per stage issued from a lone thread ran the tensor pipe at 69 %, from a converged warp at 100 %).
    if (warp == 0) {
        // ===================== TMA producer (+ tile scheduler in the leader) =====================
        uint32_t stage = 0, phase = 0;
        int ready_chan = -1;
        const uint64_t pol_last = ptx::policy_evict_last();  // ring slabs are re-read by every tile of the channel
        // the leader draws tile n + 1 from the global counter before it loads tile n: the atomic's round trip
        // (and everything the other roles do on receiving an index) overlaps the loads of the current tile
        unsigned long long w_next = 0;
        if (leader) {
            if (lane == 0) w_next = atomicAdd(p.sched, 1ull);
            w_next = __shfl_sync(0xffffffffu, w_next, 0);
        }
        for (uint32_t n = 0;; ++n) {
            long long w;
            if (leader) {
                const uint32_t slot = n % TC_RING;
                ptx::mbar_wait(bar_sempty + 8 * slot, ((n / TC_RING) & 1) ^ 1);
                w = static_cast<long long>(w_next);
                if (w >= p.ntiles) w = -1;
                if (lane == 0) {
                    if (w >= 0) w_next = atomicAdd(p.sched, 1ull);
                    asm volatile("st.shared.s64 [%0], %1;" ::"r"(ring_base + 8 * slot), "l"(w) : "memory");
                    ptx::mbar_arrive(bar_sfull + 8 * slot);
                    asm volatile("st.shared::cluster.s64 [%0], %1;" ::"r"(ptx::mapa(ring_base + 8 * slot, 1)), "l"(w) : "memory");
                    ptx::mbar_arrive_cluster(bar_sfull + 8 * slot, 1);
                }
                w_next = __shfl_sync(0xffffffffu, w_next, 0);
            } else {
                w = __shfl_sync(0xffffffffu, ring.get<true>(n, lane), 0);
            }
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const int c = tl.c;
            if (c != ready_chan) {
                // the relayout warps (of any CTA) must have written all of z[c]; their generic-proxy stores are
                // then ordered before our TMA (async proxy) reads
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
            const bool diag = tl.R == tl.Cb;
            const int xa = 256 * tl.R + 128 * static_cast<int>(rank);
            const int xb = 256 * tl.Cb + 128 * static_cast<int>(rank);
            const uint32_t cta_bytes = diag ? TC_BOX_BYTES : 2 * TC_BOX_BYTES;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                if (lane == 0) {
                    if (leader) ptx::mbar_expect_tx(bar_full + 8 * stage, 2 * cta_bytes);  // both CTAs' boxes
                    const uint32_t dst = op_base + stage * PR_STAGE_BYTES;
                    const uint32_t fullb = lead_full + 8 * stage;
                    const int t0 = kb * TC_KT;
                    ptx::tma_load_3d_cg2_hint(dst, &tmap, fullb, xa, cs, t0, pol_last);
                    if (!diag) ptx::tma_load_3d_cg2_hint(dst + TC_BOX_BYTES, &tmap, fullb, xb, cs, t0, pol_last);
                }
                __syncwarp();
                if (++stage == S) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (S3), leader only =====================
        if (leader) {
            uint32_t stage = 0, phase = 0;
            const uint32_t idesc = tc_instr_desc(256, 256);
            for (uint32_t it = 0;; ++it) {
                const long long w = __shfl_sync(0xffffffffu, ring.get<true>(it, lane), 0);
                if (w < 0) break;
                const PrWhere tl = pr_decode(w, p.tiles_per_chan);
                const bool diag = tl.R == tl.Cb;
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
                        ptx::mma_commit_cg2(bar_empty + 8 * stage, 3);
                    }
                    __syncwarp();
                    if (++stage == S) { stage = 0; phase ^= 1; }
                }
                if (lane == 0) {
                    ptx::mma_commit_cg2(bar_tfull + 8 * buf, 3);
                    // every operand load of this tile has landed in shared memory (observed through the full
                    // barriers, so a relaxed count is enough): its ring slab may be recycled
                    ptx::red_relaxed_add_u64(p.done + tl.c, 1ull);
                }
                __syncwarp();
            }
        }
    } else if (warp >= 4 && warp < 8) {
        // ===================== epilogue (S4), both CTAs =====================
        const int wq = warp - 4;
        const uint32_t stg_warp = stg_base + wq * TC_STG_WARP_BYTES;
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        uint32_t nchunks_done = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const int c = tl.c;
            const uint32_t buf = it & 1, bphase = (it >> 1) & 1;
            const int i0 = PR_BLK * tl.R + 64 * static_cast<int>(rank) + 16 * wq;  // first input row of this warp
            const int j0 = PR_BLK * tl.Cb;
            // 64-column chunks that reach the diagonal or lie below it (i0 >= j0 always: Cb <= R)
            int nchunk = (i0 + 15 - j0) / TC_CJ + 1;
            nchunk = nchunk > 2 ? 2 : nchunk;
            int32_t* const out_c = p.out + 2 * (static_cast<long long>(c) * nbl);
            if (p.accumulate && lane < 16) {
                // the L2 reduce-adds of this tile will want the old visibilities resident: start pulling this warp's
                // row segments in now, while the tile is still being contracted
                const int i_own = i0 + static_cast<int>(lane);
                int n = i_own + 1 - j0;
                n = n > PR_BLK ? PR_BLK : n;
                if (i_own < p.ninputs && n > 0) {
                    const long long e0 = static_cast<long long>(i_own) * (i_own + 1) / 2 + j0;
                    const long long ea = e0 & ~1ll, eb = (e0 + n + 1) & ~1ll;  // 16-byte aligned cover
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
        if (lane < 16) ptx::bulk_wait_read<0>();  // shared memory must outlive the bulk reads
    } else if (warp >= 8) {
        tc_relayout_role(p, lane);
    }

    ptx::tc_fence_before();
    __syncthreads();
    ptx::cluster_sync();  // no remote arrive / multicast commit may still be in flight towards a CTA that exits
    if (warp == 2) ptx::tmem_dealloc<2>(tmem_base, TC_TMEM_COLS);
    // the last CTA to finish re-arms the scheduler for the next launch
    if (threadIdx.x == 0 && atomicAdd(p.sched + 1, 1ull) == gridDim.x - 1) {
        p.sched[0] = 0;
        p.sched[1] = 0;
        p.sched[2] = 0;
    }
}

}  // namespace bfx
