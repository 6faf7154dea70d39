// xcorr_stripe.cuh -- CTA-pair contraction with a RESIDENT A block, for ci8 spans of at most 1024 samples.
//
// xcorr_pair.cuh streams both operands of every tile through its stage ring: a channel of n 128-input blocks costs
// n (n + 1) / 2 A loads and n (n - 1) / 2 B loads of (256 real rows x ntime) bytes.  Here a pair works on a whole
// STRIPE of tiles (channel c, row block R, column blocks Cb = 0 .. R): the A block (each CTA's 128 real rows x ntime
// <= 128 KiB) is loaded once, during the stripe's first tile, into ST_MAXKB resident slots and re-used by every tile
// of the stripe; only B streams through a ring, and the diagonal tile (Cb = R, B == A) loads nothing.  Operand
// traffic from the L2 drops from n^2 to n (n + 1) / 2 block loads per channel: -37 % at 512 inputs, -47 % at 2048
// (the kernel is L2-bound: profiles/round1.md).  Everything else -- real Gram embedding, TMEM double buffering,
// relayout ring, epilogue -- is xcorr_pair.cuh's.
//
// With so few operand loads left, spans of up to BFX_DIRECT_MAX_BLK row blocks are read STRAIGHT FROM THE SPAN
// (p.z == NULL: the tensor map describes x[t][c][...] itself, ring_w = nchan): the address-translation stall of
// strided boxes that made S1 necessary for xcorr_pair.cuh (one 2 MiB page per sample) costs less than the relayout
// once A is loaded once per stripe -- measured on cfg3: 1.84 ms direct against 2.19 ms through the ring; on 2048
// inputs (16 row blocks, B re-read up to 15 times) the ring still wins, 8.1 against 8.8 ms (profiles/round1.md).
//
// Barriers per CTA: a_full[kb] / a_empty[kb] per resident slot (phase = stripe parity), b_full / b_empty per ring
// stage, tfull / tempty per accumulator, the stripe-index ring.  A slot kb is released by a commit after the LAST
// tile's MMAs on it, so the next stripe's A loads trail the current stripe's last tile by one slot.
//
// Epilogue (S4), chosen per launch (profiles/round2.md):
//   accumulate = 0, span in place: tc_epilogue_direct by EIGHT warps (warp 4 + 4 h + q drains TMEM lane quarter q,
//     column half h) -- registers -> 8-byte global stores through the LSU.  The staged epilogue's warps spent 47 % of
//     their time in the serialised bulk-copy issue loop, competing with the operand loads for the TMA unit; without
//     staging memory there is room for six B stages.
//   accumulate != 0, or operands through the S1 ring: tc_epilogue_chunk by four warps -- staged rows, added at the L2 by
//     cp.reduce.async.bulk (a read-modify-write through the SM was measured slower: 3.3 against 2.15 ms on cfg3).
#pragma once
#include "xcorr_pair.cuh"

namespace bfx {

constexpr int ST_MAXKB = 1024 / TC_KT;               // resident A slots of TC_KT samples: ntime <= 1024 (8 slots of 128)

// RING: operands through the S1 ring (8 relayout warps); DIRECT_EPI: the register-direct epilogue (in place, accumulate = 0)
template <bool RING, bool DIRECT_EPI>
struct StCfg {
    static_assert(!(RING && DIRECT_EPI), "the register-direct epilogue is built for the in-place kernel only");
    static constexpr int kBStages = DIRECT_EPI ? 6 : 4;
    static constexpr int kEpiWarps = DIRECT_EPI ? 8 : 4;
    static constexpr int kThreads = DIRECT_EPI ? 32 * (4 + kEpiWarps) : 512;   // staged variants: warps 8..15 relayout (RING) or idle
    static constexpr int kStgBytes = DIRECT_EPI ? 0 : 4 * TC_STG_BUF_BYTES;   // one staging buffer per epilogue warp
    static constexpr int kSmemBytes = 1024 + (ST_MAXKB + kBStages) * TC_BOX_BYTES + kStgBytes + 512;
    static_assert(kSmemBytes <= 232448, "stripe kernel shared memory");
};

// jj-th tile of a stripe of R + 1 tiles -> column block: 0 .. R, the diagonal tile (which loads nothing) last.  (The
// diagonal tile first, so that every tile needs exactly one operand block, changed nothing: profiles/round1.md.)
__device__ __forceinline__ int st_col_block(int jj, int /*R*/) { return jj; }

template <bool RING, bool DIRECT_EPI>
__global__ void __launch_bounds__(StCfg<RING, DIRECT_EPI>::kThreads, 1)
xcorr_stripe_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    using Cfg = StCfg<RING, DIRECT_EPI>;
    constexpr int S = Cfg::kBStages;
    constexpr int EPI_WARPS = Cfg::kEpiWarps;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t a_base = smem_base;                               // ST_MAXKB resident A-half boxes
    const uint32_t b_base = a_base + ST_MAXKB * TC_BOX_BYTES;        // S streaming B-half boxes
    const uint32_t stg_base = b_base + S * TC_BOX_BYTES;             // epilogue staging
    const uint32_t bar_base = stg_base + Cfg::kStgBytes;
    const uint32_t bar_afull = bar_base;                     // [ST_MAXKB] leader: both CTAs' A boxes have landed
    const uint32_t bar_aempty = bar_afull + 8 * ST_MAXKB;    // [ST_MAXKB] both: the stripe's last MMAs on the slot are done
    const uint32_t bar_full = bar_aempty + 8 * ST_MAXKB;     // [S] leader: both CTAs' B boxes have landed
    const uint32_t bar_empty = bar_full + 8 * S;             // [S] both: the MMAs reading the stage have completed
    const uint32_t bar_tfull = bar_empty + 8 * S;            // [2] both: accumulator complete
    const uint32_t bar_tempty = bar_tfull + 16;              // [2] leader: drained by the 8 epilogue warps of the pair
    const uint32_t tmem_slot = bar_tempty + 16;
    const uint32_t bar_sfull = tmem_slot + 8;                // [TC_RING] both: stripe index published
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING;     // [TC_RING] leader: all consumer roles have read it
    const uint32_t ring_base = bar_sempty + 8 * TC_RING;     // [TC_RING] int64 stripe index, -1 = no more work

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < ST_MAXKB; ++s) {
            ptx::mbar_init(bar_afull + 8 * s, 1);
            ptx::mbar_init(bar_aempty + 8 * s, 1);
        }
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, 1);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(bar_tfull + 8 * b, 1);
            ptx::mbar_init(bar_tempty + 8 * b, 2 * EPI_WARPS);   // drained by the epilogue warps of the pair
        }
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            ptx::mbar_init(bar_sempty + 8 * s, 2 + 2 * EPI_WARPS);   // leader: MMA issuer + epilogue; peer: producer + epilogue
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
    const int nblk = (p.ninputs + PR_BLK - 1) / PR_BLK;
    constexpr bool direct = !RING;        // operands straight from the span: no ring, no relayout (see the header)
    const PrRing ring{bar_sfull, ring_base, ptx::mapa(bar_sempty, 0)};
    const uint32_t lead_full = ptx::mapa(bar_full, 0);
    const uint32_t lead_afull = ptx::mapa(bar_afull, 0);
    const uint32_t lead_tempty = ptx::mapa(bar_tempty, 0);
    // stripe index w -> channel w / nblk, row block R = nblk - 1 - w % nblk (long stripes first)

    if (warp == 0) {
        // ===================== TMA producer (+ stripe scheduler in the leader) =====================
        uint32_t stage = 0, phase = 0;
        int ready_chan = -1;
        const uint64_t pol_last = ptx::policy_evict_last();
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
                w = __shfl_sync(0xffffffffu, ring.template get<true>(n, lane), 0);
            }
            if (w < 0) break;
            const int c = static_cast<int>(static_cast<uint32_t>(w) / static_cast<uint32_t>(nblk));
            const int R = nblk - 1 - (static_cast<int>(static_cast<uint32_t>(w)) - c * nblk);
            if (!direct && c != ready_chan) {
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
            const int xa = 256 * R + 128 * static_cast<int>(rank);
            const uint32_t aphase = n & 1;
            for (int jj = 0; jj <= R; ++jj) {
                const int j = st_col_block(jj, R);
                const bool diag = j == R;
                const int xb = 256 * j + 128 * static_cast<int>(rank);
                for (int kb = 0; kb < nkb; ++kb) {
                    const int t0 = kb * TC_KT;
                    if (jj == 0) {
                        ptx::mbar_wait(bar_aempty + 8 * kb, aphase ^ 1);
                        if (lane == 0) {
                            if (leader) ptx::mbar_expect_tx(bar_afull + 8 * kb, 2 * TC_BOX_BYTES);
                            ptx::tma_load_3d_cg2_hint(a_base + kb * TC_BOX_BYTES, &tmap, lead_afull + 8 * kb, xa, cs, t0, pol_last);
                        }
                    }
                    if (!diag) {
                        ptx::mbar_wait(bar_empty + 8 * stage, phase ^ 1);
                        if (lane == 0) {
                            if (leader) ptx::mbar_expect_tx(bar_full + 8 * stage, 2 * TC_BOX_BYTES);
                            ptx::tma_load_3d_cg2_hint(b_base + stage * TC_BOX_BYTES, &tmap, lead_full + 8 * stage, xb, cs, t0, pol_last);
                        }
                        if (++stage == S) { stage = 0; phase ^= 1; }
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (S3), leader only =====================
        if (leader) {
            uint32_t stage = 0, phase = 0, tcount = 0;
            const uint32_t idesc = tc_instr_desc(256, 256);
            for (uint32_t it = 0;; ++it) {
                const long long w = __shfl_sync(0xffffffffu, ring.template get<true>(it, lane), 0);
                if (w < 0) break;
                const int c = static_cast<int>(static_cast<uint32_t>(w) / static_cast<uint32_t>(nblk));
                const int R = nblk - 1 - (static_cast<int>(static_cast<uint32_t>(w)) - c * nblk);
                const uint32_t aphase = it & 1;
                for (int jj = 0; jj <= R; ++jj, ++tcount) {
                    const bool diag = st_col_block(jj, R) == R;
                    const bool last = jj == R;   // the stripe's last tile hands the resident A slots back
                    const uint32_t buf = tcount & 1, bphase = (tcount >> 1) & 1;
                    const uint32_t d_tmem = tmem_base + buf * 256;
                    ptx::mbar_wait(bar_tempty + 8 * buf, bphase ^ 1);
                    ptx::tc_fence_after();
                    for (int kb = 0; kb < nkb; ++kb) {
                        if (jj == 0) ptx::mbar_wait(bar_afull + 8 * kb, aphase);
                        if (!diag) ptx::mbar_wait(bar_full + 8 * stage, phase);
                        ptx::tc_fence_after();
                        const uint64_t adesc = tc_smem_desc(a_base + kb * TC_BOX_BYTES, TC_BOX_BYTES);
                        const uint64_t bdesc = diag ? adesc : tc_smem_desc(b_base + stage * TC_BOX_BYTES, TC_BOX_BYTES);
                        const int trem = p.ntime - kb * TC_KT;
                        const int nk = trem >= TC_KT ? TC_KT / 32 : (trem + 31) / 32;
                        if (lane == 0) {
                            for (int k = 0; k < nk; ++k)
                                ptx::mma_i8<2>(d_tmem, adesc + 256u * k, bdesc + 256u * k, idesc, (kb | k) != 0 ? 1u : 0u);
                            if (!diag) ptx::mma_commit_cg2(bar_empty + 8 * stage, 3);
                            if (last) ptx::mma_commit_cg2(bar_aempty + 8 * kb, 3);
                        }
                        __syncwarp();
                        if (!diag && ++stage == S) { stage = 0; phase ^= 1; }
                    }
                    if (lane == 0) {
                        ptx::mma_commit_cg2(bar_tfull + 8 * buf, 3);
                        if (!direct) ptx::red_relaxed_add_u64(p.done + c, 1ull);
                    }
                    __syncwarp();
                }
            }
        }
    } else if (warp >= 4 && warp < 4 + EPI_WARPS) {
        // ===================== epilogue (S4), both CTAs =====================
        const int wq = warp & 3;                       // TMEM lane quarter of this warp
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        uint32_t tcount = 0;
        [[maybe_unused]] uint32_t nchunks_done = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.template get<true>(it, lane);
            if (w < 0) break;
            const int c = static_cast<int>(static_cast<uint32_t>(w) / static_cast<uint32_t>(nblk));
            const int R = nblk - 1 - (static_cast<int>(static_cast<uint32_t>(w)) - c * nblk);
            int32_t* const out_c = p.out + 2 * (static_cast<long long>(c) * nbl);
            const int i0 = PR_BLK * R + 64 * static_cast<int>(rank) + 16 * wq;  // first input row of this warp
            for (int jj = 0; jj <= R; ++jj, ++tcount) {
                const uint32_t buf = tcount & 1, bphase = (tcount >> 1) & 1;
                const int j0 = PR_BLK * st_col_block(jj, R);
                if constexpr (DIRECT_EPI) {
                    const int h = (warp - 4) >> 2;         // the 128-column half this warp drains
                    const int jb = j0 + 64 * h;
                    if (jb <= i0 + 15) {   // its 16 rows x 64 columns reach the diagonal or lie below it (warp-uniform)
                        const uint32_t tcol = tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + buf * 256 + h * 128;
                        tc_epilogue_direct<false, true>(p, lane, tcol, out_c, i0, jb, bar_tfull + 8 * buf, bphase, lead_tempty + 8 * buf);
                    } else {
                        // nothing to store, but the accumulator may only be handed back once it is complete (the MMA
                        // issuer counts one arrival per warp and tile)
                        ptx::mbar_wait(bar_tfull + 8 * buf, bphase);
                        tc_release_tmem(lane, lead_tempty + 8 * buf, true);
                    }
                } else {
                    const uint32_t stg_warp = stg_base + wq * TC_STG_BUF_BYTES;
                    int nchunk = (i0 + 15 - j0) / TC_CJ + 1;
                    nchunk = nchunk > 2 ? 2 : nchunk;
                    // the L2 reduce-adds of this tile will want the old visibilities resident: line prefetches through the
                    // LSU (a bulk prefetch per row costs a serialised issue loop on the TMA unit: -2.8 %, profiles/round2.md)
                    if (p.accumulate) tc_prefetch_old(p, lane, out_c, i0, j0, PR_BLK);
                    ptx::mbar_wait(bar_tfull + 8 * buf, bphase);
                    ptx::tc_fence_after();
                    for (int jc = 0; jc < nchunk; ++jc, ++nchunks_done) {
                        const uint32_t tcol = tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + buf * 256 + jc * 128;
                        tc_epilogue_chunk<false, true, 0>(p, lane, tcol, stg_warp, out_c, i0, j0 + jc * TC_CJ,
                                                          jc == nchunk - 1 ? lead_tempty + 8 * buf : 0u);
                    }
                }
            }
        }
        if constexpr (!DIRECT_EPI) {
            if (lane < 16) ptx::bulk_wait_read<0>();   // shared memory must outlive the bulk reads
        }
    } else if (RING && warp >= 8) {
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
