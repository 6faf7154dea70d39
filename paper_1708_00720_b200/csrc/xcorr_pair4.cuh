// xcorr_pair4.cuh -- the CTA-pair contraction of xcorr_pair.cuh for ci4 spans with more than 64 inputs.
//
// The pair kernel is bound by the bytes it moves through the L2 (profiles/round1.md), most of them operand boxes.
// A ci4 sample is one byte, so here the S1 ring keeps the span PACKED (z4[c % W][t][i], one byte per sample: the
// relayout warps only copy) and the operand boxes are half as large; the widening to int8 pairs happens in
// shared memory, as in xcorr_few.cuh: TMA -> raw ring -> 8 unpack warps -> 128B-swizzled int8 tiles (nibble << 4,
// the 16 x 16 scale is shifted out exactly in the epilogue) -> tcgen05.mma.cta_group::2.
//
// Per CTA (768 threads, registers moved between warpgroups with setmaxnreg):
//   warp 0       TMA producer of its own raw boxes (A-half, B-half: {64 B, 1 channel, 128 samples}); the leader's
//                also draws the tile index and publishes it to both CTAs
//   warp 1       leader: MMA issuer; peer: relay -- waits until the peer's unpack warps have written a stage and
//                arrives once on the leader's "stage full" barrier (one cluster-scope release per stage)
//   warp 2       TMEM allocation
//   warps 4..7   epilogue (as xcorr_pair.cuh, one staging buffer per warp)
//   warps 8..15  unpack
//   warps 16..23 relayout (S1: span -> packed ring)
#pragma once
#include "xcorr_pair.cuh"

namespace bfx {

constexpr int P4_RAW_BOX = TC_KT * 64;               // one raw box: TC_KT rows of 64 bytes
constexpr int P4_RAW_STAGE = 2 * P4_RAW_BOX;         // A-half, B-half
constexpr int P4_OP_STAGE = 2 * TC_BOX_BYTES;        // the same, widened
#ifndef BFX_P4_RAW
#define BFX_P4_RAW 6
#endif
#ifndef BFX_P4_OP
#define BFX_P4_OP 3
#endif
constexpr int P4_RAW_STAGES = BFX_P4_RAW, P4_OP_STAGES = BFX_P4_OP;
constexpr int P4_UNPACK_WARPS = 8;
constexpr int P4_THREADS = 768;
constexpr int P4_STG_BYTES = 4 * TC_STG_BUF_BYTES;   // one staging buffer per epilogue warp
constexpr int P4_SMEM_BYTES = 1024 + P4_OP_STAGES * P4_OP_STAGE + P4_RAW_STAGES * P4_RAW_STAGE + P4_STG_BYTES + 512;
// registers per thread after setmaxnreg; the pool is what the CTA got at launch, 768 x 80 = 61440:
// 128*40 + 128*104 + 256*64 + 256*104 = 61440
constexpr int P4_REGS_CTRL = 40, P4_REGS_EPI = 104, P4_REGS_UNPACK = 64, P4_REGS_RELAYOUT = 104;

__device__ __forceinline__ void p4_tma_load_hint(uint32_t dst, const CUtensorMap* m, uint32_t bar, int x, int y, int z, uint64_t pol)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%3, %4, %5}], "
        "[%2], %6;" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(m)), "r"(bar), "r"(x), "r"(y), "r"(z), "l"(pol)
        : "memory");
}

template <int N>
__device__ __forceinline__ void p4_regs_inc()
{
    asm volatile("setmaxnreg.inc.sync.aligned.u32 %0;" ::"n"(N));
}
template <int N>
__device__ __forceinline__ void p4_regs_dec()
{
    asm volatile("setmaxnreg.dec.sync.aligned.u32 %0;" ::"n"(N));
}

__global__ void __launch_bounds__(P4_THREADS, 1)
xcorr_pair4_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int S = P4_OP_STAGES, R = P4_RAW_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t op_base = smem_base;                         // S stages of int8 (A-half, B-half)
    const uint32_t raw_base = op_base + S * P4_OP_STAGE;        // R stages of raw (A-half, B-half)
    const uint32_t stg_base = raw_base + R * P4_RAW_STAGE;      // epilogue staging
    const uint32_t bar_base = stg_base + P4_STG_BYTES;
    const uint32_t bar_full = bar_base;                  // [S] int8 stage written: leader 8 unpack warps + relay, peer 8
    const uint32_t bar_empty = bar_full + 8 * S;         // [S] both: the MMAs reading the stage have completed
    const uint32_t bar_rfull = bar_empty + 8 * S;        // [R] own raw boxes have landed
    const uint32_t bar_rempty = bar_rfull + 8 * R;       // [R] own raw boxes consumed by the 8 unpack warps
    const uint32_t bar_tfull = bar_rempty + 8 * R;       // [2] accumulator complete
    const uint32_t bar_tempty = bar_tfull + 16;          // [2] leader: drained by the 8 epilogue warps of the pair
    const uint32_t tmem_slot = bar_tempty + 16;
    const uint32_t bar_sfull = tmem_slot + 8;            // [TC_RING] tile index published
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING; // [TC_RING] leader: every consumer role of the pair has read it
    const uint32_t ring_base = bar_sempty + 8 * TC_RING;

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();
    const uint32_t rank = ptx::cluster_ctarank();
    const bool leader = rank == 0;

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, leader ? P4_UNPACK_WARPS + 1 : P4_UNPACK_WARPS);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int s = 0; s < R; ++s) {
            ptx::mbar_init(bar_rfull + 8 * s, 1);
            ptx::mbar_init(bar_rempty + 8 * s, P4_UNPACK_WARPS);
        }
        for (int b = 0; b < 2; ++b) {
            ptx::mbar_init(bar_tfull + 8 * b, 1);
            ptx::mbar_init(bar_tempty + 8 * b, 8);
        }
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            // leader: MMA + 4 epilogue + 8 unpack; peer: producer + relay + 4 epilogue + 8 unpack
            ptx::mbar_init(bar_sempty + 8 * s, 27);
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
    const uint32_t lead_tempty = ptx::mapa(bar_tempty, 0);
    const uint32_t lead_full = ptx::mapa(bar_full, 0);

    if (warp == 0) {
        // ===================== TMA producer of raw boxes (+ tile scheduler in the leader) =====================
        p4_regs_dec<P4_REGS_CTRL>();
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
                w = __shfl_sync(0xffffffffu, ring.get<true>(n, lane), 0);
            }
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const int c = tl.c;
            if (p.z != nullptr && c != ready_chan) {   // (p.z == NULL: the packed span is read in place, no ring)
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
            const int xa = 128 * tl.R + 64 * static_cast<int>(rank);   // bytes: one per sample
            const int xb = 128 * tl.Cb + 64 * static_cast<int>(rank);
            const uint32_t tx = diag ? P4_RAW_BOX : 2 * P4_RAW_BOX;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rempty + 8 * stage, phase ^ 1);
                if (lane == 0) {
                    ptx::mbar_expect_tx(bar_rfull + 8 * stage, tx);
                    const uint32_t dst = raw_base + stage * P4_RAW_STAGE;
                    p4_tma_load_hint(dst, &tmap, bar_rfull + 8 * stage, xa, cs, kb * TC_KT, pol_last);
                    if (!diag) p4_tma_load_hint(dst + P4_RAW_BOX, &tmap, bar_rfull + 8 * stage, xb, cs, kb * TC_KT, pol_last);
                }
                __syncwarp();
                if (++stage == R) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        p4_regs_dec<P4_REGS_CTRL>();
        uint32_t stage = 0, phase = 0;
        if (leader) {
            // ===================== MMA issuer (S3) =====================
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
                    pr_mbar_wait_cluster(bar_full + 8 * stage, phase);   // the peer's half was written by the peer CTA
                    ptx::tc_fence_after();
                    const uint32_t sbase = op_base + stage * P4_OP_STAGE;
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
                    if (p.z != nullptr) ptx::red_relaxed_add_u64(p.done + tl.c, 1ull);
                }
                __syncwarp();
            }
        } else {
            // ===================== relay: peer's stage written -> one arrival on the leader's barrier =====================
            for (uint32_t it = 0;; ++it) {
                const long long w = __shfl_sync(0xffffffffu, ring.get<true>(it, lane), 0);
                if (w < 0) break;
                for (int kb = 0; kb < nkb; ++kb) {
                    ptx::mbar_wait(bar_full + 8 * stage, phase);
                    // the stage lives in this CTA's shared memory and is complete (observed through the local barrier):
                    // a plain remote arrival is enough, a cluster-scope release would cost a MEMBAR per stage
                    // (BFX_RING_ARRIVE >= 1, xcorr_pair.cuh: the build that follows the PTX memory model to the letter --
                    // tests/test_gpu_conformant_build.py runs it against this one)
#if BFX_RING_ARRIVE >= 1
                    if (lane == 0) ptx::mbar_arrive_release_cluster_addr(lead_full + 8 * stage);
#else
                    if (lane == 0) ptx::mbar_arrive_cluster_addr(lead_full + 8 * stage);
#endif
                    __syncwarp();
                    if (++stage == S) { stage = 0; phase ^= 1; }
                }
            }
        }
    } else if (warp < 4) {
        p4_regs_dec<P4_REGS_CTRL>();
    } else if (warp < 8) {
        // ===================== epilogue (S4), both CTAs =====================
        p4_regs_inc<P4_REGS_EPI>();
        const int wq = warp - 4;
        const uint32_t stg_buf = stg_base + wq * TC_STG_BUF_BYTES;
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const uint32_t buf = it & 1, bphase = (it >> 1) & 1;
            const int i0 = PR_BLK * tl.R + 64 * static_cast<int>(rank) + 16 * wq;  // first input row of this warp
            const int j0 = PR_BLK * tl.Cb;
            int nchunk = (i0 + 15 - j0) / TC_CJ + 1;   // 64-column chunks that reach the diagonal or lie below it
            nchunk = nchunk > 2 ? 2 : nchunk;
            int32_t* const out_c = p.out + 2 * (static_cast<long long>(tl.c) * nbl);
            if (p.accumulate && lane < 16) {
                // the L2 reduce-adds of this tile will want the old visibilities resident
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
            for (int jc = 0; jc < nchunk; ++jc) {
                const uint32_t tcol = tmem_base + (static_cast<uint32_t>(32 * wq) << 16) + buf * 256 + jc * 128;
                tc_epilogue_chunk<true, true, 0, true>(p, lane, tcol, stg_buf, out_c, i0, j0 + jc * TC_CJ,
                                                 jc == nchunk - 1 ? lead_tempty + 8 * buf : 0u);
            }
        }
        if (lane < 16) ptx::bulk_wait_read<0>();  // shared memory must outlive the bulk reads
    } else if (warp < 8 + P4_UNPACK_WARPS) {
        // ===================== unpack warps: raw [t][64 B] boxes -> 128B-swizzled int8 boxes (nibble << 4) =====================
        // lane -> (row t, 16-byte chunk qc): a quarter-warp reads 128 contiguous raw bytes and writes 2 rows x 4 chunks of
        // a swizzled tile, touching every bank once
        p4_regs_dec<P4_REGS_UNPACK>();
        const int uw = warp - 8, tl8 = static_cast<int>(lane >> 2), qc = static_cast<int>(lane & 3);
        uint32_t rstage = 0, rphase = 0, ostage = 0, ophase = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const int nbox = tl.R == tl.Cb ? 1 : 2;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rfull + 8 * rstage, rphase);
                ptx::mbar_wait(bar_empty + 8 * ostage, ophase ^ 1);
                const uint32_t rsrc = raw_base + rstage * P4_RAW_STAGE;
                const uint32_t odst = op_base + ostage * P4_OP_STAGE;
                for (int bx = 0; bx < nbox; ++bx) {
#pragma unroll
                    for (int t = uw * 8 + tl8; t < TC_KT; t += 8 * P4_UNPACK_WARPS) {
                        uint32_t wv[4];
                        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                     : "=r"(wv[0]), "=r"(wv[1]), "=r"(wv[2]), "=r"(wv[3])
                                     : "r"(rsrc + bx * P4_RAW_BOX + t * 64 + qc * 16));
                        // grouped real embedding (re0..re3 im0..im3 per four inputs): no byte permutes
                        uint32_t o[8];
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            o[2 * u] = wv[u] & 0xF0F0F0F0u;                   // re0..re3, each << 4
                            o[2 * u + 1] = (wv[u] << 4) & 0xF0F0F0F0u;        // im0..im3, each << 4
                        }
                        const uint32_t rowa = odst + bx * TC_BOX_BYTES + t * 128;
                        const uint32_t a0 = rowa + static_cast<uint32_t>((2 * qc) ^ (t & 7)) * 16;
                        const uint32_t a1 = rowa + static_cast<uint32_t>((2 * qc + 1) ^ (t & 7)) * 16;
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a0), "r"(o[0]), "r"(o[1]), "r"(o[2]), "r"(o[3]) : "memory");
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a1), "r"(o[4]), "r"(o[5]), "r"(o[6]), "r"(o[7]) : "memory");
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
    } else {
        // ===================== relayout warps (S1): span -> packed ring, a plain copy =====================
        p4_regs_inc<P4_REGS_RELAYOUT>();
        if (p.z != nullptr) tc_relayout_role(p, lane);
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
