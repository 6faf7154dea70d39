// xcorr_gauss4.cuh -- ci4 spans with the THREE-multiplication complex product (the paper's
// motivation: "operates on the 4+4 complex signed integers" directly).
//
// x_i conj(x_j) with x_i = a + jb, x_j = c + jd needs four real products in the Gram form the other kernels use
// (a c, b d, b c, a d).  Gauss's rearrangement needs three:
//     P1 = (a + b) c        P2 = a (c + d)        P3 = b (c - d)
//     Re = a c + b d = P1 - P3                    Im = b c - a d = P1 - P2
// The sums no longer fit a 4-bit code (a + b, c + d in [-16, 14], c - d in [-15, 15]) but they fit int8, which is why the
// trick exists for ci4 only.  Scaling: the plain planes keep the nibble in the high half of the byte (16 a, 16 b, 16 c:
// two logic operations per word, as in xcorr_pair4.cuh); the sum planes are the per-byte averages 8 (a + b), 8 (c + d),
// 8 (c - d) -- each half, 8 a etc., is a multiple of 8 in [-64, 56], so the sums lie in [-128, 120] and fit, the extreme
// code -8 - 8j included (8 (-8 + -8) = -128).  Every product is then scaled by 16 * 8 = 128, shifted out exactly in the
// epilogue; |P| <= ntime * 128 * 128 < 2^31 for every legal ntime.
//
// Three products of DIFFERENT operand pairs cannot share one wide MMA the way the four Gram products do (there one
// 256 x 256 MMA forms all four from two operands), so this is three M = 128, N = 128 MMAs per 32 samples on six operand
// planes: 3/4 of the multiply-accumulates, but 3 x the operand bytes read from shared memory per MAC, six planes to
// write per stage instead of four, and per-byte adds in the unpack.  Measured on cfg2 it is slower than
// xcorr_pair4_kernel (profiles/round2.md), so bfXcorrExecute never selects it; it is reachable with
// bfXcorrSetAlgo(BF_XCORR_ALGO_TCGEN05_GAUSS3) and runs the whole ci4 parity suite bit-exact.
//
// One CTA per tile of 128 x 128 inputs (cta_group::1), span read in place.  Roles (512 threads): warp 0 TMA producer of
// raw boxes {128 bytes = 128 inputs, 1 channel, G4_KT samples} (+ dynamic tile scheduler), warp 1 MMA issuer, warp 2 TMEM
// allocation, warps 4..7 epilogue (no lane exchange: the three accumulators share their (i, j) indexing), warps 8..15
// unpack raw boxes into the six 128B-swizzled MN-major planes.
#pragma once
#include "xcorr_pair.cuh"

namespace bfx {

constexpr int G4_KT = 64;                            // samples per stage
constexpr int G4_PLANE = G4_KT * 128;                // one operand plane of a stage: [t][128 inputs], 8 KiB
constexpr int G4_RAW_STAGES = 3, G4_OP_STAGES = 2;
constexpr int G4_RAW_STAGE = 2 * G4_PLANE;           // raw row block, raw column block
constexpr int G4_OP_STAGE = 6 * G4_PLANE;            // 8(a+b), 16a, 16b | 16c, 8(c+d), 8(c-d)
constexpr int G4_UNPACK_WARPS = 8;
constexpr int G4_THREADS = 512;
constexpr int G4_SMEM_BYTES = 1024 + G4_OP_STAGES * G4_OP_STAGE + G4_RAW_STAGES * G4_RAW_STAGE + 512;
static_assert(G4_SMEM_BYTES <= 232448, "gauss kernel shared memory");

// per-byte arithmetic shift right by one of bytes whose low bit is clear (no bit crosses a byte boundary)
__device__ __forceinline__ uint32_t g4_half(uint32_t x) { return ((x >> 1) & 0x7F7F7F7Fu) | (x & 0x80808080u); }

// one raw word (four ci4 samples) -> the three planes of its side: ROW side (8 (a + b), 16 a, 16 b), column side
// (16 c, 8 (c + d), 8 (c - d))
template <bool ROW_SIDE>
__device__ __forceinline__ void g4_widen(uint32_t w, uint32_t& p0, uint32_t& p1, uint32_t& p2)
{
    const uint32_t re16 = w & 0xF0F0F0F0u, im16 = (w << 4) & 0xF0F0F0F0u;
    const uint32_t re8 = g4_half(re16), im8 = g4_half(im16);
    if (ROW_SIDE) {
        p0 = __vadd4(re8, im8);
        p1 = re16;
        p2 = im16;
    } else {
        p0 = re16;
        p1 = __vadd4(re8, im8);
        p2 = __vsub4(re8, im8);
    }
}

__global__ void __launch_bounds__(G4_THREADS, 1)
xcorr_gauss4_kernel(const __grid_constant__ CUtensorMap tmap, const TcParams p)
{
    constexpr int S = G4_OP_STAGES, R = G4_RAW_STAGES;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (ptx::smem_u32(smem_raw) + 1023u) & ~1023u;
    const uint32_t op_base = smem_base;                         // S stages of six planes
    const uint32_t raw_base = op_base + S * G4_OP_STAGE;        // R stages of two raw boxes
    const uint32_t bar_base = raw_base + R * G4_RAW_STAGE;
    const uint32_t bar_full = bar_base;               // [S] planes written by the unpack warps
    const uint32_t bar_empty = bar_full + 8 * S;      // [S] the MMAs reading the stage have completed
    const uint32_t bar_rfull = bar_empty + 8 * S;     // [R] raw boxes landed
    const uint32_t bar_rempty = bar_rfull + 8 * R;    // [R] raw boxes consumed by the unpack warps
    const uint32_t bar_tfull = bar_rempty + 8 * R;    // accumulators complete
    const uint32_t bar_tempty = bar_tfull + 8;        // accumulators drained by the 4 epilogue warps
    const uint32_t tmem_slot = bar_tempty + 8;
    const uint32_t bar_sfull = tmem_slot + 8;
    const uint32_t bar_sempty = bar_sfull + 8 * TC_RING;
    const uint32_t ring_base = bar_sempty + 8 * TC_RING;

    const int warp = threadIdx.x >> 5;
    const uint32_t lane = ptx::lane_id();

    if (warp == 0 && lane == 0) {
        ptx::prefetch_tensormap(&tmap);
        for (int s = 0; s < S; ++s) {
            ptx::mbar_init(bar_full + 8 * s, G4_UNPACK_WARPS);
            ptx::mbar_init(bar_empty + 8 * s, 1);
        }
        for (int s = 0; s < R; ++s) {
            ptx::mbar_init(bar_rfull + 8 * s, 1);
            ptx::mbar_init(bar_rempty + 8 * s, G4_UNPACK_WARPS);
        }
        ptx::mbar_init(bar_tfull, 1);
        ptx::mbar_init(bar_tempty, 4);
        for (int s = 0; s < TC_RING; ++s) {
            ptx::mbar_init(bar_sfull + 8 * s, 1);
            ptx::mbar_init(bar_sempty + 8 * s, 5 + G4_UNPACK_WARPS);  // MMA issuer + 4 epilogue warps + unpack warps
        }
        ptx::fence_barrier_init();
    }
    if (warp == 2) {
        ptx::tmem_alloc<1>(tmem_slot, TC_TMEM_COLS);
        ptx::tmem_relinquish<1>();
    }
    ptx::tc_fence_before();
    __syncthreads();
    ptx::tc_fence_after();
    uint32_t tmem_base;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(tmem_base) : "r"(tmem_slot));

    const int nkb = (p.ntime + G4_KT - 1) / G4_KT;
    const TcRing ring{bar_sfull, bar_sempty, ring_base};

    if (warp == 0) {
        // ===================== TMA producer + tile scheduler (converged warp, lane 0 issues) =====================
        uint32_t stage = 0, phase = 0;
        unsigned long long w_next = 0;
        if (lane == 0) w_next = atomicAdd(p.sched, 1ull);
        w_next = __shfl_sync(0xffffffffu, w_next, 0);
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
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const bool diag = tl.R == tl.Cb;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rempty + 8 * stage, phase ^ 1);
                if (lane == 0) {
                    const uint32_t dst = raw_base + stage * G4_RAW_STAGE;
                    ptx::mbar_expect_tx(bar_rfull + 8 * stage, diag ? G4_PLANE : 2 * G4_PLANE);
                    ptx::tma_load_3d(dst, &tmap, bar_rfull + 8 * stage, PR_BLK * tl.R, tl.c, kb * G4_KT);
                    if (!diag) ptx::tma_load_3d(dst + G4_PLANE, &tmap, bar_rfull + 8 * stage, PR_BLK * tl.Cb, tl.c, kb * G4_KT);
                }
                __syncwarp();
                if (++stage == R) { stage = 0; phase ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer: three products per 32 samples (converged warp, lane 0 issues) =====================
        uint32_t stage = 0, phase = 0;
        const uint32_t idesc = tc_instr_desc(128, 128);
        for (uint32_t it = 0;; ++it) {
            const long long w = __shfl_sync(0xffffffffu, ring.get<true>(it, lane), 0);
            if (w < 0) break;
            ptx::mbar_wait(bar_tempty, (it & 1) ^ 1);   // single-buffered accumulators (3 x 128 columns)
            ptx::tc_fence_after();
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_full + 8 * stage, phase);
                ptx::tc_fence_after();
                const uint32_t sbase = op_base + stage * G4_OP_STAGE;
                const int trem = p.ntime - kb * G4_KT;
                const int nk = trem >= G4_KT ? G4_KT / 32 : (trem + 31) / 32;
                if (lane == 0) {
#pragma unroll
                    for (int q = 0; q < 3; ++q) {
                        // P1 = (a + b) c,  P2 = a (c + d),  P3 = b (c - d): row plane q with column plane q
                        const uint64_t adesc = tc_smem_desc(sbase + q * G4_PLANE, G4_PLANE);
                        const uint64_t bdesc = tc_smem_desc(sbase + (3 + q) * G4_PLANE, G4_PLANE);
                        for (int k = 0; k < nk; ++k)
                            ptx::mma_i8<1>(tmem_base + 128 * q, adesc + 256u * k, bdesc + 256u * k, idesc, (kb | k) != 0 ? 1u : 0u);
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
        // ===================== epilogue (S4): Re = (P1 - P3) >> 7, Im = (P1 - P2) >> 7 =====================
        // tcgen05.ld 16x256b: thread T (t8 = T / 4, t4 = T % 4) holds, for n = 0 .. 3, columns 8 n + 2 t4, + 1 of lanes
        // t8 and t8 + 8 -- here lane = input row and column = input column, so that is two adjacent visibilities of two
        // rows; the four threads of a quad cover 64 contiguous bytes of a packed-triangle row.
        const int wq = warp - 4;
        const int t4 = static_cast<int>(lane & 3), t8 = static_cast<int>(lane >> 2);
        const long long nbl = static_cast<long long>(p.ninputs) * (p.ninputs + 1) / 2;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            int32_t* const out_c = p.out + 2 * (static_cast<long long>(tl.c) * nbl);
            const int i0 = PR_BLK * tl.R + 32 * wq, j0 = PR_BLK * tl.Cb;
            ptx::mbar_wait(bar_tfull, it & 1);
            ptx::tc_fence_after();
#pragma unroll 1
            for (int hh = 0; hh < 2; ++hh) {
                const int ia = i0 + 16 * hh + t8, ib = ia + 8;
                int32_t* const rowa = out_c + 2 * (static_cast<long long>(ia) * (ia + 1) / 2);
                int32_t* const rowb = out_c + 2 * (static_cast<long long>(ib) * (ib + 1) / 2);
                const int lima = ia < p.ninputs ? ia : -1, limb = ib < p.ninputs ? ib : -1;   // last column of the row
#pragma unroll 1
                for (int cg = 0; cg < 4; ++cg) {
                    const int jg = j0 + 32 * cg;
                    if (jg > i0 + 16 * hh + 15 || i0 + 16 * hh >= p.ninputs) continue;   // above the diagonal / no such rows
                    uint32_t d1[16], d2[16], d3[16];
                    const uint32_t taddr = tmem_base + (static_cast<uint32_t>(32 * wq + 16 * hh) << 16) + 32 * cg;
                    ptx::tmem_ld_16x256b_x4(taddr, d1);
                    ptx::tmem_ld_16x256b_x4(taddr + 128, d2);
                    ptx::tmem_ld_16x256b_x4(taddr + 256, d3);
                    ptx::tmem_ld_wait();
#pragma unroll
                    for (int n = 0; n < 4; ++n) {
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            // e = 0, 1: row ia, columns j, j + 1; e = 2, 3: row ib, the same columns
                            const int j = jg + 8 * n + 2 * t4 + (e & 1);
                            const int lim = e < 2 ? lima : limb;
                            int32_t* const dst = (e < 2 ? rowa : rowb) + 2 * j;
                            const int p1 = static_cast<int>(d1[4 * n + e]);
                            int re = (p1 - static_cast<int>(d3[4 * n + e])) >> 7;
                            int im = (p1 - static_cast<int>(d2[4 * n + e])) >> 7;
                            if (j <= lim) {
                                if (p.accumulate) {
                                    const int2 o = ptx::ld_global_v2(dst);
                                    re += o.x;
                                    im += o.y;
                                }
                                ptx::st_global_v2(dst, make_int2(re, im));
                            }
                        }
                    }
                }
            }
            // all TMEM reads of this warp are done: hand the accumulators back to the MMA issuer
            tc_release_tmem(lane, bar_tempty, false);
        }
    } else if (warp >= 8) {
        // ===================== unpack warps (S1): raw [t][128 B] boxes -> six 128B-swizzled planes =====================
        // lane -> (row t, 16-byte chunk qc of the row's 128 inputs): a warp reads 4 rows = 512 contiguous raw bytes and
        // writes, per plane, 4 swizzled rows (every bank once)
        const int uw = warp - 8, tl4 = static_cast<int>(lane >> 3), qc = static_cast<int>(lane & 7);
        uint32_t rstage = 0, rphase = 0, ostage = 0, ophase = 0;
        for (uint32_t it = 0;; ++it) {
            const long long w = ring.get<true>(it, lane);
            if (w < 0) break;
            const PrWhere tl = pr_decode(w, p.tiles_per_chan);
            const bool diag = tl.R == tl.Cb;
            for (int kb = 0; kb < nkb; ++kb) {
                ptx::mbar_wait(bar_rfull + 8 * rstage, rphase);
                ptx::mbar_wait(bar_empty + 8 * ostage, ophase ^ 1);
                const uint32_t rsrc = raw_base + rstage * G4_RAW_STAGE;
                const uint32_t odst = op_base + ostage * G4_OP_STAGE;
#pragma unroll
                for (int t = uw * 4 + tl4; t < G4_KT; t += 4 * G4_UNPACK_WARPS) {
                    const uint32_t so = static_cast<uint32_t>(t * 128 + ((qc ^ (t & 7)) << 4));   // swizzled place of the chunk
                    uint32_t wa[4], wb[4];
                    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                 : "=r"(wa[0]), "=r"(wa[1]), "=r"(wa[2]), "=r"(wa[3])
                                 : "r"(rsrc + t * 128 + qc * 16));
                    if (diag) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) wb[u] = wa[u];
                    } else {
                        asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                                     : "=r"(wb[0]), "=r"(wb[1]), "=r"(wb[2]), "=r"(wb[3])
                                     : "r"(rsrc + G4_PLANE + t * 128 + qc * 16));
                    }
                    uint32_t o[6][4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        g4_widen<true>(wa[u], o[0][u], o[1][u], o[2][u]);
                        g4_widen<false>(wb[u], o[3][u], o[4][u], o[5][u]);
                    }
#pragma unroll
                    for (int q = 0; q < 6; ++q)
                        asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(odst + q * G4_PLANE + so), "r"(o[q][0]),
                                     "r"(o[q][1]), "r"(o[q][2]), "r"(o[q][3])
                                     : "memory");
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
