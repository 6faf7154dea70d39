// xcorr_common.cuh -- pieces shared by the tensor-core kernels of the X-engine (xcorr_pair.cuh, xcorr_few.cuh):
// kernel parameters, UMMA descriptors, the tile-index ring, the S4 epilogue chunk and the S1 relayout role.
//
// Real embedding: a span row x[t][c][0..N) of ci8 samples is, byte for byte, the
// int8 row z[t][0..2N) with z[2i] = re_i, z[2i+1] = im_i.  The real Gram matrix
//     G[m][n] = sum_t z[t][m] * z[t][n]                       (int8 x int8 -> int32, exact)
// holds every product the complex visibility needs (include/bfxcorr.h):
//     Re V[i][j] = G[2i][2j]   + G[2i+1][2j+1]
//     Im V[i][j] = G[2i+1][2j] - G[2i][2j+1]
// so no operand negation is needed (kind::i8 has none) and the extreme code -128 stays exact.
// z is "MN-major" for both MMA operands (the time axis is K): a TMA box {128 bytes of m, 1 channel, KT samples}
// lands in shared memory as a 128B-swizzled K-stack of 8-row atoms, exactly the canonical MN-major SWIZZLE_128B
// layout a UMMA shared-memory descriptor describes.
//
// Steps:  S1 unpack-and-transpose = relayout warps -> L2-resident ring -> TMA (pair kernel),
// or TMA -> unpack warps (few-input kernel);  S2 = dynamic hand-out of lower-triangle tiles;  S3 = tcgen05.mma
// kind::i8, int32 accumulators resident in TMEM for the whole span;  S4 = TMEM -> registers -> 2x2 combine
// (lane-pair shuffles) -> shared staging -> bulk store / L2 reduce-add into the packed triangle.
#pragma once
#include <cstdint>
#include <cuda.h>
#include "ptx_sm100.cuh"

namespace bfx {

// ---- tile geometry ----------------------------------------------------------------------------
// L2 eviction hints (A/B measured, profiles/round1.md): ring slabs evict_last, span reads and visibility writes evict_first
#ifndef BFX_KT
#define BFX_KT 128
#endif
constexpr int TC_KT = BFX_KT;   // samples per pipeline stage (TC_KT / 32 MMAs of K = 32); one TMA box = TC_KT rows
constexpr int TC_BOX_BYTES = TC_KT * 128;        // one operand box: KT rows of 128 bytes
constexpr int TC_CJ = 64;                        // visibilities (columns j) per epilogue chunk
constexpr int TC_STG_PITCH = TC_CJ * 8 + 8;      // staging row pitch: 130 words -> 16 rows hit 16 distinct bank pairs
constexpr int TC_STG_BUF_BYTES = 16 * TC_STG_PITCH;   // one warp's 16 rows x 64 visibilities
constexpr int TC_STG_WARP_BYTES = 2 * TC_STG_BUF_BYTES;  // double buffered against the asynchronous bulk copies
constexpr int TC_STG_BYTES = 4 * TC_STG_WARP_BYTES;
constexpr int TC_TMEM_COLS = 512;                // two 256-column accumulators

struct TcParams {
    int32_t* out;
    int ninputs, nchan, ntime;
    int tiles_per_chan;
    long long ntiles;  // tiles_per_chan * nchan
    int accumulate;
    unsigned long long* sched;  // [0] next tile to hand out, [1] CTAs finished (self-resetting, see tc_next_tile)
    // ---- S1 fused into the pair kernel: the operands are read from a ring `z` of ring_w channel
    // slabs, z[c % ring_w][t][2 i + part] int8, that the relayout warps fill from the span `x`
    // ahead of the tiles being contracted.  ready[c] / done[c] count, over all launches of the
    // plan, the relayout units written for channel c / the tiles of channel c whose loads have landed.
    const uint8_t* x;
    uint8_t* z;
    int row_in;             // bytes of one (t, c) row of the span
    int ring_w;
    int rl_nx, rl_units;    // 1 KiB pieces per row; relayout units per channel = rl_nx * ceil(ntime / rl_rows)
    int rl_rows;            // samples per relayout unit (a unit is about 8 KiB of span)
    int rl_row_out;         // bytes of one (t, c) row in the ring
    unsigned long long* ready;
    unsigned long long* done;
    unsigned long long epoch;  // 1, 2, ... : launch number of this plan
};

#ifndef BFX_RL_ROWS
#define BFX_RL_ROWS 8
#endif
#ifndef BFX_RL_SLEEP
#define BFX_RL_SLEEP 500
#endif
constexpr int RL_ROWS = BFX_RL_ROWS;      // samples per relayout unit (4 rounds of 16 loads per lane, one release per unit)
constexpr int RL_WARPS = 8;      // relayout warps per CTA
constexpr int RL_XBYTES = 1024;  // span bytes of one row piece per relayout unit

#ifndef BFX_TC_RING
#define BFX_TC_RING 4
#endif
constexpr int TC_RING = BFX_TC_RING;  // depth of the per-CTA ring that passes scheduled tile indices between warp roles

// UMMA shared-memory descriptor, MN-major, SWIZZLE_128B:
//   bits [0,14) start >> 4 | [16,30) LBO >> 4 (pitch between 128-byte m-blocks) |
//   [32,46) SBO >> 4 (pitch between 8-row K groups = 1024 B) | [46,48) version 1 | [61,64) layout 2
__device__ __forceinline__ uint64_t tc_smem_desc(uint32_t saddr, uint32_t lbo_bytes)
{
    uint64_t d = 0;
    d |= static_cast<uint64_t>((saddr >> 4) & 0x3FFF);
    d |= static_cast<uint64_t>((lbo_bytes >> 4) & 0x3FFF) << 16;
    d |= static_cast<uint64_t>((1024u >> 4) & 0x3FFF) << 32;
    d |= static_cast<uint64_t>(1) << 46;
    d |= static_cast<uint64_t>(2) << 61;
    return d;
}

// UMMA instruction descriptor: dense, no saturate, D = S32, A = B = signed int8, both MN-major.
__host__ __device__ constexpr uint32_t tc_instr_desc(int m, int n)
{
    return (2u << 4) | (1u << 7) | (1u << 10) | (1u << 15) | (1u << 16) | (static_cast<uint32_t>(n >> 3) << 17) |
           (static_cast<uint32_t>(m >> 4) << 24);
}

// S2, device side: tiles are handed out in table order (channel-major) by one global counter, so at any
// moment the CTAs work on a window of ~num_sms consecutive tiles = a few channels whose slabs stay in L2,
// however unequal the tiles are.  The producer lane fetches an index and publishes it to the other warp
// roles of its CTA through a small shared-memory ring.
struct TcRing {
    uint32_t bar_sfull, bar_sempty, ring_base;

    __device__ __forceinline__ void publish(uint32_t n, long long w) const
    {
        const uint32_t slot = n % TC_RING;
        asm volatile("st.shared.s64 [%0], %1;" ::"r"(ring_base + 8 * slot), "l"(w) : "memory");
        ptx::mbar_arrive(bar_sfull + 8 * slot);
    }
    __device__ __forceinline__ void wait_free(uint32_t n) const
    {
        ptx::mbar_wait(bar_sempty + 8 * (n % TC_RING), ((n / TC_RING) & 1) ^ 1);
    }
    // WARP: called by a converged warp (lane 0 releases the slot); else by a single lane
    template <bool WARP>
    __device__ __forceinline__ long long get(uint32_t n, uint32_t lane) const
    {
        const uint32_t slot = n % TC_RING;
        ptx::mbar_wait(bar_sfull + 8 * slot, (n / TC_RING) & 1);
        // lane 0 reads; the broadcast cannot issue before the load has returned, so the arrival that lets the
        // producer rewrite the slot never overtakes the read (see PrRing::get in xcorr_pair.cuh, where it did)
        long long w = 0;
        if (!WARP || lane == 0)
            asm volatile("ld.shared.s64 %0, [%1];" : "=l"(w) : "r"(ring_base + 8 * slot) : "memory");
        if (WARP) w = __shfl_sync(0xffffffffu, w, 0);
        if (!WARP || lane == 0) ptx::mbar_arrive(bar_sempty + 8 * slot);
        return w;
    }
};

// ===================== one epilogue chunk (S4): 32 TMEM lanes x 128 columns -> 16 rows x 64 visibilities ==========
// TMEM lane = real row m = 2 i + part of the A block, so lanes (2k, 2k+1) hold the re and im rows of input row
// i0 + k.  One shuffle per column pair forms Re V (even lane) / Im V (odd lane); both lanes store their 4-byte
// half of the visibility into a per-warp staging row (conflict free: pitch = 130 words).  Lanes 0..15 then each
// own one packed-triangle row segment of <= 64 visibilities and hand it to the TMA unit: a bulk store
// (accumulate = 0) or a bulk int32 reduce-add performed at the L2 (accumulate != 0), so the old values never
// travel to the SM.  Bulk copies need 16-byte alignment but triangle rows are only 8-byte aligned: a staging row
// is placed in a slot of the same address parity as its global start (rows i = 1, 2 mod 4 start on an odd
// visibility; i0 is a multiple of 16, jb of 64) and an odd head / tail visibility goes out as a scalar store / red.
// release_bar != 0: local shared address of the "accumulator drained" barrier to arrive on (cluster address of
// the leader CTA's barrier in the pair kernel) once this warp's TMEM reads are done.
template <bool SHIFT8, bool REMOTE_RELEASE = false, int PENDING = 1, bool GROUPED = false>
__device__ __forceinline__ void tc_epilogue_chunk(const TcParams& p, uint32_t lane, uint32_t tcol, uint32_t stg_buf,
                                                  int32_t* out_c, int i0, int jb, uint32_t release_bar)
{
    // Real rows / columns of the Gram matrix come interleaved (re0 im0 re1 im1 ...: the raw ci8 bytes) or, GROUPED,
    // four at a time (re0..re3 im0..im3: what the ci4 unpack of xcorr_few.cuh writes without byte permutes); the
    // partner lane / column holding the other part of the same input is then 4 away instead of 1.
    const uint32_t par = GROUPED ? (lane >> 2) & 1 : lane & 1;   // 0: re row of its input, 1: im row
    const int sgn = par ? -1 : 1;
    const uint32_t krow = GROUPED ? 4 * (lane >> 3) + (lane & 3) : lane >> 1;
    const uint32_t wr_off = (krow ^ ((krow >> 1) & 1)) * TC_STG_PITCH + 4 * par;
    // the bulk group that last read this staging buffer (two chunks ago with two buffers: PENDING = 1; the previous
    // chunk with a single buffer: PENDING = 0) must be done with it
    if (lane < 16) ptx::bulk_wait_read<PENDING>();
    __syncwarp();
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        uint32_t g[32];
        ptx::tmem_ld_32x32b_x32(tcol + q * 32, g);
        ptx::tmem_ld_wait();
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            // columns (re_j, im_j) of visibility column j = 16 q + k
            int ge = static_cast<int>(g[GROUPED ? 8 * (k >> 2) + (k & 3) : 2 * k]);
            int go = static_cast<int>(g[GROUPED ? 8 * (k >> 2) + 4 + (k & 3) : 2 * k + 1]);
            if (SHIFT8) { ge >>= 8; go >>= 8; }       // G came out scaled by 16*16, exactly
            const int v = __shfl_xor_sync(0xffffffffu, go, GROUPED ? 4 : 1);
            // even lane: Re V[i][j] = G[2i][2j] + G[2i+1][2j+1]; odd lane: Im V[i][j] = G[2i+1][2j] - G[2i][2j+1]
            const int val = ge + sgn * v;
            asm volatile("st.shared.s32 [%0], %1;" ::"r"(stg_buf + wr_off + (q * 16 + k) * 8), "r"(val) : "memory");
        }
    }
    if (release_bar) {
        // all TMEM reads of this accumulator are done: hand it back to the MMA issuer
        ptx::tc_fence_before();
        __syncwarp();
        if (lane == 0) {
            if (REMOTE_RELEASE) ptx::mbar_arrive_cluster_addr(release_bar); else ptx::mbar_arrive(release_bar);
        }
    }
    __syncwarp();
    // (Coalesced st.global / red from the staging rows instead of bulk copies was measured slower: 2.38 / 3.10 vs
    // 2.27 / 2.42 ms on cfg3, profiles/round1.md.)
    ptx::fence_proxy_async_smem();  // staging writes -> visible to the bulk-copy engine
    __syncwarp();
    if (lane < 16) {
        const uint32_t own_off = (lane ^ ((lane >> 1) & 1)) * TC_STG_PITCH;  // lanes 0..15: slot of row `lane`
        const int i_own = i0 + static_cast<int>(lane);
        int n = i_own + 1 - jb;       // row i holds columns j <= i only (S2 masking of diagonal tiles)
        n = n > TC_CJ ? TC_CJ : n;
        if (i_own >= p.ninputs) n = 0;
        if (n > 0) {
            const long long e0 = static_cast<long long>(i_own) * (i_own + 1) / 2 + jb;
            int32_t* const g0 = out_c + 2 * e0;
            const uint32_t s0 = stg_buf + own_off;
            const int head = static_cast<int>(e0 & 1);
            const int nbulk = (n - head) & ~1;
            if (head) {
                int2 v;
                asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(s0));
                if (p.accumulate) ptx::red_add_global_v2(g0, v); else ptx::st_global_v2(g0, v);
            }
            if (nbulk > 0) {
                // the visibilities stream through the L2 once per span: let them go first, the S1 ring should stay
                if (p.accumulate) ptx::bulk_reduce_add_s32_hint(g0 + 2 * head, s0 + 8 * head, 8u * nbulk, ptx::policy_evict_first());
                else ptx::bulk_store_hint(g0 + 2 * head, s0 + 8 * head, 8u * nbulk, ptx::policy_evict_first());
            }
            if (head + nbulk < n) {
                int2 v;
                asm volatile("ld.shared.v2.s32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(s0 + 8 * (n - 1)));
                if (p.accumulate) ptx::red_add_global_v2(g0 + 2 * (n - 1), v); else ptx::st_global_v2(g0 + 2 * (n - 1), v);
            }
        }
        ptx::bulk_commit();
    }
}

// ===================== register-direct epilogue (S4): 32 TMEM lanes x 128 columns -> 16 rows x 64 visibilities =====
// The staged epilogue above hands every row segment to the TMA unit, which it shares with the operand loads: on cfg3
// its warps spent 47 % of their time in the serialised UBLKCP issue loop (profiles/round2.md).  Here the visibilities go
// from registers to global memory through the LSU instead, so the TMA unit only loads operands and no staging memory
// is needed.  tcgen05.ld 16x256b gives thread T (t8 = T / 4, t4 = T % 4) two columns (re_j, im_j) of TMEM lane t8 and of
// lane t8 + 8; lanes come in (re_i, im_i) pairs, so threads T and T ^ 4 hold the four Gram entries of visibility (i, j)
// for input row t8 / 2 and for input row t8 / 2 + 4.  One exchange (two shuffles) gives the even-lane thread the
// complete visibility of the first row and the odd-lane thread that of the second; each stores its 8 bytes, the four
// threads of a quad covering 32 contiguous bytes of one packed-triangle row.  accumulate != 0: the old values are loaded
// (8-byte loads issued before the wait for the accumulator, the tile's rows were prefetched into the L2 a tile earlier)
// and added in registers -- a read-modify-write by the one warp that owns the segment, so no atomics are needed.
// tcol: TMEM address of (first lane of this warp, first column of the 128-column range).
__device__ __forceinline__ void tc_release_tmem(uint32_t lane, uint32_t release_bar, bool remote)
{
    ptx::tc_fence_before();
    __syncwarp();
    if (lane == 0) {
        if (remote) ptx::mbar_arrive_cluster_addr(release_bar); else ptx::mbar_arrive(release_bar);
    }
}

template <bool SHIFT8, bool REMOTE_RELEASE>
__device__ __forceinline__ void tc_epilogue_direct(const TcParams& p, uint32_t lane, uint32_t tcol, int32_t* out_c, int i0, int jb,
                                                   uint32_t tfull_bar, uint32_t tfull_phase, uint32_t release_bar)
{
    const int t4 = static_cast<int>(lane & 3), t8 = static_cast<int>(lane >> 2);
    const bool even = (t8 & 1) == 0;
    const int rowoff = (t8 >> 1) + 4 * (t8 & 1);   // input row of this thread inside an 8-row half
    int32_t* rowp[2];
    int rel[2];   // column offset (inside the range, for n = 0) up to which this thread's row has entries: j <= i
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
        const int irow = i0 + 8 * hh + rowoff;
        rowp[hh] = out_c + 2 * (static_cast<long long>(irow) * (irow + 1) / 2 + jb + t4);
        rel[hh] = irow < p.ninputs ? irow - jb - t4 : -1;
    }
    int2 old[2][2][8];
    if (p.accumulate) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh)
#pragma unroll
            for (int cp = 0; cp < 2; ++cp)
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const int off = 32 * cp + 4 * n;
                    old[hh][cp][n] = off <= rel[hh] ? ptx::ld_global_v2(rowp[hh] + 2 * off) : make_int2(0, 0);
                }
    }
    ptx::mbar_wait(tfull_bar, tfull_phase);
    ptx::tc_fence_after();
#pragma unroll
    for (int hh = 0; hh < 2; ++hh) {
#pragma unroll
        for (int cp = 0; cp < 2; ++cp) {
            // warp-uniform: the piece has an entry on or below the diagonal, and its rows exist
            const bool active = jb + 32 * cp <= i0 + 8 * hh + 7 && i0 + 8 * hh < p.ninputs;
            uint32_t g[32];
            if (active) {
                ptx::tmem_ld_16x256b_x8(tcol + (static_cast<uint32_t>(16 * hh) << 16) + 64 * cp, g);
                ptx::tmem_ld_wait();
            }
            if (hh == 1 && cp == 1 && release_bar) tc_release_tmem(lane, release_bar, REMOTE_RELEASE);   // this warp's TMEM reads are done
            if (active) {
#pragma unroll
                for (int n = 0; n < 8; ++n) {
                    const int a0 = static_cast<int>(g[4 * n]), a1 = static_cast<int>(g[4 * n + 1]);
                    const int b0 = static_cast<int>(g[4 * n + 2]), b1 = static_cast<int>(g[4 * n + 3]);
                    // even lanes (re rows) keep lane t8's pair and send lane t8 + 8's; odd lanes (im rows) the reverse
                    const int x0 = __shfl_xor_sync(0xffffffffu, even ? b0 : a0, 4);
                    const int x1 = __shfl_xor_sync(0xffffffffu, even ? b1 : a1, 4);
                    // Re V = G[re_i][re_j] + G[im_i][im_j],  Im V = G[im_i][re_j] - G[re_i][im_j]
                    int re = (even ? a0 : b1) + (even ? x1 : x0);
                    int im = (even ? x0 : b0) - (even ? a1 : x1);
                    if (SHIFT8) { re >>= 8; im >>= 8; }   // G came out scaled by 16 * 16, exactly
                    const int off = 32 * cp + 4 * n;
                    if (p.accumulate) { re += old[hh][cp][n].x; im += old[hh][cp][n].y; }
                    if (off <= rel[hh]) ptx::st_global_v2(rowp[hh] + 2 * off, make_int2(re, im));
                }
            }
        }
    }
}

// accumulate != 0: pull the old visibilities of (16 rows from i0) x (columns j0 .. j0 + ncol) into the L2 ahead of
// the loads of tc_epilogue_direct.  Lane l covers half of row i0 + l / 2.
__device__ __forceinline__ void tc_prefetch_old(const TcParams& p, uint32_t lane, const int32_t* out_c, int i0, int j0, int ncol)
{
    const int irow = i0 + static_cast<int>(lane >> 1);
    int n = irow + 1 - j0;
    n = n > ncol ? ncol : n;
    if (irow >= p.ninputs || n <= 0) return;
    const char* const beg = reinterpret_cast<const char*>(out_c + 2 * (static_cast<long long>(irow) * (irow + 1) / 2 + j0));
    const char* const end = beg + 8 * n;
    const char* q = reinterpret_cast<const char*>(reinterpret_cast<uintptr_t>(beg) & ~static_cast<uintptr_t>(127)) + 128 * (lane & 1);
    for (; q < end; q += 256) ptx::prefetch_l2_line(q);
}

// ===================== relayout warps (S1: unpack-and-transpose, span -> ring z) =====================
// Shared by the 1-CTA and the CTA-pair kernels; run by whole warps.
__device__ __forceinline__ void tc_relayout_role(const TcParams& p, uint32_t lane)
{
    // ===================== relayout warps (S1: unpack-and-transpose, span -> ring z) =====================
    // A unit = rl_rows samples x one 1 KiB piece of the (t, c) row of channel cc: read with coalesced 16-byte
    // loads (each span byte exactly once per launch) and written with 16-byte stores to the channel's slab: ci8
    // bytes are already the int8 (re, im) pairs, ci4 bytes stay packed (xcorr_pair4.cuh widens them in shared
    // memory).  Each warp works on its own units.
    const long long src_pitch = static_cast<long long>(p.nchan) * p.row_in;
    const int row_out = p.rl_row_out;  // bytes of one (t, c) row in the ring: 2 N (int8 pairs) or N (packed ci4)
    auto do_unit = [&](int cc, int u) {
        if (cc >= p.ring_w) {
            // the slab is still owned by channel cc - ring_w until all of its tiles have loaded their operands
            if (lane == 0) {
                const unsigned long long want = p.epoch * static_cast<unsigned long long>(p.tiles_per_chan);
                uint32_t spins = 0;
                while (ptx::ld_acquire_u64(p.done + (cc - p.ring_w)) < want) {
                    __nanosleep(BFX_RL_SLEEP);
                    if (++spins > (1u << 24)) __trap();
                }
            }
            __syncwarp();
        }
        const int t0 = (u / p.rl_nx) * p.rl_rows;
        const int xb0 = (u % p.rl_nx) * RL_XBYTES;
        const int nt = min(p.rl_rows, p.ntime - t0);
        const int nv = min(RL_XBYTES, p.row_in - xb0) >> 4;  // 16-byte vectors per row piece
        const int total = nt * nv;
        const int nv_shift = (nv & (nv - 1)) == 0 ? 31 - __clz(nv) : -1;  // rows are usually 64 vectors: avoid the division
        const uint8_t* src = p.x + (static_cast<long long>(t0) * p.nchan + cc) * p.row_in + xb0;
        uint8_t* dst = p.z + (static_cast<long long>(cc % p.ring_w) * p.ntime + t0) * row_out + xb0;
        constexpr int U = 16;
        for (int base = static_cast<int>(lane); base < total; base += U * 32) {
            uint4 v[U];
#pragma unroll
            for (int k = 0; k < U; ++k) {
                const int idx = base + 32 * k;
                const int r = nv_shift >= 0 ? idx >> nv_shift : idx / nv;
                if (idx < total) v[k] = ptx::ld_global_stream_v4(src + r * src_pitch + (idx - r * nv) * 16);
            }
#pragma unroll
            for (int k = 0; k < U; ++k) {
                const int idx = base + 32 * k;
                const int r = nv_shift >= 0 ? idx >> nv_shift : idx / nv;
                const int vi = idx - r * nv;
                // (eviction hints on these loads / stores were measured harmful: cfg3 accumulate span 2.49 vs 2.34 ms)
                if (idx < total) ptx::st_global_v4(dst + static_cast<long long>(r) * row_out + vi * 16, v[k]);
            }
        }
        // publish: every lane's stores are ordered before lane 0's release by the warp barrier (the release is
        // cumulative), and made visible to the TMA (async proxy) readers by the proxy fence
        ptx::fence_proxy_async_global();
        __syncwarp();
        if (lane == 0) ptx::red_release_add_u64(p.ready + cc, 1ull);
    };
    // Units are handed out channel-major by one global counter, independently of the tile scheduler: the relayout
    // warps of all CTAs run ahead of the contraction as far as the ring allows (do_unit waits for the slab's
    // previous channel to be done), so the span's DRAM / address-translation latency is off the critical path.
    const long long total_units = static_cast<long long>(p.nchan) * p.rl_units;
    // (Prefetching a unit's rows into the L2 two units ahead was measured slower, 2.32 vs 2.18 ms on cfg3: the
    // kernel is bound by L2 throughput, not by the latency of these loads.)
    for (;;) {
        long long u = 0;
        if (lane == 0) u = static_cast<long long>(atomicAdd(p.sched + 2, 1ull));
        u = __shfl_sync(0xffffffffu, u, 0);
        if (u >= total_units) break;
        do_unit(static_cast<int>(u / p.rl_units), static_cast<int>(u % p.rl_units));
    }
}

}  // namespace bfx
