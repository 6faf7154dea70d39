// bfxcorr.cu -- host side of the C ABI declared in include/bfxcorr.h: plan construction (tile table,
// TMA tensor map), launch of the sm_100a kernels, status codes.  No CPU compute path exists here.
#include <cstdint>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <new>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/bfxcorr.h"
#include "xcorr_simt.cuh"
#include "xcorr_dump.cuh"
#include "mem_probe.cuh"
#include "xcorr_few.cuh"
#include "xcorr_pair.cuh"
#include "xcorr_pair4.cuh"
#include "xcorr_stripe.cuh"
#include "xcorr_gauss4.cuh"
#include "xcorr_common.cuh"

namespace {

using bfx::TcParams;

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

constexpr uint32_t kMagic = 0xBFC0DE01u;

#ifndef BFX_SPAN_PROMO
#define BFX_SPAN_PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_128B
#endif
#ifndef BFX_STRIPE
#define BFX_STRIPE 1
#endif
#ifndef BFX_DIRECT_MAX_BLK
#define BFX_DIRECT_MAX_BLK 8
#endif
#ifndef BFX_DIRECT_STRIDE_KB
#define BFX_DIRECT_STRIDE_KB 1024
#endif
// ci4 pair spans through the S1 ring (0 = always in place; probe knob).  The ring was switched off for a few commits
// while accumulating launches of xcorr_pair4_kernel lost tiles; the cause was the tile-index ring (PrRing::get in
// xcorr_pair.cuh: the slot read was not complete before the remote arrival), fixed there: profiles/round1.md.
#ifndef BFX_P4_RING
#define BFX_P4_RING 1
#endif
#ifndef BFX_ST_AHEAD_MB
#define BFX_ST_AHEAD_MB 16
#endif

}  // namespace

struct bfXcorr_impl {
    uint32_t magic;
    int ninputs, nchan, ntime, dtype;
    int algo;
    int device;
    int num_sms;
    int last_cuda_error;
    int last_launch_count;
    // S2: lower-triangle tile table (device copy) for the tcgen05 kernel
    bool pair;            // ninputs > 64: CTA-pair kernel with fused S1; else the few-input kernel
    bool stripe;          // ci8 pair spans of <= 1024 samples: resident-A stripes (xcorr_stripe.cuh)
    int tiles_per_chan;
    unsigned long long* d_sched;  // dynamic tile scheduler state, re-armed by the kernel itself
    EncodeTiledFn encode;
    // S1: ring of ring_w channel slabs z[c % ring_w][ntime][2*ninputs] int8, filled ahead of the
    // contraction by the relayout warps of the same kernel (NULL: operands come from the span itself)
    uint8_t* d_z;
    int ring_w;
    unsigned long long* d_flags;  // ready[nchan], done[nchan]
    unsigned long long epoch;     // fused launches so far
    // bfXcorrExecuteHost: two device staging buffers for spans and private copy streams, so that the host->device
    // copy of span n+1 overlaps the contraction of span n and the device->host copy of the visibilities
    // (the GPU analogue of the paper's pipeline parallelism)
    void* d_stage_in[2];
    cudaStream_t s_h2d, s_d2h;
    cudaEvent_t ev_h2d[2], ev_comp[2], ev_d2h;
    unsigned long long host_calls;
    bool host_ready;   // staging buffers, copy streams and events all exist
};

namespace {

bool valid(bfXcorr p) { return p != nullptr && p->magic == kMagic; }

int cuda_fail(bfXcorr p, cudaError_t e)
{
    if (p) p->last_cuda_error = static_cast<int>(e);
    return e == cudaErrorMemoryAllocation ? BF_XCORR_MEM_ALLOC_FAILED : BF_XCORR_DEVICE_ERROR;
}

unsigned long long bytes_per_sample(int dtype) { return dtype == BF_XCORR_CI4 ? 1ull : 2ull; }

unsigned long long input_bytes(bfXcorr p)
{
    return static_cast<unsigned long long>(p->ntime) * p->nchan * p->ninputs * bytes_per_sample(p->dtype);
}

unsigned long long output_bytes(bfXcorr p)
{
    const unsigned long long n = p->ninputs;
    return static_cast<unsigned long long>(p->nchan) * (n * (n + 1) / 2) * 8ull;
}

// Where the tensor-core kernel reads its operands from: the caller's span x[t][c][...] itself (direct), or the
// plan's ring of channel-major int8 slabs z[c % W][t][...] written by the relayout warps (xcorr_common.cuh).
// Both are addressed with the same coordinates (byte in row, channel, sample); only the strides differ.
struct OperandSource {
    const void* base;
    unsigned long long row;          // bytes per (sample, channel) row
    unsigned long long chan_stride;  // bytes between channels
    unsigned long long time_stride;  // bytes between samples
    bool raw_ci4;                    // rows hold ci4 bytes (unpacked on chip), else int8 (re, im) pairs
};

OperandSource direct_source(bfXcorr p, const void* in)
{
    const unsigned long long row = static_cast<unsigned long long>(p->ninputs) * bytes_per_sample(p->dtype);
    return OperandSource{in, row, row, row * static_cast<unsigned long long>(p->nchan), p->dtype == BF_XCORR_CI4};
}

// ring rows: int8 (re, im) pairs for ci8 spans, the packed bytes themselves for ci4 spans (xcorr_pair4.cuh)
unsigned long long ring_row_bytes(bfXcorr p) { return (p->dtype == BF_XCORR_CI4 ? 1ull : 2ull) * p->ninputs; }

OperandSource ring_source(bfXcorr p)
{
    const unsigned long long row = ring_row_bytes(p);
    return OperandSource{p->d_z, row, row * static_cast<unsigned long long>(p->ntime), row, false};
}

int encode_map(bfXcorr p, CUtensorMap* m, CUtensorMapDataType type, const OperandSource& src, unsigned elem_bytes,
               unsigned box_elems, CUtensorMapSwizzle swz, int nchan_src, unsigned box_chan = 1, unsigned box_rows = bfx::TC_KT)
{
    const cuuint64_t dims[3] = {src.row / elem_bytes, static_cast<cuuint64_t>(nchan_src), static_cast<cuuint64_t>(p->ntime)};
    const cuuint64_t strides[2] = {src.chan_stride, src.time_stride};
    const cuuint32_t box[3] = {box_elems, box_chan, box_rows};
    const cuuint32_t estr[3] = {1u, 1u, 1u};
    const CUresult r = p->encode(m, type, 3, const_cast<void*>(src.base), dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                 swz, src.base == p->d_z ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : BFX_SPAN_PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        p->last_cuda_error = static_cast<int>(cudaErrorInvalidValue);
        return BF_XCORR_DEVICE_ERROR;
    }
    return BF_XCORR_OK;
}

template <bool CI4>
int launch_tcgen05(bfXcorr p, const void* in, void* out, int accumulate, cudaStream_t stream)
{
    const bool fused = p->d_z != nullptr;
    const bool pair = p->pair;
    const bool few = !pair;  // ninputs <= 64: xcorr_few.cuh, FW_NC channels per CTA tile
    const OperandSource src = fused ? ring_source(p) : direct_source(p, in);
    CUtensorMap tmap;
    // operand boxes: 64 inputs x 1 channel x TC_KT samples (128 bytes of int8 pairs); few-input ci4: whole raw rows of
    // FW_NC adjacent channels x FW_KT samples
    const bool pair4 = pair && p->dtype == BF_XCORR_CI4;  // packed ring, unpacked in shared memory
    const int st = pair4 ? encode_map(p, &tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, src, 1, 64u, CU_TENSOR_MAP_SWIZZLE_NONE, fused ? p->ring_w : p->nchan)
                   : few ? encode_map(p, &tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, src, 1, static_cast<unsigned>(src.row),
                                    CU_TENSOR_MAP_SWIZZLE_NONE, p->nchan, bfx::FW_NC, bfx::FW_KT)
                       : encode_map(p, &tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, src, 1, CI4 ? 64u : 128u,
                                    CI4 ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B, fused ? p->ring_w : p->nchan);
    if (st != BF_XCORR_OK) return st;
    TcParams prm;
    std::memset(&prm, 0, sizeof(prm));
    prm.out = static_cast<int32_t*>(out);
    prm.ninputs = p->ninputs;
    prm.nchan = p->nchan;
    prm.ntime = p->ntime;
    prm.tiles_per_chan = p->tiles_per_chan;
    prm.ntiles = static_cast<long long>(p->tiles_per_chan) * p->nchan;
    prm.accumulate = accumulate ? 1 : 0;
    prm.sched = p->d_sched;
    prm.ring_w = p->nchan;   // no ring: the operand source is the span itself
    if (fused) {
        // ci4 spans keep their bytes in the ring (xcorr_pair4.cuh widens them in shared memory)
        prm.rl_row_out = static_cast<int>(ring_row_bytes(p));
        prm.x = static_cast<const uint8_t*>(in);
        prm.z = p->d_z;
        prm.row_in = static_cast<int>(p->ninputs * bytes_per_sample(p->dtype));
        prm.ring_w = p->ring_w;
        prm.rl_nx = (prm.row_in + bfx::RL_XBYTES - 1) / bfx::RL_XBYTES;
        // a unit = rl_rows samples x one row piece of <= 1 KiB: about 8 KiB, one round of 16 loads per lane
        const int piece = prm.row_in < bfx::RL_XBYTES ? prm.row_in : bfx::RL_XBYTES;
        int rows = bfx::RL_ROWS * bfx::RL_XBYTES / piece;
        if (rows > 256) rows = 256;
        prm.rl_rows = rows;
        prm.rl_units = prm.rl_nx * ((p->ntime + rows - 1) / rows);
        prm.ready = p->d_flags;
        prm.done = p->d_flags + p->nchan;
        prm.epoch = p->epoch + 1;   // committed below, once the launch has been accepted
    }
    cudaError_t e = cudaSuccess;
    if (pair) {
        // one cluster of two CTAs per tile in flight
        const bool stripe = p->stripe && !pair4;
        if (stripe) prm.ntiles = static_cast<long long>(p->nchan) * ((p->ninputs + bfx::PR_BLK - 1) / bfx::PR_BLK);  // stripes
        long long pairs = p->num_sms / 2;
        if (prm.ntiles < pairs) pairs = prm.ntiles;
        cudaLaunchConfig_t cfg;
        std::memset(&cfg, 0, sizeof(cfg));
        cfg.gridDim = dim3(static_cast<unsigned>(2 * pairs));
        // stripe kernel variants (xcorr_stripe.cuh): through the S1 ring; in place with the register-direct epilogue
        // (accumulate = 0) or with the staged L2-reduce epilogue (accumulate != 0)
        using StRing = bfx::StCfg<true, false>;
        using StDirect = bfx::StCfg<false, true>;
        using StStaged = bfx::StCfg<false, false>;
        const int st_variant = !stripe ? -1 : fused ? 0 : accumulate ? 2 : 1;
        cfg.blockDim = dim3(pair4 ? bfx::P4_THREADS : st_variant == 0 ? StRing::kThreads : st_variant == 1 ? StDirect::kThreads
                            : st_variant == 2 ? StStaged::kThreads : bfx::PR_THREADS);
        cfg.dynamicSmemBytes = pair4 ? bfx::P4_SMEM_BYTES : st_variant == 0 ? StRing::kSmemBytes : st_variant == 1 ? StDirect::kSmemBytes
                               : st_variant == 2 ? StStaged::kSmemBytes : bfx::PR_SMEM_BYTES;
        cfg.stream = stream;
        cudaLaunchAttribute attr;
        attr.id = cudaLaunchAttributeClusterDimension;
        attr.val.clusterDim.x = 2;
        attr.val.clusterDim.y = 1;
        attr.val.clusterDim.z = 1;
        cfg.attrs = &attr;
        cfg.numAttrs = 1;
        e = pair4             ? cudaLaunchKernelEx(&cfg, bfx::xcorr_pair4_kernel, tmap, prm)
            : st_variant == 0 ? cudaLaunchKernelEx(&cfg, bfx::xcorr_stripe_kernel<true, false>, tmap, prm)
            : st_variant == 1 ? cudaLaunchKernelEx(&cfg, bfx::xcorr_stripe_kernel<false, true>, tmap, prm)
            : st_variant == 2 ? cudaLaunchKernelEx(&cfg, bfx::xcorr_stripe_kernel<false, false>, tmap, prm)
                              : cudaLaunchKernelEx(&cfg, bfx::xcorr_pair_kernel, tmap, prm);
    } else if (few) {
        prm.ntiles = (p->nchan + bfx::FW_NC - 1) / bfx::FW_NC;
        prm.row_in = static_cast<int>(src.row);
        const long long want = prm.ntiles < p->num_sms ? prm.ntiles : p->num_sms;
        bfx::xcorr_few_kernel<CI4><<<dim3(static_cast<unsigned>(want)), bfx::FW_THREADS, bfx::FwCfg<CI4>::kSmemBytes, stream>>>(tmap, prm);
    }
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e);
    if (fused) p->epoch += 1;   // the ready[] / done[] counters now run one launch further
    p->last_launch_count += 1;
    return BF_XCORR_OK;
}

// xcorr_gauss4.cuh: ci4 spans with the three-multiplication complex product, one CTA per 128 x 128-input tile, in place
int launch_gauss4(bfXcorr p, const void* in, void* out, int accumulate, cudaStream_t stream)
{
    CUtensorMap tmap;
    const int st = encode_map(p, &tmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, direct_source(p, in), 1, 128u, CU_TENSOR_MAP_SWIZZLE_NONE,
                              p->nchan, 1, bfx::G4_KT);
    if (st != BF_XCORR_OK) return st;
    const int nblk = (p->ninputs + bfx::PR_BLK - 1) / bfx::PR_BLK;
    TcParams prm;
    std::memset(&prm, 0, sizeof(prm));
    prm.out = static_cast<int32_t*>(out);
    prm.ninputs = p->ninputs;
    prm.nchan = p->nchan;
    prm.ntime = p->ntime;
    prm.tiles_per_chan = nblk * (nblk + 1) / 2;
    prm.ntiles = static_cast<long long>(prm.tiles_per_chan) * p->nchan;
    prm.accumulate = accumulate ? 1 : 0;
    prm.sched = p->d_sched;
    const long long want = prm.ntiles < p->num_sms ? prm.ntiles : p->num_sms;
    bfx::xcorr_gauss4_kernel<<<dim3(static_cast<unsigned>(want)), bfx::G4_THREADS, bfx::G4_SMEM_BYTES, stream>>>(tmap, prm);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->last_launch_count += 1;
    return BF_XCORR_OK;
}

// bfXcorrExecuteHost's staging state: released as a whole (also after a partial set-up), pointers nulled
void release_host_state(bfXcorr plan)
{
    for (int b = 0; b < 2; ++b) {
        if (plan->d_stage_in[b]) cudaFree(plan->d_stage_in[b]);
        if (plan->ev_h2d[b]) cudaEventDestroy(plan->ev_h2d[b]);
        if (plan->ev_comp[b]) cudaEventDestroy(plan->ev_comp[b]);
        plan->d_stage_in[b] = nullptr;
        plan->ev_h2d[b] = nullptr;
        plan->ev_comp[b] = nullptr;
    }
    if (plan->ev_d2h) cudaEventDestroy(plan->ev_d2h);
    if (plan->s_h2d) cudaStreamDestroy(plan->s_h2d);
    if (plan->s_d2h) cudaStreamDestroy(plan->s_d2h);
    plan->ev_d2h = nullptr;
    plan->s_h2d = nullptr;
    plan->s_d2h = nullptr;
    plan->host_ready = false;
}

int launch_simt(bfXcorr p, const void* in, void* out, int accumulate, cudaStream_t stream)
{
    const int nb = (p->ninputs + bfx::SIMT_TILE - 1) / bfx::SIMT_TILE;
    const dim3 grid(static_cast<unsigned>(nb * (nb + 1) / 2), static_cast<unsigned>(p->nchan < 65535 ? p->nchan : 65535));
    bfx::xcorr_simt_kernel<<<grid, 256, 0, stream>>>(static_cast<const uint8_t*>(in), static_cast<int32_t*>(out),
                                                     p->ninputs, p->nchan, p->ntime, p->dtype, accumulate ? 1 : 0);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->last_launch_count += 1;
    return BF_XCORR_OK;
}

// ---- bfXcorrExecuteNoAlloc: every kernel's scratch in one static device array (include/bfxcorr.h) ----------------
// layout: [0, 1024) scheduler words | [1024, 1024 + 16 * MAX_RING_CHANNELS) ready[nchan], done[nchan] | S1 ring
constexpr size_t kNaFlagsOff = 1024;
constexpr size_t kNaRingOff = kNaFlagsOff + 16ull * BF_XCORR_NOALLOC_MAX_RING_CHANNELS;
static_assert(kNaRingOff % 1024 == 0, "ring slabs are TMA sources");
static_assert(kNaRingOff + BF_XCORR_NOALLOC_RING_BYTES == BF_XCORR_NOALLOC_SCRATCH_BYTES, "header and layout agree");

// In host code this name is a host-side stand-in, not a device address: na_device_state() asks the runtime for the
// address on the current device (cudaGetSymbolAddress) and the kernels get that pointer.
static __device__ __align__(256) unsigned char g_noalloc_scratch[BF_XCORR_NOALLOC_SCRATCH_BYTES];

struct NaDevice {
    bool ready;
    unsigned char* scratch;   // device address of g_noalloc_scratch on this device
    int num_sms;
};
constexpr int kNaMaxDevices = 64;
NaDevice g_na_device[kNaMaxDevices];   // zero-initialised
EncodeTiledFn g_na_encode = nullptr;
std::mutex g_na_mutex;

// One-time set-up of the current device `dev` (no allocation).  Returns a status; *out valid on BF_XCORR_OK.
int na_device_state(int dev, NaDevice* out)
{
    if (dev < 0 || dev >= kNaMaxDevices) return BF_XCORR_UNSUPPORTED_DEVICE;
    std::lock_guard<std::mutex> lock(g_na_mutex);
    NaDevice& d = g_na_device[dev];
    if (!d.ready) {
        int major = 0, sms = 0;
        if (cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev) != cudaSuccess || major != 10) {
            cudaGetLastError();
            return BF_XCORR_UNSUPPORTED_DEVICE;
        }
        if (cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || sms <= 0) return BF_XCORR_UNSUPPORTED_DEVICE;
        if (!g_na_encode) {
            void* fn = nullptr;
            cudaDriverEntryPointQueryResult qres;
            const cudaError_t eq = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
            if (eq != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) return BF_XCORR_UNSUPPORTED_DEVICE;
            g_na_encode = reinterpret_cast<EncodeTiledFn>(fn);
        }
        void* ptr = nullptr;
        cudaError_t e = cudaGetSymbolAddress(&ptr, g_noalloc_scratch);
        if (e == cudaSuccess && !ptr) e = cudaErrorInvalidSymbol;
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_few_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::FwCfg<true>::kSmemBytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_few_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::FwCfg<false>::kSmemBytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_pair4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::P4_SMEM_BYTES);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::PR_SMEM_BYTES);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<true, false>::kSmemBytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<false, true>::kSmemBytes);
        if (e == cudaSuccess)
            e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<false, false>::kSmemBytes);
        if (e != cudaSuccess) {
            cudaGetLastError();
            return BF_XCORR_DEVICE_ERROR;
        }
        d.scratch = static_cast<unsigned char*>(ptr);
        d.num_sms = sms;
        d.ready = true;
    }
    *out = d;
    return BF_XCORR_OK;
}

}  // namespace

extern "C" {

int bfXcorrCreate(bfXcorr* plan, int ninputs, int nchan, int ntime, int dtype)
{
    if (!plan) return BF_XCORR_INVALID_POINTER;
    *plan = nullptr;
    if (ninputs <= 0 || nchan <= 0 || ntime <= 0 || ntime > 65535) return BF_XCORR_INVALID_ARGUMENT;
    if (dtype != BF_XCORR_CI4 && dtype != BF_XCORR_CI8) return BF_XCORR_INVALID_DTYPE;
    if ((static_cast<unsigned long long>(ninputs) * bytes_per_sample(dtype)) % 16ull != 0) return BF_XCORR_UNSUPPORTED_SHAPE;
    if (ninputs > 32768) return BF_XCORR_UNSUPPORTED_SHAPE;

    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0) {
        cudaGetLastError();
        return BF_XCORR_UNSUPPORTED_DEVICE;
    }
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return BF_XCORR_UNSUPPORTED_DEVICE;
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, dev) != cudaSuccess) return BF_XCORR_UNSUPPORTED_DEVICE;
    if (prop.major != 10) return BF_XCORR_UNSUPPORTED_DEVICE;

    bfXcorr p = new (std::nothrow) bfXcorr_impl;
    if (!p) return BF_XCORR_MEM_ALLOC_FAILED;
    std::memset(p, 0, sizeof(*p));
    p->magic = kMagic;
    p->ninputs = ninputs;
    p->nchan = nchan;
    p->ntime = ntime;
    p->dtype = dtype;
    p->algo = BF_XCORR_ALGO_TCGEN05;
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;

    // cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time libcuda dependency)
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
        delete p;
        return BF_XCORR_UNSUPPORTED_DEVICE;
    }
    p->encode = reinterpret_cast<EncodeTiledFn>(fn);

    // S2: tiles of a channel = 128 x 128-input blocks on or below the diagonal (xcorr_pair.cuh decodes the index);
    // up to 64 inputs: a single 64 x 64 tile per channel (xcorr_few.cuh)
    const bool pair = ninputs > 64;
    p->pair = pair;
    const int nblk = (ninputs + bfx::PR_BLK - 1) / bfx::PR_BLK;
    p->stripe = BFX_STRIPE && pair && dtype == BF_XCORR_CI8 && ntime <= bfx::ST_MAXKB * bfx::TC_KT;
    p->tiles_per_chan = pair ? nblk * (nblk + 1) / 2 : 1;
    if (pair && static_cast<unsigned long long>(p->tiles_per_chan) * nchan >= (1ull << 32)) {
        delete p;
        return BF_XCORR_UNSUPPORTED_SHAPE;
    }
    e = cudaSuccess;
    if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&p->d_sched), 4 * sizeof(unsigned long long));
    if (e == cudaSuccess) e = cudaMemset(p->d_sched, 0, 4 * sizeof(unsigned long long));
    // A channel whose tiles re-read its samples is first rewritten channel-major (S1, tc_relayout_role); with a
    // single tile per channel (ninputs <= 64) every sample is read once anyway and the span is used in place.
    // stripes of few row blocks read the span in place (xcorr_stripe.cuh): no ring, no flags
    // ... and so do ci4 pair spans, and any span whose samples lie close enough together for the TMA's address
    // translation (BFX_DIRECT_STRIDE_KB between consecutive samples of a channel; cfg2: 128 KiB).  Measured
    // (profiles/round1.md): with many row blocks AND a stride of 2 MiB or more the S1 ring still wins.
    const bool near = static_cast<unsigned long long>(nchan) * ninputs * bytes_per_sample(dtype) <= (static_cast<unsigned long long>(BFX_DIRECT_STRIDE_KB) << 10);
    const bool direct = pair && (p->stripe || dtype == BF_XCORR_CI4) &&
                        (nblk <= BFX_DIRECT_MAX_BLK || near || (dtype == BF_XCORR_CI4 && !BFX_P4_RING));
    if (e == cudaSuccess && pair && !direct) {
        // window = channels the grid works on at once (doubled: producers run a tile or two ahead of their loads);
        // on top of that the ring holds ~16 MiB of look-ahead, so a slab is complete long before its first tile is
        // drawn and stays L2-resident until its last tile is done
        const unsigned long long slab = static_cast<unsigned long long>(ntime) * ring_row_bytes(p);
        // (stripe kernel: a pair holds one of the channel's nblk stripes, so more channels are in flight at once)
        const int per_chan = p->stripe ? nblk : p->tiles_per_chan;
        const int window = (p->num_sms / 2 + per_chan - 1) / per_chan;
            long long ahead = static_cast<long long>(((p->stripe ? static_cast<unsigned long long>(BFX_ST_AHEAD_MB) : 16ull) << 20) / slab);
        if (ahead < 2) ahead = 2;
        long long ring = 2 * window + 2 + ahead;
        if (ring > nchan) ring = nchan;
        p->ring_w = static_cast<int>(ring);
        e = cudaMalloc(reinterpret_cast<void**>(&p->d_z), static_cast<size_t>(ring) * slab);
        if (e == cudaSuccess) e = cudaMalloc(reinterpret_cast<void**>(&p->d_flags), 2ull * nchan * sizeof(unsigned long long));
        if (e == cudaSuccess) e = cudaMemset(p->d_flags, 0, 2ull * nchan * sizeof(unsigned long long));
    }
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_few_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::FwCfg<true>::kSmemBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_few_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::FwCfg<false>::kSmemBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_pair4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::P4_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_pair_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::PR_SMEM_BYTES);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<true, false>::kSmemBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<false, true>::kSmemBytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::xcorr_stripe_kernel<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::StCfg<false, false>::kSmemBytes);
    if (e != cudaSuccess) {
        const int st = cuda_fail(nullptr, e);
        if (p->d_sched) cudaFree(p->d_sched);
        if (p->d_z) cudaFree(p->d_z);
        if (p->d_flags) cudaFree(p->d_flags);
        delete p;
        return st;
    }
    *plan = p;
    return BF_XCORR_OK;
}

int bfXcorrExecute(bfXcorr plan, const void* in, void* out, int accumulate, void* stream)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!in || !out) return BF_XCORR_INVALID_POINTER;
    if ((reinterpret_cast<uintptr_t>(in) & 15u) || (reinterpret_cast<uintptr_t>(out) & 15u)) return BF_XCORR_INVALID_POINTER;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != plan->device) return BF_XCORR_INVALID_ARGUMENT;   // the plan's scratch lives on another device
    plan->last_launch_count = 0;
    if (plan->algo == BF_XCORR_ALGO_SIMT) return launch_simt(plan, in, out, accumulate, s);
    if (plan->algo == BF_XCORR_ALGO_TCGEN05_GAUSS3) return launch_gauss4(plan, in, out, accumulate, s);
    if (plan->d_z) return launch_tcgen05<false>(plan, in, out, accumulate, s);  // S1 fused: dtype handled by the relayout warps
    return plan->dtype == BF_XCORR_CI4 ? launch_tcgen05<true>(plan, in, out, accumulate, s)
                                       : launch_tcgen05<false>(plan, in, out, accumulate, s);
}

int bfXcorrExecuteHost(bfXcorr plan, const void* in_host, void* out_dev, void* out_host, int accumulate, void* stream)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!in_host || !out_dev) return BF_XCORR_INVALID_POINTER;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    cudaError_t e = cudaSuccess;
    if (!plan->host_ready) {
        // first call (or a retry after a failed set-up): everything or nothing, so that a failure can be retried
        e = cudaStreamCreateWithFlags(&plan->s_h2d, cudaStreamNonBlocking);
        if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&plan->s_d2h, cudaStreamNonBlocking);
        for (int b = 0; b < 2 && e == cudaSuccess; ++b) {
            e = cudaMalloc(&plan->d_stage_in[b], input_bytes(plan));
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&plan->ev_h2d[b], cudaEventDisableTiming);
            if (e == cudaSuccess) e = cudaEventCreateWithFlags(&plan->ev_comp[b], cudaEventDisableTiming);
        }
        if (e == cudaSuccess) e = cudaEventCreateWithFlags(&plan->ev_d2h, cudaEventDisableTiming);
        if (e != cudaSuccess) {
            release_host_state(plan);
            return cuda_fail(plan, e);
        }
        plan->host_ready = true;
        plan->host_calls = 0;
    }
    const int b = static_cast<int>(plan->host_calls & 1);
    // span -> staging[b] on the copy stream, once the contraction that last read staging[b] (two calls ago) is done
    if (plan->host_calls >= 2) e = cudaStreamWaitEvent(plan->s_h2d, plan->ev_comp[b], 0);
    if (e == cudaSuccess)
        e = cudaMemcpyAsync(plan->d_stage_in[b], in_host, input_bytes(plan), cudaMemcpyHostToDevice, plan->s_h2d);
    if (e == cudaSuccess) e = cudaEventRecord(plan->ev_h2d[b], plan->s_h2d);
    if (e == cudaSuccess) e = cudaStreamWaitEvent(s, plan->ev_h2d[b], 0);
    if (e != cudaSuccess) return cuda_fail(plan, e);
    ++plan->host_calls;
    const int st = bfXcorrExecute(plan, plan->d_stage_in[b], out_dev, accumulate, stream);
    if (st != BF_XCORR_OK) return st;
    e = cudaEventRecord(plan->ev_comp[b], s);
    if (e == cudaSuccess && out_host) {
        // visibilities -> host on the other copy stream; `stream` waits for it, so that synchronising `stream`
        // covers the copy and no later launch touches out_dev while it is being read -- but the NEXT call's
        // host->device copy runs on its own stream and overlaps this one (PCIe is full duplex)
        e = cudaStreamWaitEvent(plan->s_d2h, plan->ev_comp[b], 0);
        if (e == cudaSuccess) e = cudaMemcpyAsync(out_host, out_dev, output_bytes(plan), cudaMemcpyDeviceToHost, plan->s_d2h);
        if (e == cudaSuccess) e = cudaEventRecord(plan->ev_d2h, plan->s_d2h);
        if (e == cudaSuccess) e = cudaStreamWaitEvent(s, plan->ev_d2h, 0);
    }
    if (e != cudaSuccess) return cuda_fail(plan, e);
    return BF_XCORR_OK;
}

int bfXcorrDump(bfXcorr plan, void* acc, void* out, float scale, int zero_acc, void* stream)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!acc || !out) return BF_XCORR_INVALID_POINTER;
    if ((reinterpret_cast<uintptr_t>(acc) & 15u) || (reinterpret_cast<uintptr_t>(out) & 15u)) return BF_XCORR_INVALID_POINTER;
    const long long ncomp = static_cast<long long>(output_bytes(plan) / 4);
    long long nblk = (ncomp / 4 + bfx::DUMP_THREADS - 1) / bfx::DUMP_THREADS;
    const long long cap = 8ll * plan->num_sms;
    if (nblk > cap) nblk = cap;
    if (nblk < 1) nblk = 1;
    plan->last_launch_count = 0;
    bfx::xcorr_dump_kernel<<<dim3(static_cast<unsigned>(nblk)), bfx::DUMP_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<int32_t*>(acc), static_cast<float*>(out), ncomp, scale, zero_acc ? 1 : 0);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(plan, e);
    plan->last_launch_count = 1;
    return BF_XCORR_OK;
}

int bfXcorrDumpMatrix(bfXcorr plan, void* acc, void* out, float scale, int zero_acc, void* stream)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!acc || !out) return BF_XCORR_INVALID_POINTER;
    if ((reinterpret_cast<uintptr_t>(acc) & 15u) || (reinterpret_cast<uintptr_t>(out) & 7u)) return BF_XCORR_INVALID_POINTER;
    const int nb = (plan->ninputs + bfx::DM_TILE - 1) / bfx::DM_TILE;
    const long long tiles = static_cast<long long>(nb) * (nb + 1) / 2;
    long long ychan = plan->nchan;
    const long long cap = (64ll * plan->num_sms + tiles - 1) / tiles;   // enough CTAs to fill the machine, channels strided beyond that
    if (ychan > cap) ychan = cap;
    if (ychan > 65535) ychan = 65535;
    plan->last_launch_count = 0;
    bfx::xcorr_dump_matrix_kernel<<<dim3(static_cast<unsigned>(tiles), static_cast<unsigned>(ychan)), 256, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<int32_t*>(acc), static_cast<float2*>(out), plan->ninputs, plan->nchan, scale, zero_acc ? 1 : 0);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(plan, e);
    plan->last_launch_count = 1;
    return BF_XCORR_OK;
}

int bfXcorrMemoryProbe(bfXcorr plan, const void* in, void* out, int accumulate, void* stream)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!in || !out) return BF_XCORR_INVALID_POINTER;
    if ((reinterpret_cast<uintptr_t>(in) & 15u) || (reinterpret_cast<uintptr_t>(out) & 15u)) return BF_XCORR_INVALID_POINTER;
    const long long nin = static_cast<long long>(input_bytes(plan) / 16), nout = static_cast<long long>(output_bytes(plan) / 16);
    const int grid = 4 * plan->num_sms;
    plan->last_launch_count = 0;
    bfx::mem_probe_kernel<<<grid, bfx::MP_THREADS, 0, static_cast<cudaStream_t>(stream)>>>(
        static_cast<const uint4*>(in), nin, static_cast<uint4*>(out), nout, accumulate ? 1 : 0,
        reinterpret_cast<unsigned int*>(plan->d_sched + 3));
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(plan, e);
    plan->last_launch_count = 1;
    return BF_XCORR_OK;
}

int bfXcorrDestroy(bfXcorr plan)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (plan->d_sched) cudaFree(plan->d_sched);
    release_host_state(plan);
    if (plan->d_z) cudaFree(plan->d_z);
    if (plan->d_flags) cudaFree(plan->d_flags);
    plan->magic = 0;
    delete plan;
    return BF_XCORR_OK;
}

int bfXcorrGetInputBytes(bfXcorr plan, unsigned long long* nbytes)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!nbytes) return BF_XCORR_INVALID_POINTER;
    *nbytes = input_bytes(plan);
    return BF_XCORR_OK;
}

int bfXcorrGetOutputBytes(bfXcorr plan, unsigned long long* nbytes)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!nbytes) return BF_XCORR_INVALID_POINTER;
    *nbytes = output_bytes(plan);
    return BF_XCORR_OK;
}

int bfXcorrGetMaxSafeNtime(bfXcorr plan, unsigned long long* nt)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!nt) return BF_XCORR_INVALID_POINTER;
    // |Re V| <= samples * 2 m^2 with m = 128 (ci8) or 8 (ci4); must stay <= 2^31 - 1
    const unsigned long long m = plan->dtype == BF_XCORR_CI4 ? 8ull : 128ull;
    *nt = 2147483647ull / (2ull * m * m);
    return BF_XCORR_OK;
}

int bfXcorrSetAlgo(bfXcorr plan, int algo)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (algo != BF_XCORR_ALGO_TCGEN05 && algo != BF_XCORR_ALGO_SIMT && algo != BF_XCORR_ALGO_TCGEN05_GAUSS3) return BF_XCORR_INVALID_ARGUMENT;
    if (algo == BF_XCORR_ALGO_TCGEN05_GAUSS3) {
        // the sums re + im fit int8 for 4-bit samples only
        if (plan->dtype != BF_XCORR_CI4) return BF_XCORR_INVALID_ARGUMENT;
        const int nblk = (plan->ninputs + bfx::PR_BLK - 1) / bfx::PR_BLK;
        if (static_cast<unsigned long long>(nblk) * (nblk + 1) / 2 * plan->nchan >= (1ull << 32)) return BF_XCORR_UNSUPPORTED_SHAPE;
        const cudaError_t e = cudaFuncSetAttribute(bfx::xcorr_gauss4_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::G4_SMEM_BYTES);
        if (e != cudaSuccess) return cuda_fail(plan, e);
    }
    plan->algo = algo;
    return BF_XCORR_OK;
}

const char* bfXcorrGetKernelName(bfXcorr plan, int accumulate)
{
    if (!valid(plan)) return "";
    if (plan->algo == BF_XCORR_ALGO_SIMT) return "xcorr_simt_kernel";
    if (plan->algo == BF_XCORR_ALGO_TCGEN05_GAUSS3) return "xcorr_gauss4_kernel";
    if (!plan->pair) return plan->dtype == BF_XCORR_CI4 ? "xcorr_few_kernel<ci4>" : "xcorr_few_kernel<ci8>";
    if (plan->dtype == BF_XCORR_CI4) return plan->d_z ? "xcorr_pair4_kernel (S1 ring)" : "xcorr_pair4_kernel (in place)";
    if (plan->stripe) {
        if (plan->d_z) return "xcorr_stripe_kernel<ring, staged epilogue>";
        return accumulate ? "xcorr_stripe_kernel<in place, staged L2-reduce epilogue>" : "xcorr_stripe_kernel<in place, register-direct epilogue>";
    }
    return plan->d_z ? "xcorr_pair_kernel (S1 ring)" : "xcorr_pair_kernel (in place)";
}

int bfXcorrGetLaunchCount(bfXcorr plan, int* nlaunch)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!nlaunch) return BF_XCORR_INVALID_POINTER;
    *nlaunch = plan->last_launch_count;
    return BF_XCORR_OK;
}

int bfXcorrGetLastCudaError(bfXcorr plan, int* cuda_error)
{
    if (!valid(plan)) return BF_XCORR_INVALID_HANDLE;
    if (!cuda_error) return BF_XCORR_INVALID_POINTER;
    *cuda_error = plan->last_cuda_error;
    return BF_XCORR_OK;
}

int bfXcorrExecuteNoAlloc(const void* in, void* out, int ninputs, int nchan, int ntime, int dtype, int accumulate, void* stream)
{
    // arguments: bfXcorrCreate's and bfXcorrExecute's checks, in their order
    if (ninputs <= 0 || nchan <= 0 || ntime <= 0 || ntime > 65535) return BF_XCORR_INVALID_ARGUMENT;
    if (dtype != BF_XCORR_CI4 && dtype != BF_XCORR_CI8) return BF_XCORR_INVALID_DTYPE;
    if ((static_cast<unsigned long long>(ninputs) * bytes_per_sample(dtype)) % 16ull != 0) return BF_XCORR_UNSUPPORTED_SHAPE;
    if (ninputs > 32768) return BF_XCORR_UNSUPPORTED_SHAPE;
    if (!in || !out) return BF_XCORR_INVALID_POINTER;
    if ((reinterpret_cast<uintptr_t>(in) & 15u) || (reinterpret_cast<uintptr_t>(out) & 15u)) return BF_XCORR_INVALID_POINTER;
    int ndev = 0, dev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev <= 0 || cudaGetDevice(&dev) != cudaSuccess) {
        cudaGetLastError();
        return BF_XCORR_UNSUPPORTED_DEVICE;
    }
    NaDevice nd;
    const int st = na_device_state(dev, &nd);
    if (st != BF_XCORR_OK) return st;

    // A plan on the stack, filled as bfXcorrCreate fills one (same kernel choice, same tile counts), whose scratch
    // pointers lead into the static array; it lives for this call only.
    bfXcorr_impl plan;
    std::memset(&plan, 0, sizeof(plan));
    plan.magic = kMagic;
    plan.ninputs = ninputs;
    plan.nchan = nchan;
    plan.ntime = ntime;
    plan.dtype = dtype;
    plan.algo = BF_XCORR_ALGO_TCGEN05;
    plan.device = dev;
    plan.num_sms = nd.num_sms;
    plan.encode = g_na_encode;
    const bool pair = ninputs > 64;
    const int nblk = (ninputs + bfx::PR_BLK - 1) / bfx::PR_BLK;
    plan.pair = pair;
    plan.stripe = BFX_STRIPE && pair && dtype == BF_XCORR_CI8 && ntime <= bfx::ST_MAXKB * bfx::TC_KT;
    plan.tiles_per_chan = pair ? nblk * (nblk + 1) / 2 : 1;
    if (pair && static_cast<unsigned long long>(plan.tiles_per_chan) * nchan >= (1ull << 32)) return BF_XCORR_UNSUPPORTED_SHAPE;
    plan.d_sched = reinterpret_cast<unsigned long long*>(nd.scratch);
    size_t clear_bytes = 4 * sizeof(unsigned long long);   // the scheduler words
    const bool near = static_cast<unsigned long long>(nchan) * ninputs * bytes_per_sample(dtype) <= (static_cast<unsigned long long>(BFX_DIRECT_STRIDE_KB) << 10);
    const bool direct = pair && (plan.stripe || dtype == BF_XCORR_CI4) &&
                        (nblk <= BFX_DIRECT_MAX_BLK || near || (dtype == BF_XCORR_CI4 && !BFX_P4_RING));
    if (pair && !direct) {
        // the S1 ring: bfXcorrCreate's sizing (channels in flight, doubled, + 2 + look-ahead), the look-ahead cut down
        // to what the fixed buffer holds but never below the 2 slabs bfXcorrCreate itself would accept
        if (nchan > BF_XCORR_NOALLOC_MAX_RING_CHANNELS) return BF_XCORR_SCRATCH_LIMIT;
        const unsigned long long slab = static_cast<unsigned long long>(ntime) * ring_row_bytes(&plan);
        const int per_chan = plan.stripe ? nblk : plan.tiles_per_chan;
        const int window = (plan.num_sms / 2 + per_chan - 1) / per_chan;
        long long ahead = static_cast<long long>(((plan.stripe ? static_cast<unsigned long long>(BFX_ST_AHEAD_MB) : 16ull) << 20) / slab);
        if (ahead < 2) ahead = 2;
        long long ring = 2 * window + 2 + ahead;
        long long ring_min = 2 * window + 2 + 2;
        if (ring > nchan) ring = nchan;
        if (ring_min > nchan) ring_min = nchan;
        const long long fits = static_cast<long long>(BF_XCORR_NOALLOC_RING_BYTES / slab);
        if (fits < ring_min) return BF_XCORR_SCRATCH_LIMIT;
        if (ring > fits) ring = fits;
        plan.ring_w = static_cast<int>(ring);
        plan.d_z = nd.scratch + kNaRingOff;
        plan.d_flags = reinterpret_cast<unsigned long long*>(nd.scratch + kNaFlagsOff);
        clear_bytes = kNaFlagsOff + 2ull * nchan * sizeof(unsigned long long);   // ... and ready[] / done[], which count from zero
    }
    // the array keeps what the last call (of any shape) left in it
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    const cudaError_t e = cudaMemsetAsync(nd.scratch, 0, clear_bytes, s);
    if (e != cudaSuccess) return cuda_fail(nullptr, e);
    if (plan.d_z) return launch_tcgen05<false>(&plan, in, out, accumulate, s);
    return dtype == BF_XCORR_CI4 ? launch_tcgen05<true>(&plan, in, out, accumulate, s)
                                 : launch_tcgen05<false>(&plan, in, out, accumulate, s);
}

const char* bfXcorrGetStatusString(int status)
{
    switch (status) {
        case BF_XCORR_OK: return "BF_XCORR_OK";
        case BF_XCORR_INVALID_POINTER: return "BF_XCORR_INVALID_POINTER";
        case BF_XCORR_INVALID_HANDLE: return "BF_XCORR_INVALID_HANDLE";
        case BF_XCORR_INVALID_ARGUMENT: return "BF_XCORR_INVALID_ARGUMENT";
        case BF_XCORR_INVALID_DTYPE: return "BF_XCORR_INVALID_DTYPE";
        case BF_XCORR_UNSUPPORTED_SHAPE: return "BF_XCORR_UNSUPPORTED_SHAPE";
        case BF_XCORR_UNSUPPORTED_DEVICE: return "BF_XCORR_UNSUPPORTED_DEVICE";
        case BF_XCORR_MEM_ALLOC_FAILED: return "BF_XCORR_MEM_ALLOC_FAILED";
        case BF_XCORR_DEVICE_ERROR: return "BF_XCORR_DEVICE_ERROR";
        case BF_XCORR_SCRATCH_LIMIT: return "BF_XCORR_SCRATCH_LIMIT";
        default: return "BF_XCORR_UNKNOWN_STATUS";
    }
}

}  // extern "C"
