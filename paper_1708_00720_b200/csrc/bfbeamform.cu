// bfbeamform.cu -- host side of include/bfbeamform.h: plan construction, weight re-ordering, launch of the sm_100a
// beamformer kernel (beamform.cuh).  No CPU compute path exists here.
#include <cstdint>
#include <cstring>
#include <new>

#include <cuda.h>
#include <cuda_runtime.h>

#include "../../include/bfbeamform.h"
#include "beamform.cuh"

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// ci8: row pieces per span box (2: the 5-d span map of beamform.cuh, where the shape allows it; 1: always the 3-d map)
#ifndef BFX_BM_PW
#define BFX_BM_PW 2
#endif
// ... taken when at least this many such stages fit (100 beams on cfg3: two two-piece stages 74 %, five one-piece stages 67 % of the copy peak)
#ifndef BFX_BM_MINST
#define BFX_BM_MINST 2u
#endif
#ifndef BFX_BM_GROUP_MB
#define BFX_BM_GROUP_MB 8
#endif
#ifndef BFX_BM_PROMO
#define BFX_BM_PROMO CU_TENSOR_MAP_L2_PROMOTION_L2_256B
#endif

constexpr uint32_t kMagic = 0xBFBEA301u;

}  // namespace

struct bfBeamform_impl {
    uint32_t magic;
    int ninputs, nchan, ntime, nbeam, dtype;
    int device;     // the plan's scratch lives on this device
    int num_sms;
    int last_cuda_error;
    int have_weights;
    uint8_t* d_wp;  // re-ordered, offset weights W[nchan][nb2][kp] uint8 (beamform.cuh)
    int nb2, kp;
    CUtensorMap wmap;
    EncodeTiledFn encode;
    bfx::BmParams prm;
    unsigned smem_bytes;
};

namespace {

bool valid(bfBeamform p) { return p != nullptr && p->magic == kMagic; }

int cuda_fail(bfBeamform p, cudaError_t e)
{
    if (p) p->last_cuda_error = static_cast<int>(e);
    return e == cudaErrorMemoryAllocation ? BF_XCORR_MEM_ALLOC_FAILED : BF_XCORR_DEVICE_ERROR;
}

unsigned long long bps(int dtype) { return dtype == BF_XCORR_CI4 ? 1ull : 2ull; }

void release(bfBeamform p)
{
    if (p->d_wp) cudaFree(p->d_wp);
    p->magic = 0;
    delete p;
}

}  // namespace

extern "C" {

int bfBeamformCreate(bfBeamform* plan, int ninputs, int nchan, int ntime, int nbeam, int dtype)
{
    if (!plan) return BF_XCORR_INVALID_POINTER;
    *plan = nullptr;
    if (ninputs <= 0 || nchan <= 0 || ntime <= 0 || nbeam <= 0) return BF_XCORR_INVALID_ARGUMENT;
    if (dtype != BF_XCORR_CI4 && dtype != BF_XCORR_CI8) return BF_XCORR_INVALID_DTYPE;
    if ((static_cast<unsigned long long>(ninputs) * bps(dtype)) % 16ull != 0) return BF_XCORR_UNSUPPORTED_SHAPE;
    if (ninputs > 32768 || nbeam > 127) return BF_XCORR_UNSUPPORTED_SHAPE;   // 2 nbeam + 2 accumulator columns <= 256

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

    bfBeamform p = new (std::nothrow) bfBeamform_impl;
    if (!p) return BF_XCORR_MEM_ALLOC_FAILED;
    std::memset(p, 0, sizeof(*p));
    p->magic = kMagic;
    p->ninputs = ninputs;
    p->nchan = nchan;
    p->ntime = ntime;
    p->nbeam = nbeam;
    p->dtype = dtype;
    p->device = dev;
    p->num_sms = prop.multiProcessorCount;

    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qres;
    cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qres);
    if (e != cudaSuccess || qres != cudaDriverEntryPointSuccess || !fn) {
        delete p;
        return BF_XCORR_UNSUPPORTED_DEVICE;
    }

    const bool ci4 = dtype == BF_XCORR_CI4;
    const int row_in = static_cast<int>(ninputs * bps(dtype));
    const int ks_bytes = ci4 ? 256 : 128;  // int8 K bytes per 128 span bytes
    bfx::BmParams& q = p->prm;
    q.ninputs = ninputs;
    q.nchan = nchan;
    q.ntime = ntime;
    q.nbeam = nbeam;
    q.row_in = row_in;
    q.nb2 = (2 * nbeam + 2 + 15) / 16 * 16;   // two rows per beam + the two selector rows (beamform.cuh)
    q.nks = (row_in + 127) / 128;
    q.pw = 1;
    q.ntb = (ntime + bfx::BM_MT - 1) / bfx::BM_MT;
    q.nunits = static_cast<long long>(q.ntb) * nchan;
    p->nb2 = q.nb2;
    p->kp = q.nks * ks_bytes;
    unsigned stage_bytes = static_cast<unsigned>(ks_bytes / 128) * (bfx::BM_MT * 128u + static_cast<unsigned>(q.nb2) * 128u);
    // ci8 spans whose rows are whole multiples of BFX_BM_PW pieces and whose sample count is a multiple of 8 are read through
    // the 5-d map, BFX_BM_PW pieces per box and K stage -- if at least BFX_BM_MINST such stages fit
    if (!ci4 && BFX_BM_PW > 1 && row_in % (128 * BFX_BM_PW) == 0 && ntime % 8 == 0 &&
        BFX_BM_MINST * BFX_BM_PW * stage_bytes + 1536u + bfx::BM_STG_BYTES <= static_cast<unsigned>(bfx::BM_SMEM_MAX)) {
        q.pw = BFX_BM_PW;
        q.nks = row_in / (128 * BFX_BM_PW);
        stage_bytes *= BFX_BM_PW;
    }
    // ci4: raw ring of 16 KB tiles beside the operand stages (2 when the stages are at their largest, else 4)
    const unsigned raw_tile = bfx::BM_MT * 128u;
    const unsigned fixed = 1536u + bfx::BM_STG_BYTES;
    int raw = ci4 ? (2u * stage_bytes + 4u * raw_tile + fixed <= static_cast<unsigned>(bfx::BM_SMEM_MAX) ? 4 : 2) : 0;
    int stages = static_cast<int>((bfx::BM_SMEM_MAX - fixed - raw * raw_tile) / stage_bytes);
    if (stages > bfx::BM_MAX_STAGES) stages = bfx::BM_MAX_STAGES;
    // ci8: >= 2 for every nb2 <= 256.  ci4 with nb2 > 208 (more than 103 beams): the two widened K tiles of a stage take
    // 2 * (16 KiB + 128 nb2) bytes and only ONE stage fits beside the raw ring and the staging -- loads, widening and MMA
    // then run one after the other (exact, but about 2.5 x slower per byte: DESIGN.md section 11)
    q.stages = stages;
    q.raw_stages = raw;
    p->smem_bytes = static_cast<unsigned>(stages) * stage_bytes + raw * raw_tile + fixed;
    p->encode = reinterpret_cast<EncodeTiledFn>(fn);
    // a group's weights (group * nb2 * kp bytes, about 8 MB) stay in the L2 (evict-last loads) while its sample blocks go by
    long long group = (static_cast<long long>(BFX_BM_GROUP_MB) << 20) / (static_cast<long long>(q.nb2) * p->kp);
    if (group < 1) group = 1;
    if (group > nchan) group = nchan;
    q.group = static_cast<int>(group);

    const size_t wbytes = static_cast<size_t>(nchan) * q.nb2 * p->kp;
    e = cudaMalloc(reinterpret_cast<void**>(&p->d_wp), wbytes);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::beamform_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::BM_SMEM_MAX);
    if (e == cudaSuccess)
        e = cudaFuncSetAttribute(bfx::beamform_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, bfx::BM_SMEM_MAX);
    if (e != cudaSuccess) {
        const int st = cuda_fail(nullptr, e);
        release(p);
        return st;
    }
    // weight boxes: 128 bytes of K x nb2 rows of one channel, 128B-swizzled K-major
    const cuuint64_t dims[2] = {static_cast<cuuint64_t>(p->kp), static_cast<cuuint64_t>(nchan) * q.nb2};
    const cuuint64_t strides[1] = {static_cast<cuuint64_t>(p->kp)};
    const cuuint32_t box[2] = {128u, static_cast<cuuint32_t>(q.nb2)};
    const cuuint32_t estr[2] = {1u, 1u};
    const CUresult r = reinterpret_cast<EncodeTiledFn>(fn)(&p->wmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 2, p->d_wp, dims, strides, box, estr,
                                                           CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B,
                                                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        release(p);
        return BF_XCORR_DEVICE_ERROR;
    }
    *plan = p;
    return BF_XCORR_OK;
}

int bfBeamformSetWeights(bfBeamform p, const void* weights, void* stream)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!weights || (reinterpret_cast<uintptr_t>(weights) & 1u)) return BF_XCORR_INVALID_POINTER;
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    p->have_weights = 0;
    cudaError_t e = cudaSuccess;
    const long long total = static_cast<long long>(p->nchan) * p->nb2 * p->kp;
    long long blocks = (total + 255) / 256;
    if (blocks > 32ll * p->num_sms) blocks = 32ll * p->num_sms;
    if (p->dtype == BF_XCORR_CI4)
        bfx::beamform_weights_kernel<true><<<static_cast<unsigned>(blocks), 256, 0, s>>>(
            static_cast<const int8_t*>(weights), p->d_wp, p->ninputs, p->nchan, p->nbeam, p->nb2, p->kp);
    else
        bfx::beamform_weights_kernel<false><<<static_cast<unsigned>(blocks), 256, 0, s>>>(
            static_cast<const int8_t*>(weights), p->d_wp, p->ninputs, p->nchan, p->nbeam, p->nb2, p->kp);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e);
    e = cudaStreamSynchronize(s);   // the caller's weight buffer may be reused once this call has returned
    if (e != cudaSuccess) return cuda_fail(p, e);
    p->have_weights = 1;
    return BF_XCORR_OK;
}

int bfBeamformExecute(bfBeamform p, const void* in, void* out, void* stream)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!in || !out || (reinterpret_cast<uintptr_t>(in) & 15u)) return BF_XCORR_INVALID_POINTER;
    if (reinterpret_cast<uintptr_t>(out) & ((p->nbeam & 1) ? 7u : 15u)) return BF_XCORR_INVALID_POINTER;
    if (!p->have_weights) return BF_XCORR_INVALID_ARGUMENT;
    int cur = -1;
    if (cudaGetDevice(&cur) != cudaSuccess || cur != p->device) return BF_XCORR_INVALID_ARGUMENT;   // the plan belongs to another device
    bfx::BmParams q = p->prm;
    q.x = static_cast<const uint8_t*>(in);
    q.out = static_cast<int32_t*>(out);
    const unsigned grid = static_cast<unsigned>(q.nunits < p->num_sms ? q.nunits : p->num_sms);
    cudaStream_t s = static_cast<cudaStream_t>(stream);
    // span boxes: 128 bytes of a row x 1 channel x 128 samples; rows and samples beyond the span read as zeros
    const bool ci4 = p->dtype == BF_XCORR_CI4;
    CUtensorMap xmap;
    const cuuint64_t row = static_cast<cuuint64_t>(q.row_in), sample = row * p->nchan;
    const cuuint64_t dims[3] = {row, static_cast<cuuint64_t>(p->nchan), static_cast<cuuint64_t>(p->ntime)};
    const cuuint64_t strides[2] = {row, sample};
    const cuuint32_t box[3] = {128u, 1u, static_cast<cuuint32_t>(bfx::BM_MT)};
    // q.pw > 1: {128 B, sample % 8, row piece, channel, sample / 8}, box {128, 8, pw, 1, BM_MT / 8}
    const cuuint64_t dims5[5] = {128u, 8u, row / 128u, static_cast<cuuint64_t>(p->nchan), static_cast<cuuint64_t>(p->ntime / 8)};
    const cuuint64_t strides5[4] = {sample, 128u, row, 8u * sample};
    const cuuint32_t box5[5] = {128u, 8u, static_cast<cuuint32_t>(q.pw), 1u, static_cast<cuuint32_t>(bfx::BM_MT / 8)};
    const cuuint32_t estr[5] = {1u, 1u, 1u, 1u, 1u};
    const CUresult r = q.pw > 1 ? p->encode(&xmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 5, const_cast<void*>(in), dims5, strides5, box5, estr,
                                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, BFX_BM_PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE)
                                : p->encode(&xmap, CU_TENSOR_MAP_DATA_TYPE_UINT8, 3, const_cast<void*>(in), dims, strides, box, estr,
                                 CU_TENSOR_MAP_INTERLEAVE_NONE, ci4 ? CU_TENSOR_MAP_SWIZZLE_NONE : CU_TENSOR_MAP_SWIZZLE_128B,
                                 BFX_BM_PROMO, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        p->last_cuda_error = static_cast<int>(cudaErrorInvalidValue);
        return BF_XCORR_DEVICE_ERROR;
    }
    if (ci4)
        bfx::beamform_kernel<true><<<grid, bfx::BM_THREADS, p->smem_bytes, s>>>(xmap, p->wmap, q);
    else
        bfx::beamform_kernel<false><<<grid, bfx::BM_THREADS, p->smem_bytes, s>>>(xmap, p->wmap, q);
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(p, e);
    return BF_XCORR_OK;
}

int bfBeamformDestroy(bfBeamform p)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    release(p);
    return BF_XCORR_OK;
}

int bfBeamformGetInputBytes(bfBeamform p, unsigned long long* nbytes)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!nbytes) return BF_XCORR_INVALID_POINTER;
    *nbytes = static_cast<unsigned long long>(p->ntime) * p->nchan * p->ninputs * bps(p->dtype);
    return BF_XCORR_OK;
}

int bfBeamformGetWeightBytes(bfBeamform p, unsigned long long* nbytes)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!nbytes) return BF_XCORR_INVALID_POINTER;
    *nbytes = static_cast<unsigned long long>(p->nchan) * p->nbeam * p->ninputs * 2ull;
    return BF_XCORR_OK;
}

int bfBeamformGetOutputBytes(bfBeamform p, unsigned long long* nbytes)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!nbytes) return BF_XCORR_INVALID_POINTER;
    *nbytes = static_cast<unsigned long long>(p->ntime) * p->nchan * p->nbeam * 8ull;
    return BF_XCORR_OK;
}

int bfBeamformGetLastCudaError(bfBeamform p, int* cuda_error)
{
    if (!valid(p)) return BF_XCORR_INVALID_HANDLE;
    if (!cuda_error) return BF_XCORR_INVALID_POINTER;
    *cuda_error = p->last_cuda_error;
    return BF_XCORR_OK;
}

}  // extern "C"
