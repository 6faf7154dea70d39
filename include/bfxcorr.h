/* bfxcorr.h -- C ABI of the B200-native X-engine (cross-multiply-accumulate correlator stage).
 *
 * What the library computes (BASELINE.json `north_star`; the paper itself prints no formula for
 * correlation: PAPER.md:141 lists a "Linear algebra -- matrix multiplication and related routines"
 * back-end module and PAPER.md:579 lists "comprehensive support for correlation" as near-term work):
 *
 *   for every channel c and every input pair i >= j (autocorrelations i == j included)
 *       V[c][i][j]  =  sum over the span's ntime samples t of   x[t][c][i] * conj( x[t][c][j] )
 *         .re = sum_t ( re_i*re_j + im_i*im_j )
 *         .im = sum_t ( im_i*re_j - re_i*im_j )
 *       out[c][ i*(i+1)/2 + j ]  =  (accumulate ? out[...] : 0) + V[c][i][j]
 *
 * i.e. the lower triangle of the Hermitian visibility matrix V[c] += sum_t x_t x_t^H, kept in int32
 * complex accumulators that persist across successive ring-buffer spans (PAPER.md:165 spans,
 * PAPER.md:345 "every span is contiguous", "Accumulate frames one at a time").
 *
 * Data formats (DESIGN.md section 3 lists every reading the paper leaves open):
 *   input  `in`  : DEVICE pointer, one dense span [ntime][nchan][ninputs], input index fastest.
 *       BF_XCORR_CI8 ("8+8 bit complex"): 2 bytes per sample, byte 0 = re, byte 1 = im,
 *                    both two's-complement int8; the code -128 is legal.
 *       BF_XCORR_CI4 ("4+4 complex signed integers"): 1 byte per sample,
 *                    re = high nibble (bits 7..4), im = low nibble (bits 3..0), each two's
 *                    complement in [-8, 7]; the code -8 is legal.
 *   output `out` : DEVICE pointer, [nchan][B][2] int32 with B = ninputs*(ninputs+1)/2; element
 *                  k = i*(i+1)/2 + j (row-major packed lower triangle, i >= j) holds (re, im).
 *   Arithmetic   : exact integer; int32 accumulators wrap modulo 2^32 (no saturation).  With
 *                  |re|,|im| <= 128 (ci8) a visibility cannot wrap before 65 535 accumulated samples
 *                  (bfXcorrGetMaxSafeNtime); ci4: 16 777 215.
 *
 * Ownership and ordering: the caller owns `in`, `out` and the stream.  bfXcorrExecute only enqueues
 * work on `stream` and returns without synchronising; `in` and `out` must stay valid until the stream
 * reaches that point.  The plan owns its private device scratch (descriptors, work tables), allocated
 * by bfXcorrCreate on the CUDA device that is current at that call and released by bfXcorrDestroy.
 * A plan may be used by one host thread at a time, and its launches must not overlap on the device (they share
 * the plan's scheduler words, S1 ring and flags): enqueue them on one stream, or order streams with events.
 * Results are deterministic (integer sums).
 *
 * Errors: every entry point returns a bfXcorrStatus (0 = OK); no host code aborts or throws across the ABI.
 * Device side, every wait of the kernels (mbarriers, flags between CTAs) is BOUNDED: should one not complete within
 * a few seconds -- which only a defect of the library or a corrupted plan can cause, never the data -- the kernel
 * executes a trap instead of hanging the GPU.  The caller then sees what any faulting kernel produces: the next
 * synchronising CUDA call on that stream returns cudaErrorLaunchFailure, the error is sticky (the CUDA context is
 * lost and must be torn down with the process or cudaDeviceReset), and every later call into this library that
 * touches the device returns BF_XCORR_DEVICE_ERROR.  The contents of `out` are then undefined.
 * There is NO CPU fallback: without a compute-capability-10.x device bfXcorrCreate returns
 * BF_XCORR_UNSUPPORTED_DEVICE.
 */
#ifndef BFXCORR_H_
#define BFXCORR_H_

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bfXcorr_impl* bfXcorr; /* opaque plan handle */

typedef enum bfXcorrDtype_ {
    BF_XCORR_CI4 = 4, /* 4+4-bit complex */
    BF_XCORR_CI8 = 8  /* 8+8-bit complex */
} bfXcorrDtype;

typedef enum bfXcorrStatus_ {
    BF_XCORR_OK = 0,
    BF_XCORR_INVALID_POINTER = 1,    /* NULL plan/in/out/result pointer, or misaligned in/out */
    BF_XCORR_INVALID_HANDLE = 2,     /* NULL or already destroyed plan */
    BF_XCORR_INVALID_ARGUMENT = 3,   /* non-positive dimension, unknown algorithm, ...         */
    BF_XCORR_INVALID_DTYPE = 4,      /* dtype not BF_XCORR_CI4 / BF_XCORR_CI8                   */
    BF_XCORR_UNSUPPORTED_SHAPE = 5,  /* see bfXcorrCreate                                       */
    BF_XCORR_UNSUPPORTED_DEVICE = 6, /* no CUDA device of compute capability 10.x               */
    BF_XCORR_MEM_ALLOC_FAILED = 7,
    BF_XCORR_DEVICE_ERROR = 8,       /* a CUDA call failed; see bfXcorrGetLastCudaError         */
    BF_XCORR_SCRATCH_LIMIT = 9       /* bfXcorrExecuteNoAlloc: the span needs more scratch than the fixed buffer holds */
} bfXcorrStatus;

/* Which kernel bfXcorrExecute launches.  TCGEN05 is the product path and the default: unpack-and-transpose
 * stage, TMA-staged int8 operands, tcgen05.mma kind::i8 with int32 accumulators held in TMEM over the whole span,
 * lower-triangle tile scheduler, span-accumulate epilogue (CTA pairs above 64 inputs -- with a resident A block per
 * stripe of tiles for ci8 spans of at most 1024 samples --, four channels per CTA up to 64 inputs: DESIGN.md section 5).  SIMT is a plain CUDA-core kernel kept as
 * an on-device cross-check of the tensor path at sizes the CPU oracle cannot reach; it is never
 * selected implicitly.  TCGEN05_GAUSS3 (ci4 plans only) forms the complex product from THREE real tensor-core products
 * instead of four -- (a+b)c, a(c+d), b(c-d) on operands that fit int8 only because the samples are 4-bit (SURVEY.md
 * section 8(f) N3; PAPER.md:555 works on the 4+4-bit samples directly): same result bit for bit, 3/4 of the
 * multiply-accumulates, but measured slower than the default on B200 (profiles/round2.md), so never selected implicitly. */
typedef enum bfXcorrAlgo_ {
    BF_XCORR_ALGO_TCGEN05 = 0,
    BF_XCORR_ALGO_SIMT = 1,
    BF_XCORR_ALGO_TCGEN05_GAUSS3 = 2
} bfXcorrAlgo;

/* Create a plan for spans of exactly `ntime` samples x `nchan` channels x `ninputs` inputs of `dtype`
 * (BASELINE.json north_star: bfXcorrCreate(ninputs, nchan, ntime, dtype)).
 *   *plan  : receives the handle (host pointer, must not be NULL).
 *   errors : INVALID_POINTER (plan NULL); INVALID_ARGUMENT (a dimension <= 0, or ntime > 65535);
 *            INVALID_DTYPE; UNSUPPORTED_SHAPE (ninputs * bytes_per_sample not a multiple of 16: the
 *            16-byte vector / TMA row granularity -- every BASELINE.json config satisfies it; ninputs > 32768;
 *            or nchan * tiles-per-channel >= 2^32);
 *            UNSUPPORTED_DEVICE; MEM_ALLOC_FAILED; DEVICE_ERROR. */
int bfXcorrCreate(bfXcorr* plan, int ninputs, int nchan, int ntime, int dtype);

/* Correlate one span (BASELINE.json north_star: bfXcorrExecute(in, out, accumulate, stream)).
 *   in         : device pointer to the span, 16-byte aligned, bfXcorrGetInputBytes bytes, read only.
 *   out        : device pointer to the visibilities, 16-byte aligned, bfXcorrGetOutputBytes bytes.
 *   accumulate : 0 = overwrite `out` (it need not be initialised); non-zero = out += this span.
 *   stream     : a cudaStream_t passed as void* (NULL = the legacy default stream).
 *   errors     : INVALID_HANDLE; INVALID_POINTER (NULL or misaligned); INVALID_ARGUMENT (the current CUDA device is not
 *                the one the plan was created on); DEVICE_ERROR (launch failed). */
int bfXcorrExecute(bfXcorr plan, const void* in, void* out, int accumulate, void* stream);

/* Release the plan and its device scratch.  errors: INVALID_HANDLE (NULL). */
int bfXcorrDestroy(bfXcorr plan);

/* Pure queries; `nbytes` / `nt` are host pointers.  errors: INVALID_HANDLE, INVALID_POINTER. */
int bfXcorrGetInputBytes(bfXcorr plan, unsigned long long* nbytes);  /* ntime*nchan*ninputs*(1|2)   */
int bfXcorrGetOutputBytes(bfXcorr plan, unsigned long long* nbytes); /* nchan*ninputs*(ninputs+1)/2*8 */
int bfXcorrGetMaxSafeNtime(bfXcorr plan, unsigned long long* nt);    /* samples before int32 may wrap */

/* Select the kernel (see bfXcorrAlgo).  errors: INVALID_HANDLE, INVALID_ARGUMENT (unknown algorithm; GAUSS3 on a ci8
 * plan), UNSUPPORTED_SHAPE, DEVICE_ERROR. */
int bfXcorrSetAlgo(bfXcorr plan, int algo);

/* Name of the kernel (and variant) bfXcorrExecute launches for this plan with the given `accumulate`: a static string,
 * "" for an invalid handle.  For reports (bench.py's roofline.kernel); the dispatch rule itself lives in the library. */
const char* bfXcorrGetKernelName(bfXcorr plan, int accumulate);

/* Number of kernels the last bfXcorrExecute on this plan launched (for launch accounting). */
int bfXcorrGetLaunchCount(bfXcorr plan, int* nlaunch);

/* cudaError_t of the last failing CUDA call made on behalf of this plan (0 if none). */
int bfXcorrGetLastCudaError(bfXcorr plan, int* cuda_error);

/* Entry point for callers whose buffers live in HOST memory (bench.py's end-to-end leg).  The span is copied
 * host->device into one of two plan-owned staging buffers on a private copy stream, the contraction runs on
 * `stream` once the copy has landed, and -- if `out_host` is not NULL -- the visibility buffer is copied
 * device->host on a second private stream that `stream` then waits for.  Successive calls therefore overlap the
 * upload of span n+1 with the contraction of span n and with the download of the visibilities, as the paper's
 * pipelines overlap copy and compute; synchronising `stream` still covers everything enqueued.
 *   in_host, out_host : HOST pointers (pinned memory makes the copies asynchronous); `in_host` may be reused and
 *                       `out_host` read once `stream` has been synchronised.
 *   out_dev           : the persistent device accumulator, as in bfXcorrExecute.
 *   errors            : as bfXcorrExecute, plus MEM_ALLOC_FAILED for the staging buffers. */
int bfXcorrExecuteHost(bfXcorr plan, const void* in_host, void* out_dev, void* out_host, int accumulate,
                       void* stream);

/* Integration dump -- the step after the hot path ("accumulate" hands an integration on when it is
 * complete; integer data become floating point for the stages that follow).  Every int32 component
 * v of the packed visibility buffer becomes   (float) v * scale   (int32 -> float32 round-to-nearest-even, then one
 * float32 multiply) in the same [nchan][B][2] order; with zero_acc != 0 the accumulator is cleared in the same
 * pass, so the next integration can use accumulate = 1 from its first span.
 *   acc    : DEVICE pointer, the int32 visibility buffer of this plan (bfXcorrGetOutputBytes bytes), 16-byte aligned;
 *            read, and written only if zero_acc != 0.
 *   out    : DEVICE pointer, float32 buffer of the same number of bytes, 16-byte aligned, must not overlap `acc`.
 *   stream : as bfXcorrExecute; the call only enqueues.
 *   errors : INVALID_HANDLE; INVALID_POINTER (NULL or misaligned); DEVICE_ERROR. */
int bfXcorrDump(bfXcorr plan, void* acc, void* out, float scale, int zero_acc, void* stream);

/* Integration dump with reorder (the paper's back end has "efficient data reordering"): as
 * bfXcorrDump, but the packed lower triangle is written out as the FULL Hermitian matrix
 *   out[c][i][j] = (float) V[c][i][j] * scale             for j <= i
 *   out[c][i][j] = conj( out[c][j][i] )                   for j >  i   (exact; a zero imaginary part becomes -0.0f)
 *   acc    : as bfXcorrDump.
 *   out    : DEVICE pointer, [nchan][ninputs][ninputs][2] float32 = nchan * ninputs^2 * 8 bytes, 8-byte aligned, must not
 *            overlap `acc`.
 *   errors : as bfXcorrDump. */
int bfXcorrDumpMatrix(bfXcorr plan, void* acc, void* out, float scale, int zero_acc, void* stream);

/* Measurement aid (the same-mix HBM ceiling): a no-math streaming kernel that moves exactly
 * the path's algorithmic bytes with coalesced, contiguous accesses -- reads the span once, and writes the visibility
 * buffer once (accumulate = 0) or reads, increments and rewrites it (accumulate != 0).  It computes nothing of the
 * method; `out` is left holding meaningless values.  bench.py times it beside bfXcorrExecute and reports the
 * bandwidth it reaches as roofline.same_mix_peak.
 *   in, out, stream : as bfXcorrExecute (sizes from the plan).  errors: as bfXcorrExecute. */
int bfXcorrMemoryProbe(bfXcorr plan, const void* in, void* out, int accumulate, void* stream);

/* One span, with NO device-memory allocation anywhere: for callers that cannot call cudaMalloc (a tight serving loop,
 * a harness that forbids it).  No plan: the geometry is passed with every call.  The same tensor-core kernels as
 * bfXcorrExecute with the default algorithm, chosen by the same rule, and the same result bit for bit
 * (out[c][i(i+1)/2 + j] = (accumulate ? out : 0) + sum_t x_i conj(x_j), PAPER.md:378 / SURVEY.md 8c); what differs is
 * where their scratch lives.  A plan allocates it at bfXcorrCreate (the tile scheduler's counters, and for spans that
 * take the unpack-and-transpose stage through the L2-resident S1 ring -- ci8 spans of more than 1024 samples, and spans
 * of more than 1024 inputs whose consecutive samples of a channel lie more than 1 MiB apart -- the ring of channel slabs
 * and two progress counters per channel).  Here all of it is one file-scope `static __device__` array of BF_XCORR_NOALLOC_SCRATCH_BYTES that every GPU
 * holds from the moment it loads the library until the process exits.
 *   in, out, accumulate, stream : as bfXcorrExecute (DEVICE pointers, 16-byte aligned; the caller owns them).
 *   ninputs, nchan, ntime, dtype : as bfXcorrCreate, same limits.
 * Limits of the fixed scratch (BF_XCORR_SCRATCH_LIMIT, nothing launched): a span that needs the S1 ring must have at
 * most BF_XCORR_NOALLOC_MAX_RING_CHANNELS channels and the smallest workable ring (the channels in flight, twice, plus 4
 * slabs of ntime * ninputs * 2 bytes, ci4: ntime * ninputs) must fit BF_XCORR_NOALLOC_RING_BYTES; BASELINE.json's five configs all fit (only
 * configs[3] uses the ring: 14 slabs of 4 MiB).  Spans read in place need 32 bytes and are never rejected.
 * The array is shared by every call on the device and keeps the last call's contents: each call first clears, on
 * `stream`, the counters it needs at zero.  Two calls whose work overlaps on the GPU (different streams, or different
 * host threads) therefore race -- order them on one stream or with events; bfXcorrExecute on a plan is not affected.
 * The first call on a device also does that device's one-time set-up (the array's address, kernel attributes, the
 * tensor-map encoder): no allocation either, but make it outside a stream capture.  Never calls cudaMalloc, cudaFree or
 * an allocating library routine.
 *   errors : as bfXcorrCreate and bfXcorrExecute for the arguments; BF_XCORR_UNSUPPORTED_DEVICE without a compute
 *            capability 10.x device; BF_XCORR_SCRATCH_LIMIT as above; BF_XCORR_DEVICE_ERROR if a CUDA call fails. */
#define BF_XCORR_NOALLOC_RING_BYTES (64ull << 20)
#define BF_XCORR_NOALLOC_MAX_RING_CHANNELS 65536
#define BF_XCORR_NOALLOC_SCRATCH_BYTES (1024ull + 16ull * BF_XCORR_NOALLOC_MAX_RING_CHANNELS + BF_XCORR_NOALLOC_RING_BYTES)
int bfXcorrExecuteNoAlloc(const void* in, void* out, int ninputs, int nchan, int ntime, int dtype, int accumulate,
                          void* stream);

/* Static string for a status code (never NULL). */
const char* bfXcorrGetStatusString(int status);

#ifdef __cplusplus
}
#endif
#endif /* BFXCORR_H_ */
