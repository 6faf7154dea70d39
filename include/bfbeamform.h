/* bfbeamform.h -- C ABI of the phase-and-sum beamformer that runs on the same spans as the X-engine
 * (SURVEY.md section 8(f) N1).  It is the GPU stage the paper's deployment actually runs on the "4+4 complex
 * signed integers" of the station; the paper prints no formula for it, so the
 * definition below is this build's reading.  Same library (libbfxcorr.so), same status
 * codes and dtype codes as include/bfxcorr.h.
 *
 * What it computes:
 *
 *   for every sample t, channel c and beam k
 *       b[t][c][k]  =  sum over the inputs i of   w[c][k][i] * x[t][c][i]         (complex product, no conjugate)
 *         .re = sum_i ( wr*xr - wi*xi )
 *         .im = sum_i ( wr*xi + wi*xr )
 *       out[t][c][k] = b                                                           (int32 re, int32 im)
 *
 * Data formats:
 *   span `in`     : DEVICE pointer, [ntime][nchan][ninputs] ci4 or ci8, exactly as in include/bfxcorr.h.
 *   weights       : DEVICE pointer, dense [nchan][nbeam][ninputs], input fastest, always 8+8 bit: byte 0 = re,
 *                   byte 1 = im, two's-complement int8.  Every code is legal for both parts, -128 included (the plan
 *                   holds the weights as unsigned bytes with an offset that the kernel takes out again, exactly).
 *   output `out`  : DEVICE pointer, [ntime][nchan][nbeam][2] int32.
 *   Arithmetic    : exact integer.  |b| components are below 2 * ninputs * 128 * 128 <= 2^30 for every legal plan,
 *                   so int32 never wraps.
 *
 * Ownership and ordering: as include/bfxcorr.h.  The plan keeps its own re-ordered copy of the weights
 * (bfBeamformSetWeights), so the caller's weight buffer may be reused once that call has returned.  Launches of one
 * plan must not overlap bfBeamformSetWeights of the same plan.
 *
 * Errors: every entry point returns a bfXcorrStatus.  There is NO CPU fallback.
 */
#ifndef BFBEAMFORM_H_
#define BFBEAMFORM_H_

#include "bfxcorr.h"

#ifdef __cplusplus
extern "C" {
#endif

typedef struct bfBeamform_impl* bfBeamform; /* opaque plan handle */

/* Create a plan for spans of `ntime` samples x `nchan` channels x `ninputs` inputs of `dtype` and `nbeam` beams.
 *   errors : INVALID_POINTER (plan NULL); INVALID_ARGUMENT (a dimension <= 0); INVALID_DTYPE;
 *            UNSUPPORTED_SHAPE (ninputs * bytes_per_sample not a multiple of 16; ninputs > 32768; nbeam > 127: two
 *            accumulator columns per beam plus two for the offset sums must fit one 256-column MMA);
 *            UNSUPPORTED_DEVICE; MEM_ALLOC_FAILED; DEVICE_ERROR. */
int bfBeamformCreate(bfBeamform* plan, int ninputs, int nchan, int ntime, int nbeam, int dtype);

/* Load a weight set.  The weights are re-ordered on the device into the plan's unsigned 8-bit operand layout (one row
 * (wr + 128, 127 - wi) and one (wi + 128, wr + 128) per beam, matching the order in which the kernel unpacks the
 * voltages).  The call synchronises `stream` before it returns.
 *   weights : device pointer, [nchan][nbeam][ninputs] ci8, 2-byte aligned.
 *   errors  : INVALID_HANDLE; INVALID_POINTER; DEVICE_ERROR. */
int bfBeamformSetWeights(bfBeamform plan, const void* weights, void* stream);

/* Beamform one span with the weights loaded last.
 *   in     : device pointer to the span, 16-byte aligned, read only.
 *   out    : device pointer, bfBeamformGetOutputBytes bytes, 8-byte aligned (16 if nbeam is even); overwritten.
 *   stream : a cudaStream_t passed as void*; the call only enqueues.
 *   errors : INVALID_HANDLE; INVALID_POINTER (NULL or misaligned); INVALID_ARGUMENT (no weights loaded, or the
 *            current CUDA device is not the one the plan was created on); DEVICE_ERROR. */
int bfBeamformExecute(bfBeamform plan, const void* in, void* out, void* stream);

/* Release the plan and its device scratch.  errors: INVALID_HANDLE. */
int bfBeamformDestroy(bfBeamform plan);

/* Pure queries; `nbytes` is a host pointer.  errors: INVALID_HANDLE, INVALID_POINTER. */
int bfBeamformGetInputBytes(bfBeamform plan, unsigned long long* nbytes);   /* ntime*nchan*ninputs*(1|2)   */
int bfBeamformGetWeightBytes(bfBeamform plan, unsigned long long* nbytes);  /* nchan*nbeam*ninputs*2       */
int bfBeamformGetOutputBytes(bfBeamform plan, unsigned long long* nbytes);  /* ntime*nchan*nbeam*8         */

/* cudaError_t of the last failing CUDA call made on behalf of this plan (0 if none). */
int bfBeamformGetLastCudaError(bfBeamform plan, int* cuda_error);

#ifdef __cplusplus
}
#endif
#endif /* BFBEAMFORM_H_ */
