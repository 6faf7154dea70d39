"""paper_1708_00720_b200 -- B200-native X-engine (cross-multiply-accumulate) of a Bifrost-style
correlator back end (arXiv:1708.00720).  The product is the C-ABI library declared in
include/bfxcorr.h and include/bfbeamform.h (built from csrc/ into libbfxcorr.so); this package is its thin ctypes binding.
"""
from .binding import (  # noqa: F401
    BF_XCORR_ALGO_SIMT,
    BF_XCORR_ALGO_TCGEN05,
    BF_XCORR_ALGO_TCGEN05_GAUSS3,
    BF_XCORR_CI4,
    BF_XCORR_CI8,
    BF_XCORR_OK,
    BfXcorrError,
    SIGNATURES,
    bfBeamformCreate,
    bfBeamformDestroy,
    bfBeamformExecute,
    bfBeamformGetInputBytes,
    bfBeamformGetLastCudaError,
    bfBeamformGetOutputBytes,
    bfBeamformGetWeightBytes,
    bfBeamformSetWeights,
    bfXcorrCreate,
    bfXcorrDestroy,
    bfXcorrDump,
    bfXcorrDumpMatrix,
    bfXcorrExecute,
    bfXcorrExecuteHost,
    bfXcorrGetInputBytes,
    bfXcorrGetKernelName,
    bfXcorrGetLastCudaError,
    bfXcorrGetLaunchCount,
    bfXcorrGetMaxSafeNtime,
    bfXcorrGetOutputBytes,
    bfXcorrGetStatusString,
    bfXcorrMemoryProbe,
    bfXcorrSetAlgo,
    lib,
)
from ._build import build, LIB_PATH  # noqa: F401
