"""ctypes binding of include/bfxcorr.h -- argument marshalling only.

Same names as the C ABI.  Every step of the hot path (unpack, tile scheduling, tensor-core
contraction, span-accumulate epilogue) runs inside libbfxcorr.so's CUDA kernels; this module never
computes anything and never falls back to a CPU implementation: if the library cannot be built or
loaded, importing callers get an exception.  torch is used by callers for device memory and streams.
"""
from __future__ import annotations

import ctypes
from typing import Optional

from . import _build

BF_XCORR_CI4 = 4
BF_XCORR_CI8 = 8
BF_XCORR_OK = 0
BF_XCORR_SCRATCH_LIMIT = 9
BF_XCORR_ALGO_TCGEN05 = 0
BF_XCORR_ALGO_SIMT = 1
BF_XCORR_ALGO_TCGEN05_GAUSS3 = 2

_vp = ctypes.c_void_p
_i = ctypes.c_int
_ullp = ctypes.POINTER(ctypes.c_ulonglong)
_ip = ctypes.POINTER(ctypes.c_int)

# name -> (restype, argtypes); mirrors include/bfxcorr.h and include/bfbeamform.h one to one
SIGNATURES = {
    "bfXcorrCreate": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i]),
    "bfXcorrExecute": (_i, [_vp, _vp, _vp, _i, _vp]),
    "bfXcorrDestroy": (_i, [_vp]),
    "bfXcorrGetInputBytes": (_i, [_vp, _ullp]),
    "bfXcorrGetOutputBytes": (_i, [_vp, _ullp]),
    "bfXcorrGetMaxSafeNtime": (_i, [_vp, _ullp]),
    "bfXcorrSetAlgo": (_i, [_vp, _i]),
    "bfXcorrGetLaunchCount": (_i, [_vp, _ip]),
    "bfXcorrGetLastCudaError": (_i, [_vp, _ip]),
    "bfXcorrExecuteHost": (_i, [_vp, _vp, _vp, _vp, _i, _vp]),
    "bfXcorrDump": (_i, [_vp, _vp, _vp, ctypes.c_float, _i, _vp]),
    "bfXcorrDumpMatrix": (_i, [_vp, _vp, _vp, ctypes.c_float, _i, _vp]),
    "bfXcorrMemoryProbe": (_i, [_vp, _vp, _vp, _i, _vp]),
    "bfXcorrExecuteNoAlloc": (_i, [_vp, _vp, _i, _i, _i, _i, _i, _vp]),
    "bfXcorrGetStatusString": (ctypes.c_char_p, [_i]),
    "bfXcorrGetKernelName": (ctypes.c_char_p, [_vp, _i]),
    # include/bfbeamform.h
    "bfBeamformCreate": (_i, [ctypes.POINTER(_vp), _i, _i, _i, _i, _i]),
    "bfBeamformSetWeights": (_i, [_vp, _vp, _vp]),
    "bfBeamformExecute": (_i, [_vp, _vp, _vp, _vp]),
    "bfBeamformDestroy": (_i, [_vp]),
    "bfBeamformGetInputBytes": (_i, [_vp, _ullp]),
    "bfBeamformGetWeightBytes": (_i, [_vp, _ullp]),
    "bfBeamformGetOutputBytes": (_i, [_vp, _ullp]),
    "bfBeamformGetLastCudaError": (_i, [_vp, _ip]),
}

_LIB: Optional[ctypes.CDLL] = None


def lib() -> ctypes.CDLL:
    """Load (building if needed) libbfxcorr.so and declare every prototype."""
    global _LIB
    if _LIB is None:
        handle = ctypes.CDLL(_build.build())
        for name, (res, args) in SIGNATURES.items():
            fn = getattr(handle, name)
            fn.restype = res
            fn.argtypes = args
        _LIB = handle
    return _LIB


class BfXcorrError(RuntimeError):
    def __init__(self, status: int, where: str):
        self.status = status
        super().__init__("%s failed: %s (%d)" % (where, bfXcorrGetStatusString(status), status))


def _check(status: int, where: str) -> None:
    if status != BF_XCORR_OK:
        raise BfXcorrError(status, where)


def bfXcorrGetStatusString(status: int) -> str:
    return lib().bfXcorrGetStatusString(int(status)).decode()


def bfXcorrCreate(ninputs: int, nchan: int, ntime: int, dtype: int) -> _vp:
    plan = _vp()
    _check(lib().bfXcorrCreate(ctypes.byref(plan), ninputs, nchan, ntime, dtype), "bfXcorrCreate")
    return plan


def bfXcorrExecute(plan: _vp, in_ptr: int, out_ptr: int, accumulate: bool, stream: int = 0) -> None:
    """in_ptr / out_ptr: device addresses (tensor.data_ptr()); stream: cudaStream_t as int."""
    _check(lib().bfXcorrExecute(plan, _vp(in_ptr), _vp(out_ptr), 1 if accumulate else 0, _vp(stream)),
           "bfXcorrExecute")


def bfXcorrExecuteHost(plan: _vp, in_host_ptr: int, out_dev_ptr: int, out_host_ptr: int, accumulate: bool,
                       stream: int = 0) -> None:
    _check(lib().bfXcorrExecuteHost(plan, _vp(in_host_ptr), _vp(out_dev_ptr), _vp(out_host_ptr or None),
                                    1 if accumulate else 0, _vp(stream)), "bfXcorrExecuteHost")


def bfXcorrDump(plan: _vp, acc_ptr: int, out_ptr: int, scale: float = 1.0, zero_acc: bool = False, stream: int = 0) -> None:
    """acc_ptr: device int32 visibilities; out_ptr: device float32 buffer of the same size."""
    _check(lib().bfXcorrDump(plan, _vp(acc_ptr), _vp(out_ptr), ctypes.c_float(scale), 1 if zero_acc else 0, _vp(stream)),
           "bfXcorrDump")


def bfXcorrDumpMatrix(plan: _vp, acc_ptr: int, out_ptr: int, scale: float = 1.0, zero_acc: bool = False, stream: int = 0) -> None:
    """acc_ptr: device int32 visibilities; out_ptr: device float32 [nchan][ninputs][ninputs][2] (full Hermitian matrices)."""
    _check(lib().bfXcorrDumpMatrix(plan, _vp(acc_ptr), _vp(out_ptr), ctypes.c_float(scale), 1 if zero_acc else 0, _vp(stream)),
           "bfXcorrDumpMatrix")


def bfXcorrMemoryProbe(plan: _vp, in_ptr: int, out_ptr: int, accumulate: bool, stream: int = 0) -> None:
    """No-math streaming kernel with the path's HBM access mix (measurement aid); `out` is left with meaningless values."""
    _check(lib().bfXcorrMemoryProbe(plan, _vp(in_ptr), _vp(out_ptr), 1 if accumulate else 0, _vp(stream)), "bfXcorrMemoryProbe")


def bfXcorrExecuteNoAlloc(in_ptr: int, out_ptr: int, ninputs: int, nchan: int, ntime: int, dtype: int, accumulate: bool,
                          stream: int = 0) -> None:
    """One span without a plan and without any device allocation (scratch in the library's static device array)."""
    _check(lib().bfXcorrExecuteNoAlloc(_vp(in_ptr), _vp(out_ptr), ninputs, nchan, ntime, dtype, 1 if accumulate else 0, _vp(stream)),
           "bfXcorrExecuteNoAlloc")


def bfXcorrDestroy(plan: _vp) -> None:
    _check(lib().bfXcorrDestroy(plan), "bfXcorrDestroy")


def _get_ull(fn_name: str, plan: _vp) -> int:
    v = ctypes.c_ulonglong(0)
    _check(getattr(lib(), fn_name)(plan, ctypes.byref(v)), fn_name)
    return int(v.value)


def bfXcorrGetInputBytes(plan: _vp) -> int:
    return _get_ull("bfXcorrGetInputBytes", plan)


def bfXcorrGetOutputBytes(plan: _vp) -> int:
    return _get_ull("bfXcorrGetOutputBytes", plan)


def bfXcorrGetMaxSafeNtime(plan: _vp) -> int:
    return _get_ull("bfXcorrGetMaxSafeNtime", plan)


def bfXcorrSetAlgo(plan: _vp, algo: int) -> None:
    _check(lib().bfXcorrSetAlgo(plan, algo), "bfXcorrSetAlgo")


def bfXcorrGetKernelName(plan: _vp, accumulate: bool) -> str:
    return lib().bfXcorrGetKernelName(plan, 1 if accumulate else 0).decode()


def bfXcorrGetLaunchCount(plan: _vp) -> int:
    v = ctypes.c_int(0)
    _check(lib().bfXcorrGetLaunchCount(plan, ctypes.byref(v)), "bfXcorrGetLaunchCount")
    return int(v.value)


def bfXcorrGetLastCudaError(plan: _vp) -> int:
    v = ctypes.c_int(0)
    _check(lib().bfXcorrGetLastCudaError(plan, ctypes.byref(v)), "bfXcorrGetLastCudaError")
    return int(v.value)


# ---- include/bfbeamform.h ---------------------------------------------------------------------
def bfBeamformCreate(ninputs: int, nchan: int, ntime: int, nbeam: int, dtype: int) -> _vp:
    plan = _vp()
    _check(lib().bfBeamformCreate(ctypes.byref(plan), ninputs, nchan, ntime, nbeam, dtype), "bfBeamformCreate")
    return plan


def bfBeamformSetWeights(plan: _vp, weights_ptr: int, stream: int = 0) -> None:
    """weights_ptr: device address of the ci8 weights [nchan][nbeam][ninputs]; synchronises `stream`."""
    _check(lib().bfBeamformSetWeights(plan, _vp(weights_ptr), _vp(stream)), "bfBeamformSetWeights")


def bfBeamformExecute(plan: _vp, in_ptr: int, out_ptr: int, stream: int = 0) -> None:
    _check(lib().bfBeamformExecute(plan, _vp(in_ptr), _vp(out_ptr), _vp(stream)), "bfBeamformExecute")


def bfBeamformDestroy(plan: _vp) -> None:
    _check(lib().bfBeamformDestroy(plan), "bfBeamformDestroy")


def bfBeamformGetInputBytes(plan: _vp) -> int:
    return _get_ull("bfBeamformGetInputBytes", plan)


def bfBeamformGetWeightBytes(plan: _vp) -> int:
    return _get_ull("bfBeamformGetWeightBytes", plan)


def bfBeamformGetOutputBytes(plan: _vp) -> int:
    return _get_ull("bfBeamformGetOutputBytes", plan)


def bfBeamformGetLastCudaError(plan: _vp) -> int:
    v = ctypes.c_int(0)
    _check(lib().bfBeamformGetLastCudaError(plan, ctypes.byref(v)), "bfBeamformGetLastCudaError")
    return int(v.value)
