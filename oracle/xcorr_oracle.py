"""ctypes loader for oracle/xcorr_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Builds the plain-C oracle with gcc (`-O3 -march=native -fopenmp`) into a per-machine
directory (the GPU box's host CPU may differ from the build container's, and built `.so`
files travel with gpurun snapshots) and exposes it on numpy arrays.  No arithmetic of the
method lives here: argument marshalling only.  See xcorr_oracle.c for the definition
(BASELINE.json north_star).
"""
from __future__ import annotations

import ctypes
import hashlib
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "xcorr_oracle.c")
_LIB: Optional[ctypes.CDLL] = None


def _machine_tag() -> str:
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags") or line.startswith("model name"):
                    flags += line
                    if line.startswith("flags"):
                        break
    except OSError:
        pass
    with open(_SRC, "rb") as f:
        src = f.read()
    return hashlib.sha1(flags.encode() + src).hexdigest()[:12]


def build(force: bool = False) -> str:
    """Compile the oracle for this machine; returns the path of the shared library."""
    out_dir = os.path.join(_HERE, "_build", _machine_tag())
    so = os.path.join(out_dir, "libxcorr_oracle.so")
    if force or not os.path.exists(so):
        os.makedirs(out_dir, exist_ok=True)
        tmp = so + ".tmp%d" % os.getpid()
        cmd = ["gcc", "-std=c11", "-O3", "-march=native", "-fopenmp", "-shared", "-fPIC",
               "-o", tmp, _SRC]
        subprocess.run(cmd, check=True)
        os.replace(tmp, so)
    return so


def _lib() -> ctypes.CDLL:
    global _LIB
    if _LIB is None:
        lib = ctypes.CDLL(build())
        lib.xcorr_oracle.restype = ctypes.c_longlong
        lib.xcorr_oracle.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int,
                                     ctypes.c_int, ctypes.c_int, ctypes.c_int]
        lib.xcorr_oracle_entries.restype = ctypes.c_int
        lib.xcorr_oracle_entries.argtypes = [ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                             ctypes.c_int, ctypes.c_longlong, ctypes.c_void_p,
                                             ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p]
        lib.xcorr_oracle_threads.restype = ctypes.c_int
        lib.xcorr_oracle_set_threads.argtypes = [ctypes.c_int]
        _LIB = lib
    return _LIB


def _check_in(x: np.ndarray, ninputs: int, nchan: int, ntime: int, dtype: int) -> np.ndarray:
    x = np.ascontiguousarray(x).view(np.uint8).reshape(-1)
    bps = 1 if dtype == 4 else 2
    if x.size != ntime * nchan * ninputs * bps:
        raise ValueError("input span has %d bytes, expected %d" % (x.size, ntime * nchan * ninputs * bps))
    return x


def xcorr(x: np.ndarray, ninputs: int, nchan: int, ntime: int, dtype: int,
          out: Optional[np.ndarray] = None, accumulate: bool = False,
          return_nwrap: bool = False):
    """Whole span -> int32 [nchan][B][2].  `out` (if given) is updated in place."""
    x = _check_in(x, ninputs, nchan, ntime, dtype)
    nb = ninputs * (ninputs + 1) // 2
    if out is None:
        if accumulate:
            raise ValueError("accumulate needs an existing `out`")
        out = np.empty((nchan, nb, 2), dtype=np.int32)
    if out.dtype != np.int32 or out.size != nchan * nb * 2 or not out.flags.c_contiguous:
        raise ValueError("`out` must be C-contiguous int32 [nchan][B][2]")
    nwrap = _lib().xcorr_oracle(x.ctypes.data, out.ctypes.data, ninputs, nchan, ntime, dtype,
                                1 if accumulate else 0)
    if nwrap < 0:
        raise ValueError("xcorr_oracle rejected its arguments")
    return (out, int(nwrap)) if return_nwrap else out


def xcorr_entries(x: np.ndarray, ninputs: int, nchan: int, ntime: int, dtype: int,
                  c: np.ndarray, i: np.ndarray, j: np.ndarray) -> np.ndarray:
    """Selected (c, i, j) entries, any i, j (upper triangle too) -> int64 [n][2] (not wrapped)."""
    x = _check_in(x, ninputs, nchan, ntime, dtype)
    c = np.ascontiguousarray(c, dtype=np.int32)
    i = np.ascontiguousarray(i, dtype=np.int32)
    j = np.ascontiguousarray(j, dtype=np.int32)
    n = c.size
    if i.size != n or j.size != n:
        raise ValueError("c, i, j must have the same length")
    vals = np.empty((n, 2), dtype=np.int64)
    rc = _lib().xcorr_oracle_entries(x.ctypes.data, ninputs, nchan, ntime, dtype, n,
                                     c.ctypes.data, i.ctypes.data, j.ctypes.data, vals.ctypes.data)
    if rc != 0:
        raise ValueError("xcorr_oracle_entries rejected its arguments")
    return vals


def dump(acc: np.ndarray, scale: float = 1.0, zero_acc: bool = False) -> np.ndarray:
    """Integration dump: int32 [..][2] accumulator -> float32 of the same shape, `acc` cleared in place if asked."""
    if acc.dtype != np.int32 or not acc.flags.c_contiguous:
        raise ValueError("`acc` must be C-contiguous int32")
    out = np.empty(acc.shape, dtype=np.float32)
    fn = _lib().xcorr_oracle_dump
    fn.restype = ctypes.c_longlong
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_longlong, ctypes.c_float, ctypes.c_int]
    if fn(acc.ctypes.data, out.ctypes.data, acc.size, float(scale), 1 if zero_acc else 0) != acc.size:
        raise ValueError("xcorr_oracle_dump rejected its arguments")
    return out


def dump_matrix(acc: np.ndarray, ninputs: int, scale: float = 1.0, zero_acc: bool = False) -> np.ndarray:
    """Integration dump with reorder: int32 [nchan][B][2] -> float32 full Hermitian matrices [nchan][ninputs][ninputs][2]."""
    nb = ninputs * (ninputs + 1) // 2
    if acc.dtype != np.int32 or not acc.flags.c_contiguous or acc.ndim != 3 or acc.shape[1:] != (nb, 2):
        raise ValueError("`acc` must be C-contiguous int32 [nchan][B][2]")
    nchan = acc.shape[0]
    out = np.empty((nchan, ninputs, ninputs, 2), dtype=np.float32)
    fn = _lib().xcorr_oracle_dump_matrix
    fn.restype = ctypes.c_longlong
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int, ctypes.c_int, ctypes.c_float, ctypes.c_int]
    if fn(acc.ctypes.data, out.ctypes.data, ninputs, nchan, float(scale), 1 if zero_acc else 0) != nchan * ninputs * ninputs:
        raise ValueError("xcorr_oracle_dump_matrix rejected its arguments")
    return out


def beamform(x: np.ndarray, w: np.ndarray, ninputs: int, nchan: int, ntime: int, nbeam: int, dtype: int,
             return_nwrap: bool = False):
    """Phase-and-sum beamformer: span x, ci8 weights [nchan][nbeam][ninputs] -> int32 [ntime][nchan][nbeam][2]."""
    x = _check_in(x, ninputs, nchan, ntime, dtype)
    w = np.ascontiguousarray(w).view(np.uint8).reshape(-1)
    if w.size != nchan * nbeam * ninputs * 2:
        raise ValueError("weights have %d bytes, expected %d" % (w.size, nchan * nbeam * ninputs * 2))
    out = np.empty((ntime, nchan, nbeam, 2), dtype=np.int32)
    fn = _lib().xcorr_oracle_beamform
    fn.restype = ctypes.c_longlong
    fn.argtypes = [ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p] + [ctypes.c_int] * 5
    nwrap = fn(x.ctypes.data, w.ctypes.data, out.ctypes.data, ninputs, nchan, ntime, nbeam, dtype)
    if nwrap < 0:
        raise ValueError("xcorr_oracle_beamform rejected its arguments")
    return (out, int(nwrap)) if return_nwrap else out


def threads() -> int:
    return int(_lib().xcorr_oracle_threads())


def set_threads(n: int) -> None:
    _lib().xcorr_oracle_set_threads(int(n))
