"""Test-side helpers: byte packing for hand-made spans and golden-file parsing.

Holds none of the method's arithmetic (no products, no time sums): the independent
evaluations the pins use live in the test files themselves.
"""
from __future__ import annotations

import os

import numpy as np

GOLDEN = os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden")


def pack_ci8(re: np.ndarray, im: np.ndarray) -> np.ndarray:
    """int arrays [T][C][N] -> uint8 [T][C][2N]  (byte 0 = re, byte 1 = im; reading A5)."""
    re = np.asarray(re, dtype=np.int64)
    im = np.asarray(im, dtype=np.int64)
    assert re.shape == im.shape and re.min() >= -128 and re.max() <= 127
    assert im.min() >= -128 and im.max() <= 127
    b = np.stack((re & 0xFF, im & 0xFF), axis=-1).astype(np.uint8)
    return b.reshape(*re.shape[:-1], re.shape[-1] * 2)


def pack_ci4(re: np.ndarray, im: np.ndarray) -> np.ndarray:
    """int arrays [T][C][N] -> uint8 [T][C][N]  (re = high nibble, im = low nibble; reading A4)."""
    re = np.asarray(re, dtype=np.int64)
    im = np.asarray(im, dtype=np.int64)
    assert re.shape == im.shape and re.min() >= -8 and re.max() <= 7
    assert im.min() >= -8 and im.max() <= 7
    return (((re & 0xF) << 4) | (im & 0xF)).astype(np.uint8)


def pack(dtype: int, re, im) -> np.ndarray:
    return pack_ci4(re, im) if dtype == 4 else pack_ci8(re, im)


def tri_index(i: int, j: int) -> int:
    return i * (i + 1) // 2 + j


def read_golden(name: str):
    """Parse tests/golden/<name>: returns dict(x=[(t,i,re,im)], ci8={t:bytes}, ci4={t:bytes}, v=[(k,re,im)])."""
    out = {"x": [], "ci8": {}, "ci4": {}, "v": [], "dims": {}}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            s = line.strip()
            if s.startswith("# ninputs="):
                for tok in s[2:].split():
                    if "=" in tok:
                        k, v = tok.split("=")
                        if v.isdigit():
                            out["dims"][k] = int(v)
                continue
            if not s or s.startswith("#"):
                continue
            p = s.split()
            if p[0] == "x":
                out["x"].append(tuple(int(v) for v in p[1:5]))
            elif p[0] in ("ci8", "ci4"):
                out[p[0]][int(p[1])] = bytes(int(h, 16) for h in p[2:])
            elif p[0] == "v":
                out["v"].append(tuple(int(v) for v in p[1:4]))
    return out
