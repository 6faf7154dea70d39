"""Counter-based integer generator for X-engine input spans.

Every real component (re or im of one complex sample) has a global 64-bit counter

    g = 2 * ((((span * T) + t) * C + c) * N + i) + part        part: 0 = re, 1 = im

and its value is a pure function of (seed, g).  Host (torch CPU) and device (torch CUDA)
evaluate the same int64 expressions, so they produce identical bytes; subsets (one
channel, a few time rows) can be regenerated anywhere without the full span.

    z  = seed XOR (g * 0x9E3779B97F4A7C15)              (mod 2^64)
    z  = (z XOR (z >> 30)) * 0xBF58476D1CE4E5B9         (splitmix64 finaliser)
    z  = (z XOR (z >> 27)) * 0x94D049BB133111EB
    z  =  z XOR (z >> 31)
    r  = z >> 32                                         (32 uniform bits)

    uniform127 : v = (r mod 255) - 127
    gauss      : v = #{k : r >= thr[k]} - clip,  thr[k] = floor(2^32 * Phi((k - clip + 1/2) / sigma))
                 i.e. round(N(0, sigma)) clipped to [-clip, clip]  (BASELINE.json configs:
                 the second parameter is read as the standard deviation, reading A11)

Optional tone (BASELINE.json configs[2]): in the listed channels a per-input constant
integer offset (round(A cos phi_i), round(A sin phi_i)) is added before clipping.

Byte formats (include/bfxcorr.h): ci8 = (int8 re, int8 im); ci4 = one byte, re in the high
nibble, im in the low nibble, both two's complement.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional, Sequence, Tuple

import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    """Python int -> the int64 with the same low 64 bits."""
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_GOLDEN = _s64(0x9E3779B97F4A7C15)
_MUL1 = _s64(0xBF58476D1CE4E5B9)
_MUL2 = _s64(0x94D049BB133111EB)


@dataclass(frozen=True)
class XcorrConfig:
    name: str
    ninputs: int
    nchan: int
    ntime: int
    dtype: int  # 4 = ci4, 8 = ci8
    nspans: int
    dist: str  # "uniform127" | "gauss"
    sigma: float = 0.0
    clip: int = 127
    seed: int = 0
    tone_channels: Tuple[int, ...] = ()
    tone_amplitude: int = 0
    note: str = ""

    @property
    def bytes_per_sample(self) -> int:
        return 1 if self.dtype == 4 else 2

    @property
    def nbaselines(self) -> int:
        return self.ninputs * (self.ninputs + 1) // 2

    @property
    def span_bytes(self) -> int:
        return self.ntime * self.nchan * self.ninputs * self.bytes_per_sample

    @property
    def out_bytes(self) -> int:
        return self.nchan * self.nbaselines * 8


# BASELINE.json configs[0..4]
CONFIGS = {
    "cfg1": XcorrConfig("cfg1", 16, 4, 256, 8, 1, "uniform127", seed=0xB1F00001,
                        note="tiny correctness case"),
    "cfg2": XcorrConfig("cfg2", 512, 256, 2048, 4, 4, "gauss", sigma=2.5, clip=7, seed=0xB1F00002,
                        note="LWA-station-shaped ci4, 4 spans"),
    "cfg3": XcorrConfig("cfg3", 512, 3072, 1024, 8, 2, "gauss", sigma=16.0, clip=127, seed=0xB1F00003,
                        tone_channels=tuple(191 + 384 * m for m in range(8)), tone_amplitude=24,
                        note="LWA-station-shaped ci8 with a common tone in 8 channels, 2 spans"),
    "cfg4": XcorrConfig("cfg4", 2048, 1024, 1024, 8, 1, "gauss", sigma=16.0, clip=127, seed=0xB1F00004,
                        note="larger array ci8, single span"),
    "cfg5": XcorrConfig("cfg5", 64, 16384, 4096, 4, 1, "gauss", sigma=2.5, clip=7, seed=0xB1F00005,
                        note="few-input bandwidth-bound ci4, single span"),
}


def gauss_thresholds(sigma: float, clip: int) -> list:
    """Cumulative table of round(N(0,sigma)) clipped to [-clip,clip], scaled to 2^32.

    thr[k] (k = 0 .. 2*clip-1) = floor(2^32 * P(v <= k - clip)); tails fold into +-clip.
    """
    thr = []
    for k in range(2 * clip):
        v = k - clip
        p = 0.5 * (1.0 + math.erf((v + 0.5) / (sigma * math.sqrt(2.0))))
        thr.append(min((1 << 32) - 1, int(math.floor(p * 4294967296.0))))
    return thr


def tone_offsets(ninputs: int, amplitude: int) -> Tuple[list, list]:
    """Per-input integer tone offsets: phi_i = 2 pi frac(i * 0.6180339887)."""
    re, im = [], []
    for i in range(ninputs):
        phi = 2.0 * math.pi * math.fmod(i * 0.6180339887, 1.0)
        re.append(int(round(amplitude * math.cos(phi))))
        im.append(int(round(amplitude * math.sin(phi))))
    return re, im


def _lsr(z: torch.Tensor, s: int) -> torch.Tensor:
    """Logical right shift of int64 (torch's >> is arithmetic)."""
    return (z >> s) & ((1 << (64 - s)) - 1)


def _uniform32(seed: int, g: torch.Tensor) -> torch.Tensor:
    """32 uniform bits (as non-negative int64) for each int64 counter in g."""
    z = (g * _GOLDEN) ^ _s64(seed)
    z = (z ^ _lsr(z, 30)) * _MUL1
    z = (z ^ _lsr(z, 27)) * _MUL2
    z = z ^ _lsr(z, 31)
    return _lsr(z, 32)


def component_values(cfg: XcorrConfig, span: int, t: torch.Tensor, c: torch.Tensor,
                     i: torch.Tensor) -> Tuple[torch.Tensor, torch.Tensor]:
    """Integer (re, im) of the samples at broadcastable int64 index tensors (t, c, i)."""
    dev = t.device
    lin = ((span * cfg.ntime + t) * cfg.nchan + c) * cfg.ninputs + i
    out = []
    for part in (0, 1):
        r = _uniform32(cfg.seed, lin * 2 + part)
        if cfg.dist == "uniform127":
            v = torch.remainder(r, 255) - 127
        elif cfg.dist == "gauss":
            thr = torch.tensor(gauss_thresholds(cfg.sigma, cfg.clip), dtype=torch.int64, device=dev)
            v = torch.bucketize(r, thr, right=True) - cfg.clip
        else:
            raise ValueError(cfg.dist)
        out.append(v)
    re, im = out
    if cfg.tone_channels:
        tre, tim = tone_offsets(cfg.ninputs, cfg.tone_amplitude)
        tre = torch.tensor(tre, dtype=torch.int64, device=dev)
        tim = torch.tensor(tim, dtype=torch.int64, device=dev)
        is_tone = torch.zeros(cfg.nchan, dtype=torch.bool, device=dev)
        is_tone[list(cfg.tone_channels)] = True
        m = is_tone[c].to(torch.int64)
        re = torch.clamp(re + m * tre[i], -cfg.clip, cfg.clip)
        im = torch.clamp(im + m * tim[i], -cfg.clip, cfg.clip)
    return re, im


def _pack(cfg: XcorrConfig, re: torch.Tensor, im: torch.Tensor) -> torch.Tensor:
    """(re, im) int64 [..., N] -> uint8 [..., N * bytes_per_sample]."""
    if cfg.dtype == 8:
        b = torch.stack((re & 0xFF, im & 0xFF), dim=-1).to(torch.uint8)
        return b.reshape(*re.shape[:-1], re.shape[-1] * 2)
    return (((re & 0xF) << 4) | (im & 0xF)).to(torch.uint8)


def generate_span(cfg: XcorrConfig, span: int, device="cpu", out: Optional[torch.Tensor] = None,
                  max_chunk_components: int = 1 << 25) -> torch.Tensor:
    """One dense span [ntime][nchan][ninputs * bytes_per_sample] of uint8 on `device`."""
    T, C, N = cfg.ntime, cfg.nchan, cfg.ninputs
    row = N * cfg.bytes_per_sample
    if out is None:
        out = torch.empty((T, C, row), dtype=torch.uint8, device=device)
    assert out.shape == (T, C, row) and out.dtype == torch.uint8
    dev = out.device
    c = torch.arange(C, dtype=torch.int64, device=dev).view(1, C, 1)
    i = torch.arange(N, dtype=torch.int64, device=dev).view(1, 1, N)
    rows_per_chunk = max(1, max_chunk_components // (C * N))
    for t0 in range(0, T, rows_per_chunk):
        t1 = min(T, t0 + rows_per_chunk)
        t = torch.arange(t0, t1, dtype=torch.int64, device=dev).view(-1, 1, 1)
        re, im = component_values(cfg, span, t, c, i)
        out[t0:t1] = _pack(cfg, re, im)
    return out


def generate_channel_slab(cfg: XcorrConfig, span: int, channels: Sequence[int],
                          device="cpu") -> torch.Tensor:
    """The bytes of selected channels only: uint8 [ntime][len(channels)][row bytes]."""
    T, N = cfg.ntime, cfg.ninputs
    t = torch.arange(T, dtype=torch.int64, device=device).view(T, 1, 1)
    c = torch.tensor(list(channels), dtype=torch.int64, device=device).view(1, -1, 1)
    i = torch.arange(N, dtype=torch.int64, device=device).view(1, 1, N)
    re, im = component_values(cfg, span, t, c, i)
    return _pack(cfg, re, im)


def generate_weights(seed: int, nchan: int, nbeam: int, ninputs: int, channels: Optional[Sequence[int]] = None,
                     device="cpu") -> torch.Tensor:
    """Beamformer weights, ci8 [nchan][nbeam][2 * ninputs] uint8 (byte 0 = re, byte 1 = im), each component a seeded
    uniform integer over the whole int8 range [-128, 127]; they stand in for quantised steering phasors (SURVEY.md
    section 8(f) N1).  `channels` selects rows of the same draw."""
    cs = list(range(nchan)) if channels is None else list(channels)
    c = torch.tensor(cs, dtype=torch.int64, device=device).view(-1, 1, 1)
    k = torch.arange(nbeam, dtype=torch.int64, device=device).view(1, -1, 1)
    j = torch.arange(2 * ninputs, dtype=torch.int64, device=device).view(1, 1, -1)
    r = _uniform32(seed ^ 0x5EED0BEA, (c * nbeam + k) * (2 * ninputs) + j)
    return (r & 0xFF).to(torch.uint8)   # 256 equally likely codes = uniform over [-128, 127] in two's complement
