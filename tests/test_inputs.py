"""The seeded synthetic-span generator (xcorr_inputs): determinism, formats, distributions.

It stands in for LWA-SV F-engine captures; recipe in DESIGN.md section 4.
"""
import math

import numpy as np
import pytest
import torch

from xcorr_inputs import CONFIGS, XcorrConfig, generate_channel_slab, generate_span, gauss_thresholds, tone_offsets


def small(cfg: XcorrConfig, **kw) -> XcorrConfig:
    d = dict(cfg.__dict__)
    d.update(kw)
    return XcorrConfig(**d)


def unpack(cfg, b: torch.Tensor):
    a = b.numpy()
    if cfg.dtype == 8:
        v = a.view(np.int8).reshape(*a.shape[:-1], -1, 2)
        return v[..., 0].astype(np.int64), v[..., 1].astype(np.int64)
    hi = (a >> 4).astype(np.int64)
    lo = (a & 0xF).astype(np.int64)
    return np.where(hi > 7, hi - 16, hi), np.where(lo > 7, lo - 16, lo)


def test_config_sizes_match_baseline_json():
    c = CONFIGS
    assert (c["cfg1"].ninputs, c["cfg1"].nchan, c["cfg1"].ntime, c["cfg1"].dtype, c["cfg1"].nspans) == (16, 4, 256, 8, 1)
    assert c["cfg1"].nbaselines == 136
    assert (c["cfg2"].ninputs, c["cfg2"].nchan, c["cfg2"].ntime, c["cfg2"].dtype, c["cfg2"].nspans) == (512, 256, 2048, 4, 4)
    assert (c["cfg3"].ninputs, c["cfg3"].nchan, c["cfg3"].ntime, c["cfg3"].dtype, c["cfg3"].nspans) == (512, 3072, 1024, 8, 2)
    assert len(c["cfg3"].tone_channels) == 8
    assert (c["cfg4"].ninputs, c["cfg4"].nchan, c["cfg4"].ntime, c["cfg4"].dtype, c["cfg4"].nspans) == (2048, 1024, 1024, 8, 1)
    assert c["cfg4"].nbaselines == 2098176 and c["cfg4"].out_bytes == 17188257792
    assert (c["cfg5"].ninputs, c["cfg5"].nchan, c["cfg5"].ntime, c["cfg5"].dtype, c["cfg5"].nspans) == (64, 16384, 4096, 4, 1)
    assert c["cfg3"].span_bytes == 3 * 2**30 and c["cfg5"].span_bytes == 2**32


def test_deterministic_and_chunk_independent():
    cfg = small(CONFIGS["cfg2"], nchan=6, ntime=40, ninputs=32)
    a = generate_span(cfg, 1)
    b = generate_span(cfg, 1, max_chunk_components=1000)
    assert torch.equal(a, b)
    assert not torch.equal(a, generate_span(cfg, 0))
    slab = generate_channel_slab(cfg, 1, [4, 1])
    assert torch.equal(slab[:, 0], a[:, 4]) and torch.equal(slab[:, 1], a[:, 1])


def test_cfg1_uniform_range():
    cfg = CONFIGS["cfg1"]
    x = generate_span(cfg, 0)
    assert x.shape == (256, 4, 32) and x.dtype == torch.uint8
    re, im = unpack(cfg, x)
    for v in (re, im):
        assert v.min() >= -127 and v.max() <= 127 and -128 not in v
        assert abs(v.mean()) < 4.0 and abs(v.std() - math.sqrt((255**2 - 1) / 12)) < 2.0


@pytest.mark.parametrize("name,sigma,clip", [("cfg2", 2.5, 7), ("cfg4", 16.0, 127)])
def test_gauss_distribution(name, sigma, clip):
    cfg = small(CONFIGS[name], nchan=8, ntime=64, ninputs=64)
    re, im = unpack(cfg, generate_span(cfg, 0))
    for v in (re, im):
        assert v.min() >= -clip and v.max() <= clip
        n = v.size
        assert abs(v.mean()) < 5 * sigma / math.sqrt(n)
        var = sigma**2 + 1.0 / 12.0 if clip > 4 * sigma else None
        if var is not None:
            assert abs(v.var() - var) < 0.05 * var
    # the table is a proper CDF: monotone, symmetric tails
    thr = gauss_thresholds(sigma, clip)
    assert all(b >= a for a, b in zip(thr, thr[1:])) and len(thr) == 2 * clip
    assert abs(thr[clip - 1] + thr[clip] - 2**32) <= 2      # P(v<=-1) + P(v<=0) = 1


def test_cfg3_tone_is_constant_offset_in_tone_channels_only():
    full = CONFIGS["cfg3"]
    cfg = small(full, nchan=400, ntime=16, ninputs=32, tone_channels=(191,))
    noise = small(cfg, tone_channels=(), tone_amplitude=0)
    xr, xi = unpack(cfg, generate_span(cfg, 0))
    nr, ni = unpack(noise, generate_span(noise, 0))
    tre, tim = tone_offsets(cfg.ninputs, cfg.tone_amplitude)
    other = [c for c in range(cfg.nchan) if c != 191]
    assert (xr[:, other] == nr[:, other]).all() and (xi[:, other] == ni[:, other]).all()
    assert (xr[:, 191] == np.clip(nr[:, 191] + np.array(tre), -127, 127)).all()
    assert (xi[:, 191] == np.clip(ni[:, 191] + np.array(tim), -127, 127)).all()
    assert all(abs(r * r + i * i - 24 * 24) <= 2 * 24 + 1 for r, i in zip(tre, tim))


@pytest.mark.gpu
def test_device_generation_matches_host():
    for name in ("cfg1", "cfg2", "cfg3"):
        cfg = small(CONFIGS[name], nchan=min(CONFIGS[name].nchan, 200), ntime=32, ninputs=64)
        if cfg.tone_channels:
            cfg = small(cfg, tone_channels=(191,))
        assert torch.equal(generate_span(cfg, 1), generate_span(cfg, 1, device="cuda").cpu())


def test_weights_cover_the_whole_int8_range():
    """generate_weights draws every code, -128 included, for both parts (reading B4)."""
    from xcorr_inputs import generate_weights
    w = generate_weights(7, 4, 8, 256).view(torch.int8).reshape(4, 8, 256, 2)
    for part in (0, 1):
        v = w[..., part]
        assert int(v.min()) == -128 and int(v.max()) == 127
        assert abs(float(v.float().mean())) < 3.0
    sub = generate_weights(7, 4, 8, 256, channels=[2])
    assert torch.equal(sub[0], generate_weights(7, 4, 8, 256)[2])
