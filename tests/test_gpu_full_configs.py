"""`-m gpu` parity at BASELINE.json's FULL sizes (configs[1..4]), in the launch configuration bench.py times:
same generator, same plan, all spans accumulated into one persistent buffer on the device.

What is compared, per config:
  * the oracle, bit for bit: the WHOLE output of cfg2 / cfg3 / cfg5 (the oracle needs 8 / 24 / 4 s of the box's host
    threads for them) and 64 evenly spaced channels of cfg4 (its whole output would take a minute), in channel chunks
    (channels are independent, so the oracle's output for a channel subset is exact for those channels);
  * the library's CUDA-core kernel (its own decode, tiling and indexing), bit for bit, on the WHOLE output;
  * on EVERY channel, with integer arithmetic on the device, the identities that hold at any size:
    Im V_ii = 0, Re V_ii >= 0, trace = total power, and the beam-power identity
        sum_i |w_i|^2 V_ii + 2 Re sum_{i>j} w_i conj(w_j) V_ij  =  sum_t | sum_i w_i x_i |^2
    for w = 1 (sees every Re V_ij) and w_i = j^i (sees every Im V_ij and a swapped conjugate): an O(NT) check of the
    O(N^2 T) result that touches every off-diagonal entry.
"""
from dataclasses import replace

import numpy as np
import pytest
import torch

import oracle
import paper_1708_00720_b200 as bfx
from xcorr_inputs import CONFIGS, generate_channel_slab, generate_span

pytestmark = pytest.mark.gpu


def _decode(x: torch.Tensor, cfg, nt: int):
    """(re, im) int32 [nt][C][N] of a span piece on the device (test-side arithmetic, not the product's)."""
    if cfg.dtype == 8:
        v = x.view(torch.int8).reshape(nt, cfg.nchan, cfg.ninputs, 2).to(torch.int32)
        return v[..., 0], v[..., 1]
    b = x.reshape(nt, cfg.nchan, cfg.ninputs).to(torch.int32)
    return ((b >> 4) ^ 8) - 8, ((b & 15) ^ 8) - 8


def _span_sums(x: torch.Tensor, cfg, acc):
    """Adds this span's per-channel power, |sum_i x_i|^2 and |sum_i j^i x_i|^2 (int64 [C] each) into acc."""
    dev = x.device
    q = torch.arange(cfg.ninputs, device=dev) % 4
    # j^i x = (re, im), (-im, re), (-re, -im), (im, -re)
    s_re_re = torch.tensor([1, 0, -1, 0], device=dev, dtype=torch.int32)[q]
    s_re_im = torch.tensor([0, -1, 0, 1], device=dev, dtype=torch.int32)[q]
    s_im_re = torch.tensor([0, 1, 0, -1], device=dev, dtype=torch.int32)[q]
    s_im_im = torch.tensor([1, 0, -1, 0], device=dev, dtype=torch.int32)[q]
    step = max(1, cfg.ntime // 16)
    rows = x.reshape(cfg.ntime, -1)
    for t0 in range(0, cfg.ntime, step):
        t1 = min(cfg.ntime, t0 + step)
        re, im = _decode(rows[t0:t1].reshape(-1), cfg, t1 - t0)
        acc["power"] += (re * re + im * im).sum(dim=2, dtype=torch.int64).sum(dim=0)
        yr, yi = re.sum(dim=2, dtype=torch.int64), im.sum(dim=2, dtype=torch.int64)
        acc["ones"] += (yr * yr + yi * yi).sum(dim=0)
        zr = (re * s_re_re + im * s_re_im).sum(dim=2, dtype=torch.int64)
        zi = (re * s_im_re + im * s_im_im).sum(dim=2, dtype=torch.int64)
        acc["jpow"] += (zr * zr + zi * zi).sum(dim=0)
        del re, im


def _beam_power_lhs(out: torch.Tensor, cfg):
    """sum_i |w_i|^2 V_ii + 2 Re sum_{i>j} w_i conj(w_j) V_ij per channel for w = 1 and w_i = j^i (int64 [C] each)."""
    dev = out.device
    n = cfg.ninputs
    i = torch.arange(n, device=dev).repeat_interleave(torch.arange(1, n + 1, device=dev))   # row of packed element k
    k = torch.arange(cfg.nbaselines, device=dev)
    j = k - i * (i + 1) // 2
    off = (i != j).to(torch.int64)
    d = (i - j) % 4
    # w_i conj(w_j) = j^(i-j): Re(j^d V) = re, -im, -re, +im for d = 0 .. 3
    c_re = (1 + off) * torch.tensor([1, 0, -1, 0], device=dev, dtype=torch.int64)[d]
    c_im = (1 + off) * torch.tensor([0, -1, 0, 1], device=dev, dtype=torch.int64)[d]
    ones = torch.empty(cfg.nchan, dtype=torch.int64, device=dev)
    jpow = torch.empty(cfg.nchan, dtype=torch.int64, device=dev)
    chunk = max(1, (1 << 26) // cfg.nbaselines)
    for c0 in range(0, cfg.nchan, chunk):
        v = out[c0:c0 + chunk].to(torch.int64)
        ones[c0:c0 + chunk] = (v[..., 0] * (1 + off)).sum(dim=1)
        jpow[c0:c0 + chunk] = (v[..., 0] * c_re + v[..., 1] * c_im).sum(dim=1)
        del v
    return ones, jpow


# Shapes beside BASELINE.json's that force the S1-ring code paths now that small spans are read in place (more than 8 row
# blocks AND more than 1 MiB between a channel's samples): the ci4 pair kernel and the ci8 stripe kernel through the
# ring, two accumulated spans, a sample count that is no multiple of the stage.
DERIVED = {
    "ring4": replace(CONFIGS["cfg2"], name="ring4", ninputs=1152, nchan=1024, ntime=200, nspans=2),
    "ring8": replace(CONFIGS["cfg3"], name="ring8", ninputs=1152, nchan=512, ntime=200, nspans=2, tone_channels=(3, 100)),
}

# channels compared with the oracle: None = all of them
ORACLE_CHANNELS = {"cfg2": None, "cfg3": None, "cfg5": None, "cfg4": 64, "ring4": 48, "ring8": 48}


@pytest.mark.parametrize("name", ["cfg2", "cfg3", "cfg4", "cfg5", "ring4", "ring8"])
def test_full_config_whole_output(name):
    cfg = CONFIGS[name] if name in CONFIGS else DERIVED[name]
    dev = torch.device("cuda:0")
    free, _ = torch.cuda.mem_get_info()
    need = 2 * cfg.out_bytes + 2 * cfg.span_bytes + (4 << 30)
    if free < need:
        pytest.skip("needs %.1f GB of device memory" % (need / 1e9))
    stream = torch.cuda.current_stream().cuda_stream
    plan = bfx.bfXcorrCreate(cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
    ref_plan = bfx.bfXcorrCreate(cfg.ninputs, cfg.nchan, cfg.ntime, cfg.dtype)
    bfx.bfXcorrSetAlgo(ref_plan, bfx.BF_XCORR_ALGO_SIMT)
    out = torch.full((cfg.nchan, cfg.nbaselines, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
    ref = torch.full((cfg.nchan, cfg.nbaselines, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
    sums = {k: torch.zeros(cfg.nchan, dtype=torch.int64, device=dev) for k in ("power", "ones", "jpow")}
    try:
        for s in range(cfg.nspans):
            x = generate_span(cfg, s, device=dev)
            bfx.bfXcorrExecute(plan, x.data_ptr(), out.data_ptr(), s > 0, stream)
            bfx.bfXcorrExecute(ref_plan, x.data_ptr(), ref.data_ptr(), s > 0, stream)
            _span_sums(x, cfg, sums)
            torch.cuda.synchronize()
            del x
    finally:
        bfx.bfXcorrDestroy(plan)
        bfx.bfXcorrDestroy(ref_plan)

    # the whole output against the CUDA-core kernel of the same library
    assert torch.equal(out, ref), "tensor-core output differs from the CUDA-core kernel"
    del ref

    # every channel: autocorrelations are real, non-negative and sum to the total power; beam-power identities
    i = torch.arange(cfg.ninputs, device=dev, dtype=torch.int64)
    autos = out[:, i * (i + 1) // 2 + i, :]
    assert int((autos[..., 1] != 0).sum()) == 0
    assert int((autos[..., 0] < 0).sum()) == 0
    assert torch.equal(autos[..., 0].sum(dim=1, dtype=torch.int64), sums["power"])
    ones, jpow = _beam_power_lhs(out, cfg)
    assert torch.equal(ones, sums["ones"]), "beam-power identity with w = 1 fails"
    assert torch.equal(jpow, sums["jpow"]), "beam-power identity with w_i = j^i fails"

    # the oracle, bit for bit, in channel chunks (spans regenerated per chunk on the device)
    want = ORACLE_CHANNELS[name]
    if want is None or want >= cfg.nchan:
        chans = list(range(cfg.nchan))
    else:
        chans = sorted(set(int(round(k * (cfg.nchan - 1) / (want - 1))) for k in range(want)))
    per = max(1, min(len(chans), (256 << 20) // (cfg.ntime * cfg.ninputs * cfg.bytes_per_sample)))
    per = max(per, min(len(chans), 4 * oracle.threads()))
    for a in range(0, len(chans), per):
        sub = chans[a:a + per]
        slabs = [generate_channel_slab(cfg, s, sub, device=dev).cpu().numpy() for s in range(cfg.nspans)]
        exp, nwrap = oracle.xcorr(slabs[0], cfg.ninputs, len(sub), cfg.ntime, cfg.dtype, return_nwrap=True)
        for sl in slabs[1:]:
            oracle.xcorr(sl, cfg.ninputs, len(sub), cfg.ntime, cfg.dtype, out=exp, accumulate=True)
        assert nwrap == 0
        got = out[torch.tensor(sub, device=dev)].cpu().numpy()
        np.testing.assert_array_equal(got, exp, err_msg="channels %d..%d of %s" % (sub[0], sub[-1], name))
