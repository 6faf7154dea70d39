"""Test-side driver of the C ABI on a CUDA device (argument marshalling only; torch provides device
memory and the stream).  Used by the `-m gpu` parity tests."""
from __future__ import annotations

from typing import Sequence

import numpy as np
import torch

import paper_1708_00720_b200 as bfx


def run_spans(spans: Sequence, ninputs: int, nchan: int, ntime: int, dtype: int, algo: int = bfx.BF_XCORR_ALGO_TCGEN05,
              poison: bool = True, first_accumulate: bool = False, init: torch.Tensor = None) -> np.ndarray:
    """Execute every span in order into one persistent device buffer (accumulate = 0 for the first
    unless `first_accumulate`), return it as int32 [nchan][B][2] on the host."""
    dev = torch.device("cuda:0")
    nb = ninputs * (ninputs + 1) // 2
    plan = bfx.bfXcorrCreate(ninputs, nchan, ntime, dtype)
    try:
        bfx.bfXcorrSetAlgo(plan, algo)
        assert bfx.bfXcorrGetOutputBytes(plan) == nchan * nb * 8
        out = torch.empty((nchan, nb, 2), dtype=torch.int32, device=dev)
        if init is not None:
            out.copy_(init)
        elif poison:
            out.fill_(0x5A5A5A5A)  # accumulate=0 must ignore whatever is there
        stream = torch.cuda.current_stream().cuda_stream
        keep = []
        for s, x in enumerate(spans):
            xd = torch.as_tensor(np.ascontiguousarray(x)).to(dev) if not isinstance(x, torch.Tensor) else x.to(dev)
            xd = xd.contiguous().view(torch.uint8).reshape(-1)
            assert xd.numel() == bfx.bfXcorrGetInputBytes(plan)
            keep.append(xd)
            bfx.bfXcorrExecute(plan, xd.data_ptr(), out.data_ptr(), first_accumulate or s > 0, stream)
        torch.cuda.synchronize()
        return out.cpu().numpy()
    finally:
        bfx.bfXcorrDestroy(plan)
