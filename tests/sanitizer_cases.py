"""Driver for compute-sanitizer runs (racecheck / synccheck on small configs; the mbarrier and TMEM
protocols are the risk).  Runs the tensor-core path on BASELINE.json configs[0], on one shape that reads the span in place
and on one that goes through the S1 ring (more than 8 row blocks and more than 1 MiB between a channel's samples),
two accumulating launches each, and compares with the library's CUDA-core kernel.  Not collected by pytest:

    compute-sanitizer --tool racecheck python tests/sanitizer_cases.py
    compute-sanitizer --tool synccheck python tests/sanitizer_cases.py
"""
import os
import sys

import torch

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
import paper_1708_00720_b200 as bfx  # noqa: E402

SHAPES = [(16, 4, 256, 8), (192, 6, 160, 8), (128, 3, 96, 4), (64, 8, 200, 4), (1152, 460, 130, 8), (1152, 920, 130, 4)]


def main():
    dev = torch.device("cuda:0")
    stream = torch.cuda.current_stream().cuda_stream
    only = [int(a) for a in sys.argv[1:]] or range(len(SHAPES))
    for k in only:
        N, C, T, dt = SHAPES[k]
        nb = N * (N + 1) // 2
        g = torch.Generator(device=dev)
        g.manual_seed(N + C + T + dt)
        spans = [torch.randint(0, 256, (T * C * N * (1 if dt == 4 else 2),), dtype=torch.uint8, device=dev, generator=g)
                 for _ in range(2)]
        res = []
        for algo in (bfx.BF_XCORR_ALGO_TCGEN05, bfx.BF_XCORR_ALGO_SIMT):
            plan = bfx.bfXcorrCreate(N, C, T, dt)
            bfx.bfXcorrSetAlgo(plan, algo)
            out = torch.full((C, nb, 2), 0x5A5A5A5A, dtype=torch.int32, device=dev)
            for s, x in enumerate(spans):
                bfx.bfXcorrExecute(plan, x.data_ptr(), out.data_ptr(), s > 0, stream)
            torch.cuda.synchronize()
            if algo == bfx.BF_XCORR_ALGO_TCGEN05:
                print("shape", SHAPES[k], bfx.bfXcorrGetKernelName(plan, False), "|", bfx.bfXcorrGetKernelName(plan, True), flush=True)
            bfx.bfXcorrDestroy(plan)
            res.append(out)
        assert torch.equal(res[0], res[1]), "tensor-core output differs from the CUDA-core kernel: %s" % (SHAPES[k],)
    print("sanitizer cases OK")


if __name__ == "__main__":
    main()
