"""oracle/ -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

Plain CPU definition of the X-engine result (oracle/xcorr_oracle.c) plus the ctypes loader
that builds and calls it.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
`--impl reference` legs may import this package.  It imports nothing from
paper_1708_00720_b200/ and shares no code with the CUDA path.
"""
from .xcorr_oracle import (  # noqa: F401
    build,
    xcorr,
    xcorr_entries,
    dump,
    dump_matrix,
    beamform,
    threads,
    set_threads,
)
