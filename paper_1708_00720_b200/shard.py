"""Channel sharding for more than one GPU.

Channels are independent -- V[c] depends only on x[.][c][.] -- so the X-engine shards by channel with no
exchange step: rank r of `world` owns a contiguous block of channels, its own input shard
x[t][c0:c1][i] and its own output slab out[c0:c1][B].  No collective touches the data path; this module is
host-side index arithmetic only (the deployment splits the band across servers
in the same way).
"""
from __future__ import annotations

from typing import Tuple


def channel_shard(nchan: int, world: int, rank: int) -> Tuple[int, int]:
    """[c0, c1) of `rank`: contiguous, disjoint, covering [0, nchan), sizes differing by at most one."""
    if world <= 0 or not 0 <= rank < world or nchan < 0:
        raise ValueError("bad shard request: nchan=%d world=%d rank=%d" % (nchan, world, rank))
    base, extra = divmod(nchan, world)
    c0 = rank * base + min(rank, extra)
    return c0, c0 + base + (1 if rank < extra else 0)
