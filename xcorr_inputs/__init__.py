"""Seeded synthetic station-shaped voltages for the X-engine (shared by tests, bench and smoke).

This module holds NONE of the method's arithmetic (no products, no sums over time, no
triangle indexing): it only draws integers from a counter-based generator and packs them
into the ci4 / ci8 byte formats of `include/bfxcorr.h`.  It is the one module that both
the CUDA path's callers and the oracle's callers may import (task statement, section (3)).

The synthetic spans stand in for LWA-SV F-engine captures, which are not available here:
station shape from PAPER.md:531 (256 dual-pol antennas = 512 inputs)
(25 kHz channels, 40 us samples) and PAPER.md:543 ("4+4 complex signed integers");
value distributions from BASELINE.json `configs[0..4]`; recipe in DESIGN.md section 4.
"""
from .gen import (  # noqa: F401
    CONFIGS,
    XcorrConfig,
    component_values,
    generate_span,
    generate_channel_slab,
    gauss_thresholds,
    tone_offsets,
    generate_weights,
)
