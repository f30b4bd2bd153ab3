"""Seeded synthetic tone sets shaped like the paper's workloads.

This package is the ONLY code shared by the oracle (``oracle/``) and the CUDA
path (``paper_2403_15582_b200/``).  It holds no synthesis arithmetic: it draws
random numbers and lays out per-tone parameter arrays, nothing else.  No phase,
no sine, no quantiser lives here.

The five configurations are the ones listed in ``BASELINE.json`` ``configs``
(recipe and draw order: ``SURVEY.md`` section 8(d), restated in ``DESIGN.md``).
They stand in for the paper's own workloads, none of which is a public data
set: the equally spaced comb of PAPER.md:198-206 (section V.A), the streaming
capacity runs of PAPER.md:221-227 (section V.B) and the 1000-tone / 35 ms
playback of PAPER.md:246 (section V.C).
"""
from .configs import (  # noqa: F401
    PROFILE_STATIC,
    PROFILE_LINEAR,
    PROFILE_MINJERK,
    PROFILE_EXP,
    DEFAULT_SCALE,
    Update,
    Workload,
    config1,
    config2,
    config3,
    config4,
    config5_cell,
    config5_grid,
    capacity_toneset,
    comb_toneset,
    fast_mover_stream,
    by_name,
)
