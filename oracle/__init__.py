"""ORACLE -- test infrastructure, not product code.  See awg_oracle.py for what it computes.

Only ``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` /
``--impl reference`` legs may import this package.  The CUDA path never does.
"""
from .awg_oracle import (  # noqa: F401
    LD,
    PROFILE_STATIC,
    PROFILE_LINEAR,
    PROFILE_MINJERK,
    PROFILE_EXP,
    OraclePlan,
    Segment,
    plan_from_workload,
    snap_frequency,
    mux_channels,
    segment_phase,
    segment_freq,
)
from .c_evaluator import build_c_oracle, c_waveform, c_codes, c_num_threads  # noqa: F401
