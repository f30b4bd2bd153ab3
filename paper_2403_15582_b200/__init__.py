"""B200-native additive waveform synthesis (the hot path of arXiv 2403.15582).

The product is the C-ABI library ``libawg_b200.so`` (``include/awg.h``; sources under ``csrc/``);
this package is its thin ctypes binding.  Importing it without the built library raises
ImportError: there is no CPU fallback.
"""
from .binding import *  # noqa: F401,F403
from .binding import (  # noqa: F401
    AwgError,
    Plan,
    Ring,
    synthesize_chunk_mux,
    EXPORTED,
    LIB_PATH,
)
