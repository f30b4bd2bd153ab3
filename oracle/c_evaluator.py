"""ORACLE -- test infrastructure.  ctypes loader for the plain-C evaluator (awg_oracle_c.c).

``build_c_oracle()`` compiles it with gcc (-O2 -fopenmp) into ``oracle/libawg_oracle.so``;
the other functions evaluate an ``OraclePlan``'s segment table with it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess
import threading

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "awg_oracle_c.c")
_LIB = os.path.join(_HERE, "libawg_oracle.so")
_lock = threading.Lock()
_lib = None


def build_c_oracle(force: bool = False) -> str:
    """gcc -O2 -fopenmp -shared; rebuilt when the source is newer than the library."""
    with _lock:
        if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
            tmp = _LIB + f".tmp{os.getpid()}"
            cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, _SRC, "-lm"]
            subprocess.run(cmd, check=True, capture_output=True)
            os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build_c_oracle())
        lib.awg_oracle_waveform.restype = ctypes.c_int
        lib.awg_oracle_waveform.argtypes = [
            ctypes.c_int32, ctypes.c_double, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64,
            ctypes.c_void_p, ctypes.c_int32]
        lib.awg_oracle_waveform_amp.restype = ctypes.c_int
        lib.awg_oracle_waveform_amp.argtypes = [
            ctypes.c_int32, ctypes.c_double, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_int64, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p, ctypes.c_void_p,
            ctypes.c_void_p, ctypes.c_int64, ctypes.c_int64, ctypes.c_void_p, ctypes.c_int32]
        lib.awg_oracle_quantise.restype = ctypes.c_int
        lib.awg_oracle_quantise.argtypes = [ctypes.c_void_p, ctypes.c_int64, ctypes.c_double, ctypes.c_void_p]
        lib.awg_oracle_num_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def c_num_threads() -> int:
    return int(_load().awg_oracle_num_threads())


def c_waveform(plan, n0: int, n1: int, n_threads: int = 0) -> np.ndarray:
    """float64 V[n0:n1] of ``plan`` (an OraclePlan) evaluated by the C oracle."""
    if np.dtype(np.longdouble).itemsize != ctypes.sizeof(ctypes.c_longdouble):
        raise RuntimeError("numpy longdouble does not match C long double on this platform")
    lib = _load()
    off, n_begin, reals, prof = plan.flat_segments()
    A = np.ascontiguousarray(plan.A, dtype=np.float64)
    V = np.empty(n1 - n0, dtype=np.float64)
    ramps = getattr(plan, "amp_ramps", None)
    if ramps is None:
        rc = lib.awg_oracle_waveform(plan.n_tones, float(plan.fs), off.ctypes.data, n_begin.ctypes.data,
                                     reals.ctypes.data, reals.shape[1], prof.ctypes.data, A.ctypes.data,
                                     n0, n1, V.ctypes.data, n_threads)
    else:
        A1, ts, T = (np.ascontiguousarray(x, dtype=np.float64) for x in ramps[:3])
        ap = np.ascontiguousarray(ramps[3], dtype=np.int32)
        rc = lib.awg_oracle_waveform_amp(plan.n_tones, float(plan.fs), off.ctypes.data, n_begin.ctypes.data,
                                         reals.ctypes.data, reals.shape[1], prof.ctypes.data, A.ctypes.data,
                                         A1.ctypes.data, ts.ctypes.data, T.ctypes.data, ap.ctypes.data,
                                         n0, n1, V.ctypes.data, n_threads)
    if rc != 0:
        raise RuntimeError("awg_oracle_waveform failed")
    return V


def c_codes(plan, n0: int, n1: int, n_threads: int = 0) -> np.ndarray:
    """int16 codes [n0, n1) via the C oracle's own quantiser."""
    lib = _load()
    V = c_waveform(plan, n0, n1, n_threads)
    out = np.empty(V.shape[0], dtype=np.int16)
    if lib.awg_oracle_quantise(V.ctypes.data, V.shape[0], float(plan.scale), out.ctypes.data) != 0:
        raise RuntimeError("awg_oracle_quantise failed")
    return out
