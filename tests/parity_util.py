"""Helpers for the GPU parity tests: acceptance bar and oracle windows.

The bar is BASELINE.json north_star's: int16 codes within +-1 LSB of the oracle on >= 99.99 % of
samples with a maximum of 2 LSB; pre-quantisation fp32 sum within 1e-5 of full scale.
"""
from __future__ import annotations

import numpy as np

import oracle

LSB_OK_FRACTION = 0.9999
LSB_MAX = 2
F32_TOL = 1e-5


def assert_codes_close(got: np.ndarray, want: np.ndarray, what: str = ""):
    got = np.asarray(got).astype(np.int32)
    want = np.asarray(want).astype(np.int32)
    assert got.shape == want.shape, f"{what}: shape {got.shape} vs {want.shape}"
    d = np.abs(got - want)
    frac_ok = float(np.mean(d <= 1)) if d.size else 1.0
    dmax = int(d.max()) if d.size else 0
    assert dmax <= LSB_MAX, f"{what}: max |diff| = {dmax} LSB at {int(np.argmax(d))}"
    assert frac_ok >= LSB_OK_FRACTION, f"{what}: only {frac_ok:.6f} of samples within 1 LSB"
    return float(np.mean(d == 0)), dmax


def assert_f32_close(got: np.ndarray, want: np.ndarray, what: str = "", tol: float = F32_TOL):
    got = np.asarray(got, dtype=np.float64)
    err = np.abs(got - np.asarray(want, dtype=np.float64))
    emax = float(err.max()) if err.size else 0.0
    assert emax <= tol, f"{what}: max |V_gpu - V_oracle| = {emax:.3e} > {tol:g} at {int(np.argmax(err))}"
    return emax


def oracle_windows(oplan, windows):
    """[(a, b)] -> list of (float64 V, int16 codes) computed by the C oracle."""
    out = []
    for a, b in windows:
        V = oracle.c_waveform(oplan, a, b)
        out.append((V, oplan.quantise(V)))
    return out


def sample_windows(n_samples: int, width: int, count: int, seed: int, must=()):
    """`count` random windows of `width` samples plus the first, the last and windows centred on
    the sample indices in `must` (clipped, aligned to 8)."""
    rng = np.random.default_rng(seed)
    width = min(width, n_samples)
    starts = [0, n_samples - width]
    starts += [int(x) for x in rng.integers(0, max(1, n_samples - width), count)]
    starts += [int(m) - width // 2 for m in must]
    wins = []
    for s in starts:
        s = max(0, min(n_samples - width, s))
        s -= s % 8
        wins.append((s, s + width))
    return sorted(set(wins))
