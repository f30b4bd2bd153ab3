"""Seeded generators for the five BASELINE.json configurations.

Only random draws and array layout: no phase, sine or quantiser arithmetic.
Draw order is part of the recipe; every generator
uses ``numpy.random.default_rng(seed)`` (PCG64) and draws in the order listed
in its docstring, so oracle and CUDA path see identical numbers.

Units at this level are the C-ABI's: Hz, full-scale fraction, radians, seconds.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Dict, List, Optional

import numpy as np

PROFILE_STATIC = 0
PROFILE_LINEAR = 1
PROFILE_MINJERK = 2
PROFILE_EXP = 3      # exponential chirp f(t) = f0 (f1/f0)^(tau/T), named at PAPER.md:137

#: int16 full-scale factor named by BASELINE.json config 1 ("int16 scale 0.9*32767").
DEFAULT_SCALE = 0.9 * 32767.0


@dataclasses.dataclass
class Update:
    """One per-chunk trajectory update: at the first sample of ``chunk_idx`` the
    listed tones start a new move towards ``f1`` lasting ``t_dur`` seconds."""

    chunk_idx: int
    tone_idx: np.ndarray  # int32
    f1: np.ndarray  # float64, Hz
    t_dur: np.ndarray  # float64, s
    profile: np.ndarray  # int32


@dataclasses.dataclass
class Workload:
    name: str
    sample_rate: float  # Hz (the paper writes "MB/s" for mega-samples/s, PAPER.md:10 vs 77)
    chunk_len: int  # samples per chunk (the paper's L_s)
    n_chunks: int
    f0: np.ndarray
    f1: np.ndarray
    A: np.ndarray
    phi0: np.ndarray  # radians
    t_start: np.ndarray
    t_dur: np.ndarray
    profile: np.ndarray  # int32
    scale: float = DEFAULT_SCALE
    updates: List[Update] = dataclasses.field(default_factory=list)
    seed: Optional[object] = None

    @property
    def n_tones(self) -> int:
        return int(self.f0.shape[0])

    @property
    def n_samples(self) -> int:
        return self.chunk_len * self.n_chunks

    @property
    def tone_samples(self) -> int:
        return self.n_tones * self.n_samples

    def updates_by_chunk(self) -> Dict[int, Update]:
        return {u.chunk_idx: u for u in self.updates}

    def rechunked(self, chunk_len: int) -> "Workload":
        """Same tone table, different chunking (only for workloads without updates)."""
        if self.updates:
            raise ValueError("rechunking would move the update instants")
        if self.n_samples % chunk_len:
            raise ValueError("chunk_len must divide the total length")
        return dataclasses.replace(self, chunk_len=chunk_len, n_chunks=self.n_samples // chunk_len)


def _f64(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.float64)


def _i32(x) -> np.ndarray:
    return np.ascontiguousarray(x, dtype=np.int32)


def config1() -> Workload:
    """C1 "PR1 ref", seed 0: 16 tones at 560 MS/s, 2^20 samples (one chunk).

    Draws: f0 = U(80e6,120e6,16); phi0 = U(0,2pi,16); mag = U(0.5e6,2e6,4);
    sign = choice(+-1,4).  Tones 0-11 STATIC, tones 12-15 LINEAR to f0+sign*mag
    over the full span; A = 1/16.
    """
    rng = np.random.default_rng(0)
    fs, n, N = 560e6, 1 << 20, 16
    f0 = rng.uniform(80e6, 120e6, N)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    mag = rng.uniform(0.5e6, 2e6, 4)
    sign = rng.choice(np.array([-1.0, 1.0]), 4)
    f1 = f0.copy()
    f1[12:] = f0[12:] + sign * mag
    profile = np.zeros(N, np.int32)
    profile[12:] = PROFILE_LINEAR
    t_dur = np.zeros(N)
    t_dur[12:] = n / fs
    return Workload("C1", fs, n, 1, _f64(f0), _f64(f1), _f64(np.full(N, 1.0 / N)), _f64(phi0),
                    _f64(np.zeros(N)), _f64(t_dur), _i32(profile), seed=0)


def config2() -> Workload:
    """C2, seed 1: 100 tones at 560 MS/s for 10 ms (5.6 M samples, 25 chunks of 224 000).

    Draws: phi0 = U(0,2pi,100); A = U(0.8,1.2,100)/100; moving = permutation(100)[:50];
    mag = U(0.5e6,5e6,50); sign = choice(+-1,50); t_dur = U(50e-6,500e-6,50);
    t_start = U(0, 10e-3 - t_dur).  f0 = 75 MHz + 0.5 MHz*k; movers are MINJERK.
    """
    rng = np.random.default_rng(1)
    fs, N = 560e6, 100
    chunk_len, n_chunks = 224_000, 25
    span = chunk_len * n_chunks / fs
    f0 = 75e6 + 0.5e6 * np.arange(N)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    A = rng.uniform(0.8, 1.2, N) / N
    moving = rng.permutation(N)[:50]
    mag = rng.uniform(0.5e6, 5e6, 50)
    sign = rng.choice(np.array([-1.0, 1.0]), 50)
    dur = rng.uniform(50e-6, 500e-6, 50)
    start = rng.uniform(0.0, span - dur)
    f1 = f0.copy()
    f1[moving] = f0[moving] + sign * mag
    profile = np.zeros(N, np.int32)
    profile[moving] = PROFILE_MINJERK
    t_dur = np.zeros(N)
    t_dur[moving] = dur
    t_start = np.zeros(N)
    t_start[moving] = start
    return Workload("C2", fs, chunk_len, n_chunks, _f64(f0), _f64(f1), _f64(A), _f64(phi0),
                    _f64(t_start), _f64(t_dur), _i32(profile), seed=1)


def config3(n_tones: int = 1000) -> Workload:
    """C3, seed 2: 1000 tones at 560 MS/s, all MINJERK over 35 ms ("precomputed"/Playback).

    Length follows the paper's rule L_d = L_s*ceil(T*fs/L_s) with
    L_s = 2^20: 19 chunks = 19 922 944 samples.  Draws: phi0 = U(0,2pi,N);
    f1 = f0 + U(-10e6,10e6,N).  f0 = 50 MHz + 0.1 MHz*k; A = 1/N.
    """
    rng = np.random.default_rng(2)
    fs, N = 560e6, n_tones
    chunk_len = 1 << 20
    T = 35e-3
    n_chunks = int(math.ceil(T * fs / chunk_len))
    f0 = 50e6 + 0.1e6 * np.arange(N)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    f1 = f0 + rng.uniform(-10e6, 10e6, N)
    return Workload("C3", fs, chunk_len, n_chunks, _f64(f0), _f64(f1), _f64(np.full(N, 1.0 / N)),
                    _f64(phi0), _f64(np.zeros(N)), _f64(np.full(N, T)),
                    _i32(np.full(N, PROFILE_MINJERK)), seed=2)


def config4(n_chunks: int = 382) -> Workload:
    """C4, seed 3: streaming, 194 tones at 100 MS/s, 2^18-sample chunks for 1 s (382 chunks).

    Draws: phi0 = U(0,2pi,194); then for each chunk c in order:
    idx = choice(194,19,replace=False); mag = U(0.2e6,3e6,19); sign = choice(+-1,19).
    Each listed tone starts a 100 us MINJERK move to (its current target) + sign*mag at
    the first sample of chunk c.  f0 = 60 MHz + 0.2 MHz*k; A = 1/194; all STATIC at start.
    The bookkeeping of "current target" below is list handling, not synthesis arithmetic.
    """
    rng = np.random.default_rng(3)
    fs, N = 100e6, 194
    chunk_len = 1 << 18
    n_move = 19  # round(0.1*194)
    f0 = 60e6 + 0.2e6 * np.arange(N)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    f_now = f0.copy()
    updates: List[Update] = []
    for c in range(n_chunks):
        idx = rng.choice(N, n_move, replace=False)
        mag = rng.uniform(0.2e6, 3e6, n_move)
        sign = rng.choice(np.array([-1.0, 1.0]), n_move)
        tgt = f_now[idx] + sign * mag
        f_now[idx] = tgt
        updates.append(Update(c, _i32(idx), _f64(tgt), _f64(np.full(n_move, 100e-6)),
                              _i32(np.full(n_move, PROFILE_MINJERK))))
    return Workload("C4", fs, chunk_len, n_chunks, _f64(f0), _f64(f0.copy()), _f64(np.full(N, 1.0 / N)),
                    _f64(phi0), _f64(np.zeros(N)), _f64(np.zeros(N)), _i32(np.zeros(N)),
                    updates=updates, seed=3)


C5_TONES = (20, 64, 256, 1024, 4096)
C5_CHUNKS = (1 << 16, 1 << 18, 1 << 20, 1 << 22)


def config5_cell(n_tones: int, chunk_len: int, whole_chunk_moves: bool = False) -> Workload:
    """One cell of C5, seed [4, N, log2(chunk_len)]: N tones at 560 MS/s, one chunk.

    Draws: f0 = U(20e6,250e6,N); phi0 = U(0,2pi,N); sign = choice(+-1,N-N//2);
    t_start = U(0, max(0, chunk_len/fs - 200e-6), N-N//2).  Tones < N/2 STATIC, the rest
    MINJERK to f0+-5 MHz over 200 us.  ``whole_chunk_moves`` is the supplementary worst case:
    t_start = 0 and t_dur = chunk_len/fs so every mover moves for the whole chunk.
    """
    log2c = int(round(math.log2(chunk_len)))
    if (1 << log2c) != chunk_len:
        raise ValueError("C5 chunk lengths are powers of two")
    rng = np.random.default_rng([4, n_tones, log2c])
    fs, N = 560e6, n_tones
    n_static = N // 2
    n_mov = N - n_static
    f0 = rng.uniform(20e6, 250e6, N)
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    sign = rng.choice(np.array([-1.0, 1.0]), n_mov)
    hi = max(0.0, chunk_len / fs - 200e-6)
    start = rng.uniform(0.0, hi, n_mov) if hi > 0.0 else np.zeros(n_mov)
    f1 = f0.copy()
    f1[n_static:] = f0[n_static:] + sign * 5e6
    profile = np.zeros(N, np.int32)
    profile[n_static:] = PROFILE_MINJERK
    t_dur = np.zeros(N)
    t_start = np.zeros(N)
    if whole_chunk_moves:
        t_dur[n_static:] = chunk_len / fs
    else:
        t_dur[n_static:] = 200e-6
        t_start[n_static:] = start
    name = f"C5[N={N},L=2^{log2c}{',whole' if whole_chunk_moves else ''}]"
    return Workload(name, fs, chunk_len, 1, _f64(f0), _f64(f1), _f64(np.full(N, 1.0 / N)), _f64(phi0),
                    _f64(t_start), _f64(t_dur), _i32(profile), seed=(4, N, log2c))


def config5_grid():
    """All 20 (N, chunk_len) cells of C5 as (n_tones, chunk_len) pairs."""
    return [(n, c) for n in C5_TONES for c in C5_CHUNKS]


def capacity_toneset(n_tones: int, sample_rate: float, chunk_len: int, mix: str = "half",
                     n_chunks: int = 1, seed: int = 5) -> Workload:
    """Tone set for the real-time capacity search: drawn like a C5 cell.

    ``mix``: "static" (no mover), "half" (second half MINJERK +-5 MHz over 200 us, as C5) or
    "moving" (every tone MINJERK +-5 MHz for the whole span, the worst case).
    Draws: f0 = U(0.05,0.45,N)*fs; phi0 = U(0,2pi,N); sign = choice(+-1,N); t_start = U(0,hi,N).
    """
    rng = np.random.default_rng([seed, n_tones])
    N = n_tones
    span = chunk_len * n_chunks / sample_rate
    f0 = rng.uniform(0.05, 0.45, N) * sample_rate
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    sign = rng.choice(np.array([-1.0, 1.0]), N)
    hi = max(0.0, span - 200e-6)
    start = rng.uniform(0.0, hi, N) if hi > 0.0 else np.zeros(N)
    f1 = f0.copy()
    profile = np.zeros(N, np.int32)
    t_dur = np.zeros(N)
    t_start = np.zeros(N)
    if mix == "static":
        pass
    elif mix == "half":
        h = N // 2
        f1[h:] = f0[h:] + sign[h:] * 5e6
        profile[h:] = PROFILE_MINJERK
        t_dur[h:] = min(200e-6, span)
        t_start[h:] = start[h:]
    elif mix == "moving":
        f1 = f0 + sign * 5e6
        profile[:] = PROFILE_MINJERK
        t_dur[:] = span
    else:
        raise ValueError(f"unknown mix {mix!r}")
    return Workload(f"CAP[{mix},N={N}]", sample_rate, chunk_len, n_chunks, _f64(f0), _f64(f1),
                    _f64(np.full(N, 1.0 / N)), _f64(phi0), _f64(t_start), _f64(t_dur), _i32(profile),
                    seed=(seed, N))


def fast_mover_stream(n_tones: int, sample_rate: float = 560e6, chunk_len: int = 1 << 18, n_chunks: int = 8,
                      seed: int = 6) -> Workload:
    """Every tone is inside a short minimum-jerk move ALL the time ("chirp indefinitely"): all tones start
    static; at every chunk boundary every tone starts a new move that lasts exactly one chunk (2^18 samples at 560 MS/s =
    468 us, inside the 100-500 us range of tweezer moves) to f_now +- U(0.5, 5) MHz, the sign chosen to stay inside
    [0.05, 0.45] fs.  Draws: f0 = U(0.1, 0.4, N) fs; phi0 = U(0, 2pi, N); then per chunk mag = U(0.5e6, 5e6, N),
    sign = choice(+-1, N) (flipped where the target would leave the band)."""
    rng = np.random.default_rng([seed, n_tones])
    N = n_tones
    f0 = rng.uniform(0.1, 0.4, N) * sample_rate
    phi0 = rng.uniform(0.0, 2.0 * math.pi, N)
    f_now = f0.copy()
    T = chunk_len / sample_rate
    updates: List[Update] = []
    for c in range(n_chunks):
        mag = rng.uniform(0.5e6, 5e6, N)
        sign = rng.choice(np.array([-1.0, 1.0]), N)
        tgt = f_now + sign * mag
        bad = (tgt < 0.05 * sample_rate) | (tgt > 0.45 * sample_rate)
        tgt[bad] = f_now[bad] - sign[bad] * mag[bad]
        f_now = tgt
        updates.append(Update(c, _i32(np.arange(N)), _f64(tgt), _f64(np.full(N, T)), _i32(np.full(N, PROFILE_MINJERK))))
    z = np.zeros(N)
    return Workload(f"FAST[N={N}]", sample_rate, chunk_len, n_chunks, _f64(f0), _f64(f0.copy()), _f64(np.full(N, 1.0 / N)),
                    _f64(phi0), _f64(z), _f64(z), _i32(np.zeros(N)), updates=updates, seed=(seed, N))


def comb_toneset(n_tones: int, n_samples: int, sample_rate: float = 560e6, f_first: float = 50e6,
                 spacing: float = 1e6) -> Workload:
    """The paper's static benchmark signal a*sum_j sin(2pi(f0 + j*df)t), f0 = 50 MHz, df = 1 MHz,
    zero phases (section V.A).  Deterministic, no draws."""
    N = n_tones
    f0 = f_first + spacing * np.arange(N)
    z = np.zeros(N)
    return Workload(f"COMB[N={N}]", sample_rate, n_samples, 1, _f64(f0), _f64(f0.copy()),
                    _f64(np.full(N, 1.0 / N)), _f64(z), _f64(z), _f64(z), _i32(np.zeros(N)))


def by_name(name: str) -> Workload:
    name = name.upper()
    if name == "C1":
        return config1()
    if name == "C2":
        return config2()
    if name == "C3":
        return config3()
    if name == "C4":
        return config4()
    raise KeyError(name)
