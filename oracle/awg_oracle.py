"""ORACLE -- test infrastructure, not product code.

A plain, slow, obviously-correct CPU implementation of the additive waveform
synthesis of arXiv 2403.15582 (Tu & Subhankar).  It is the *plain definition*
written out: one ``sin`` per (tone, sample), phases in x87 extended precision
(``numpy.longdouble``, 64-bit mantissa), sum in float64, no tiling, no
recurrences, no tables.  It shares no code with the CUDA path
(``paper_2403_15582_b200/``) and must never be imported by it; only ``tests/``,
``__graft_entry__.smoke()`` and ``bench.py``'s ``cpu_baseline`` / ``--impl
reference`` legs may use it.

What it computes (paper citations are PAPER.md:<line>):

* ``V[n] = sum_k A_k sin(2 pi frac(Phi_k[n]))``                -- Eq. 9 with the
  range reduction of Eq. 14; static tones are Eq. 8 evaluated at the
  absolute sample index ``n`` (reading G4/G13 in DESIGN.md: no ``mod L_s`` loop buffer, no
  frequency snapping on this path).
* ``Phi_k`` is the closed-form time integral of the tone's frequency trajectory, in cycles:
    - STATIC, or before the move starts (tau <= 0):   Phi = theta + f0 t            (Eq. 8)
    - LINEAR, 0 < tau < T, s = tau/T:                 Phi = theta + f0 t + D T s^2/2
      (the paper names the linear chirp without a formula; this is its integral)
    - MINJERK, 0 < tau < T:                           Phi = theta + f0 t + D T (5/2 s^4 - 3 s^5 + s^6)
      (Eq. 10 / p(i), *as corrected* -- reading G1 in DESIGN.md: the printed
      prefactor i/fs of p(i) does not integrate a minimum-jerk ramp; the prefactor must be T)
    - after the move (tau >= T, either profile):      Phi = theta + f0 t_s + f1 tau + T (f0 - f1)/2
      (Eq. 10 branch 2; with t_s = 0 it is 2 pi f_finish i/fs + pi T (f_start - f_finish) rad)
  with t = n/fs, tau = t - t_s, D = f1 - f0.
* ``code[n] = clamp(rint(scale * V[n]), -32768, 32767)`` as int16, round-half-to-even
  ("One sample is 2 bytes", PAPER.md:196 16-bit DAC; scale = 0.9*32767 from
  BASELINE.json config 1; reading G9 in DESIGN.md).
* Per-chunk updates (streaming pathway, Fig. 7): at the first sample of chunk c a
  tone starts a new move from its current instantaneous frequency and phase (reading G12).

Every function here is pinned by ``tests/test_oracle_pins.py`` against values the
paper and the mathematics fix (closed forms, FFT bins, numerical integration of
the frequency profile, 50-digit arithmetic); nothing is "parity unpinned".
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import numpy as np

LD = np.longdouble

PROFILE_STATIC = 0
PROFILE_LINEAR = 1
PROFILE_MINJERK = 2

TWO_PI_LD = LD(2) * np.arccos(LD(-1))
TWO_PI = 2.0 * np.pi


@dataclasses.dataclass
class Segment:
    """One piece of a tone's trajectory.  ``n_begin`` is the first absolute sample the
    segment applies to (None = from minus infinity: the segment given to
    ``set_trajectories``).  All reals are longdouble; theta is in cycles."""

    n_begin: Optional[int]
    t_s: LD
    T: LD
    f0: LD
    f1: LD
    profile: int
    theta: LD


def _frac(x):
    """Fractional part in [0,1): the modf of Eq. 14; floor- or trunc-based
    makes no difference to sin(2 pi x) (reading G11)."""
    return x - np.floor(x)


def segment_phase(seg: Segment, t):
    """Unwrapped phase Phi(t) in cycles of one segment at times ``t`` (longdouble array)."""
    t = np.asarray(t, dtype=LD)
    tau = t - seg.t_s
    static = seg.theta + seg.f0 * t  # Eq. 8
    if seg.profile == PROFILE_STATIC:
        return static
    D = seg.f1 - seg.f0
    after = seg.theta + seg.f0 * seg.t_s + seg.f1 * tau + seg.T * (seg.f0 - seg.f1) / LD(2)  # Eq. 10 branch 2
    if seg.T > 0:
        s = tau / seg.T
        if seg.profile == PROFILE_LINEAR:
            g = s * s / LD(2)
        elif seg.profile == PROFILE_MINJERK:
            s2 = s * s
            s4 = s2 * s2
            g = LD(5) / LD(2) * s4 - LD(3) * s4 * s + s4 * s2  # Eq. 10 p(i), prefactor T (G1)
        else:
            raise ValueError("unknown profile")
        during = seg.theta + seg.f0 * t + D * seg.T * g
    else:
        during = after
    return np.where(tau <= 0, static, np.where(tau >= seg.T, after, during))


def segment_freq(seg: Segment, t):
    """Instantaneous frequency (Hz) of one segment: STATIC f0; LINEAR f0 + D s;
    MINJERK f0 + D (10 s^3 - 15 s^4 + 6 s^5); after the move f1."""
    t = np.asarray(t, dtype=LD)
    tau = t - seg.t_s
    f0 = np.full_like(t, seg.f0)
    if seg.profile == PROFILE_STATIC:
        return f0
    D = seg.f1 - seg.f0
    if seg.T > 0:
        s = tau / seg.T
        if seg.profile == PROFILE_LINEAR:
            h = s
        elif seg.profile == PROFILE_MINJERK:
            s3 = s * s * s
            h = LD(10) * s3 - LD(15) * s3 * s + LD(6) * s3 * s * s
        else:
            raise ValueError("unknown profile")
        during = seg.f0 + D * h
    else:
        during = np.full_like(t, seg.f1)
    return np.where(tau <= 0, f0, np.where(tau >= seg.T, np.full_like(t, seg.f1), during))


class OraclePlan:
    """Mirror of the C-ABI plan (include/awg.h) for the oracle: same calls, same units
    (Hz, full-scale fraction, radians, seconds), full segment history per tone."""

    def __init__(self, n_tones: int, sample_rate: float, chunk_len: int, scale: float = 0.9 * 32767.0):
        if n_tones < 1 or not (sample_rate > 0) or chunk_len < 1:
            raise ValueError("bad plan arguments")
        self.n_tones = int(n_tones)
        self.fs = LD(sample_rate)
        self.chunk_len = int(chunk_len)
        self.scale = float(scale)
        self.A = np.zeros(n_tones)
        self.segments: List[List[Segment]] = [[] for _ in range(n_tones)]

    # ---- trajectory table -------------------------------------------------------------
    def set_trajectories(self, f0, f1, A, phi0, t_start, t_dur, profile) -> None:
        N = self.n_tones
        arrs = [np.asarray(a, dtype=np.float64) for a in (f0, f1, A, phi0, t_start, t_dur)]
        prof = np.asarray(profile, dtype=np.int64)
        if any(a.shape != (N,) for a in arrs) or prof.shape != (N,):
            raise ValueError("arrays must have length n_tones")
        f0, f1, A, phi0, t_start, t_dur = arrs
        if not all(np.all(np.isfinite(a)) for a in arrs) or np.any(t_dur < 0):
            raise ValueError("non-finite input or negative duration")
        self.A = A.copy()
        self.segments = []
        for k in range(N):
            theta = LD(phi0[k]) / TWO_PI_LD  # radians -> cycles (theta_j of Eq. 8/9)
            self.segments.append([Segment(None, LD(t_start[k]), LD(t_dur[k]), LD(f0[k]), LD(f1[k]),
                                          int(prof[k]), theta)])

    def update_trajectories(self, chunk_idx: int, tone_idx, f1, t_dur, profile) -> None:
        """At the first sample of ``chunk_idx`` each listed tone starts a new move from its
        current instantaneous frequency and phase (phase- and frequency-continuous, G12)."""
        n_u = int(chunk_idx) * self.chunk_len
        t_u = LD(n_u) / self.fs
        tone_idx = np.asarray(tone_idx, dtype=np.int64)
        if len(set(tone_idx.tolist())) != len(tone_idx):
            raise ValueError("duplicate tone in one update")
        for j, k in enumerate(tone_idx):
            segs = self.segments[int(k)]
            last = segs[-1]
            if last.n_begin is not None and n_u < last.n_begin:
                raise ValueError("updates must be applied in non-decreasing chunk order")
            f_now = segment_freq(last, np.array([t_u], dtype=LD))[0]
            phi_now = segment_phase(last, np.array([t_u], dtype=LD))[0]
            theta_new = _frac(_frac(phi_now) - _frac(f_now * t_u))
            segs.append(Segment(n_u, t_u, LD(float(t_dur[j])), f_now, LD(float(f1[j])), int(profile[j]),
                                theta_new))

    # ---- evaluation -------------------------------------------------------------------
    def _pieces(self, k: int, n0: int, n1: int):
        """Yield (segment, a, b): segment covering absolute samples [a, b) within [n0, n1)."""
        segs = self.segments[k]
        for i, seg in enumerate(segs):
            lo = n0 if seg.n_begin is None else max(n0, seg.n_begin)
            hi = n1 if i + 1 == len(segs) else min(n1, segs[i + 1].n_begin)
            if lo < hi:
                yield seg, lo, hi

    def phase(self, k: int, n) -> np.ndarray:
        """Unwrapped phase Phi_k[n] in cycles (longdouble) at absolute sample indices ``n``."""
        n = np.asarray(n, dtype=np.int64)
        out = np.empty(n.shape, dtype=LD)
        segs = self.segments[k]
        begins = np.array([-(1 << 62) if s.n_begin is None else s.n_begin for s in segs], dtype=np.int64)
        which = np.searchsorted(begins, n, side="right") - 1
        for i, seg in enumerate(segs):
            m = which == i
            if np.any(m):
                out[m] = segment_phase(seg, n[m].astype(LD) / self.fs)
        return out

    def inst_freq(self, k: int, n) -> np.ndarray:
        n = np.asarray(n, dtype=np.int64)
        out = np.empty(n.shape, dtype=LD)
        segs = self.segments[k]
        begins = np.array([-(1 << 62) if s.n_begin is None else s.n_begin for s in segs], dtype=np.int64)
        which = np.searchsorted(begins, n, side="right") - 1
        for i, seg in enumerate(segs):
            m = which == i
            if np.any(m):
                out[m] = segment_freq(seg, n[m].astype(LD) / self.fs)
        return out

    def waveform(self, n0: int, n1: int, tones: Optional[Sequence[int]] = None) -> np.ndarray:
        """V[n0:n1] in float64: sum over tones of A_k sin(2 pi frac(Phi_k[n]))  (Eq. 9 + Eq. 14)."""
        V = np.zeros(n1 - n0, dtype=np.float64)
        ks = range(self.n_tones) if tones is None else tones
        for k in ks:
            for seg, a, b in self._pieces(k, n0, n1):
                t = np.arange(a, b, dtype=np.int64).astype(LD) / self.fs
                turns = _frac(segment_phase(seg, t)).astype(np.float64)
                V[a - n0:b - n0] += self.A[k] * np.sin(TWO_PI * turns)
        return V

    def quantise(self, V: np.ndarray) -> np.ndarray:
        """int16 DAC codes: rint (half-to-even) of scale*V, saturated (G9)."""
        q = np.rint(self.scale * np.asarray(V, dtype=np.float64))
        return np.clip(q, -32768.0, 32767.0).astype(np.int16)

    def codes(self, n0: int, n1: int) -> np.ndarray:
        return self.quantise(self.waveform(n0, n1))

    def chunk(self, chunk_idx: int) -> np.ndarray:
        """int16 codes of chunk ``chunk_idx``: samples [c*chunk_len, (c+1)*chunk_len)."""
        return self.codes(chunk_idx * self.chunk_len, (chunk_idx + 1) * self.chunk_len)

    def chunk_f64(self, chunk_idx: int) -> np.ndarray:
        return self.waveform(chunk_idx * self.chunk_len, (chunk_idx + 1) * self.chunk_len)

    # ---- flat segment table (for the C evaluator in awg_oracle_c.c) ------------------------
    def flat_segments(self):
        off = np.zeros(self.n_tones + 1, dtype=np.int64)
        rows = []
        for k, segs in enumerate(self.segments):
            off[k + 1] = off[k] + len(segs)
            rows.extend(segs)
        S = len(rows)
        n_begin = np.array([-(1 << 62) if s.n_begin is None else s.n_begin for s in rows], dtype=np.int64)
        reals = np.empty((5, S), dtype=LD)  # t_s, T, f0, f1, theta
        for i, s in enumerate(rows):
            reals[:, i] = (s.t_s, s.T, s.f0, s.f1, s.theta)
        prof = np.array([s.profile for s in rows], dtype=np.int32)
        return off, n_begin, np.ascontiguousarray(reals), prof


def plan_from_workload(w, apply_updates_upto: Optional[int] = None) -> OraclePlan:
    """Build an OraclePlan from an ``awg_workloads.Workload`` (all updates applied unless
    ``apply_updates_upto`` limits them to chunks < that index; the oracle keeps full history so
    applying every update up front does not change earlier chunks)."""
    p = OraclePlan(w.n_tones, w.sample_rate, w.chunk_len, w.scale)
    p.set_trajectories(w.f0, w.f1, w.A, w.phi0, w.t_start, w.t_dur, w.profile)
    for u in w.updates:
        if apply_updates_upto is not None and u.chunk_idx >= apply_updates_upto:
            break
        p.update_trajectories(u.chunk_idx, u.tone_idx, u.f1, u.t_dur, u.profile)
    return p
