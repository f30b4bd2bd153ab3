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

* Exponential chirp (PAPER.md:137 names "linear, exponential" frequency chirps and prints no formula; DESIGN.md
  reading G20): f(tau) = f0 (f1/f0)^(tau/T), phase = its integral, f0 T ((f1/f0)^s - 1)/ln(f1/f0) cycles since the
  start of the move; f0 and f1 of the same sign.  Pinned in tests/test_oracle_pins_next.py.
* Four-channel multiplexed output (the paper's WM kernel, Fig. 4): the codes of the
  channels' independent tone sets interleaved "in groups of four", ``out[4 i + c] = code_c[i]``
  (``mux_channels``).
* Static-buffer pathway (section IV A/B): Eq. 6 frequency snapping (``snap_frequency``);
  the looped buffer ``X_static[i mod L_s]`` of Eq. 7-8 (``static_buffer``); Eq. 9 with
  only the other tones evaluated per sample (``waveform_static_pathway``); and the hand-back
  of Eq. 10 branch 3: after ``L_d`` a moved tone is a looped static wavetable at its
  final frequency with the phase offset theta' (``handback_theta``, ``fold_into_static_buffer``).
* Time-varying amplitude ``a_j[i]`` (Eq. 9; constant in the paper's worked case):
  per tone ``a(t) = A0`` before ``t_a``, ``A0 + (A1 - A0) h((t - t_a)/T_a)`` during the ramp and ``A1`` after,
  with ``h(s) = s`` (LINEAR) or the minimum-jerk ramp ``10 s^3 - 15 s^4 + 6 s^5`` (MINJERK) -- reading G7 in
  DESIGN.md: the paper allows ``a_j[i]`` without giving a profile; the frequency ramp's profile is reused
  (``set_amplitude_ramps``).

Every function here is pinned by ``tests/test_oracle_pins.py`` / ``tests/test_oracle_pins_next.py`` against
values the paper and the mathematics fix (closed forms, FFT bins, numerical integration of the frequency
profile, 50-digit arithmetic); nothing is "parity unpinned".
"""
from __future__ import annotations

import dataclasses
from typing import List, Optional, Sequence

import numpy as np

LD = np.longdouble

PROFILE_STATIC = 0
PROFILE_LINEAR = 1
PROFILE_MINJERK = 2
PROFILE_EXP = 3

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
    if seg.profile == PROFILE_EXP:
        # Exponential chirp (named, without a formula, at PAPER.md:137; reading G20): the frequency runs
        # geometrically, f(tau) = f0 r^(tau/T) with r = f1/f0 > 0, so the phase gained since the start of the move is
        # the integral f0 T (r^s - 1)/ln r, and T (f1 - f0)/ln r over the whole move.
        if D == 0 or not seg.T > 0:
            r_gain_total = seg.f0 * seg.T
        else:
            Lr = np.log(seg.f1 / seg.f0)
            r_gain_total = seg.T * D / Lr
        after = seg.theta + seg.f0 * seg.t_s + r_gain_total + seg.f1 * (tau - seg.T)
        if seg.T > 0 and D != 0:
            s = np.clip(tau / seg.T, LD(0), LD(1))
            during = seg.theta + seg.f0 * seg.t_s + seg.f0 * seg.T * np.expm1(Lr * s) / Lr
        elif seg.T > 0:
            during = static
        else:
            during = after
        return np.where(tau <= 0, static, np.where(tau >= seg.T, after, during))
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
    MINJERK f0 + D (10 s^3 - 15 s^4 + 6 s^5); EXP f0 (f1/f0)^s; after the move f1."""
    t = np.asarray(t, dtype=LD)
    tau = t - seg.t_s
    f0 = np.full_like(t, seg.f0)
    if seg.profile == PROFILE_STATIC:
        return f0
    D = seg.f1 - seg.f0
    if seg.profile == PROFILE_EXP:
        if seg.T > 0 and D != 0:
            s = np.clip(tau / seg.T, LD(0), LD(1))
            during = seg.f0 * np.exp(np.log(seg.f1 / seg.f0) * s)
        else:
            during = np.full_like(t, seg.f1 if not seg.T > 0 else seg.f0)
        return np.where(tau <= 0, f0, np.where(tau >= seg.T, np.full_like(t, seg.f1), during))
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
        self.amp_ramps = None  # (A1, t_a, T_a, profile) arrays once set_amplitude_ramps has been called

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
        self.amp_ramps = None
        self.segments = []
        for k in range(N):
            theta = LD(phi0[k]) / TWO_PI_LD  # radians -> cycles (theta_j of Eq. 8/9)
            self.segments.append([Segment(None, LD(t_start[k]), LD(t_dur[k]), LD(f0[k]), LD(f1[k]),
                                          int(prof[k]), theta)])

    def set_amplitude_ramps(self, A1, t_start, t_dur, profile) -> None:
        """Time-varying amplitude a_j[i] of Eq. 9: tone k goes from the amplitude given to
        ``set_trajectories`` to ``A1[k]`` over ``[t_start[k], t_start[k] + t_dur[k]]`` along ``profile[k]``
        (STATIC = constant amplitude, LINEAR, or MINJERK = 10 s^3 - 15 s^4 + 6 s^5; reading G7)."""
        N = self.n_tones
        A1, ts, T = (np.asarray(a, dtype=np.float64) for a in (A1, t_start, t_dur))
        prof = np.asarray(profile, dtype=np.int64)
        if A1.shape != (N,) or ts.shape != (N,) or T.shape != (N,) or prof.shape != (N,):
            raise ValueError("arrays must have length n_tones")
        if not (np.all(np.isfinite(A1)) and np.all(np.isfinite(ts)) and np.all(np.isfinite(T))) or np.any(T < 0):
            raise ValueError("non-finite input or negative duration")
        if np.any((prof < PROFILE_STATIC) | (prof > PROFILE_MINJERK)):
            raise ValueError("unknown profile")
        self.amp_ramps = (A1.copy(), ts.copy(), T.copy(), prof.copy())

    def amplitude(self, k: int, n) -> np.ndarray:
        """a_k at absolute sample indices ``n`` (float64)."""
        n = np.asarray(n, dtype=np.int64)
        A0 = float(self.A[k])
        if self.amp_ramps is None or int(self.amp_ramps[3][k]) == PROFILE_STATIC:
            return np.full(n.shape, A0)
        A1, ts, T, prof = (x[k] for x in self.amp_ramps)
        t = n.astype(LD) / self.fs
        tau = t - LD(ts)
        if T > 0:
            sfrac = np.clip((tau / LD(T)).astype(np.float64), 0.0, 1.0)
        else:
            sfrac = (tau >= 0).astype(np.float64)
        if int(prof) == PROFILE_LINEAR:
            h = sfrac
        else:
            h = sfrac ** 3 * (10.0 + sfrac * (6.0 * sfrac - 15.0))
        return A0 + (float(A1) - A0) * h

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
                if self.amp_ramps is None:
                    V[a - n0:b - n0] += self.A[k] * np.sin(TWO_PI * turns)
                else:
                    V[a - n0:b - n0] += self.amplitude(k, np.arange(a, b, dtype=np.int64)) * np.sin(TWO_PI * turns)
        return V

    # ---- static-buffer pathway (section IV A/B) ----------------------------------------------
    def static_buffer(self, tones: Sequence[int], L_s: Optional[int] = None) -> np.ndarray:
        """X_static[i], i in [0, L_s): sum over the listed tones of a_j sin(2 pi f_j/fs i + theta_j), Eq. 7-8
        (PAPER.md:102-105).  The tones must be STATIC first segments; L_s defaults to chunk_len."""
        L = self.chunk_len if L_s is None else int(L_s)
        X = np.zeros(L, dtype=np.float64)
        i = np.arange(L, dtype=np.int64).astype(LD)
        for k in tones:
            seg = self.segments[int(k)][0]
            if seg.profile != PROFILE_STATIC or len(self.segments[int(k)]) != 1:
                raise ValueError("the static buffer holds static tones only")
            turns = _frac(seg.theta + seg.f0 / self.fs * i).astype(np.float64)
            X += self.A[int(k)] * np.sin(TWO_PI * turns)
        return X

    def waveform_static_pathway(self, n0: int, n1: int, X_static: np.ndarray, dynamic_tones: Sequence[int]) -> np.ndarray:
        """V[i] = X_static[i mod L_s] + sum over the dynamic tones of a_j[i] sin(phi_j[i] + theta_j), Eq. 9."""
        L = X_static.shape[0]
        idx = np.arange(n0, n1, dtype=np.int64) % L
        return X_static[idx] + self.waveform(n0, n1, tones=list(dynamic_tones))

    def handback_theta(self, k: int, L_d: int) -> LD:
        """theta'_j of Eq. 10 in cycles, reduced mod 1: the phase of tone k at sample L_d, which
        becomes the phase offset of its looped static wavetable for i > L_d (Eq. 10 branch 3)."""
        return _frac(self.phase(k, np.array([L_d], dtype=np.int64))[0])

    def fold_into_static_buffer(self, X_static: np.ndarray, tones: Sequence[int], L_d: int) -> np.ndarray:
        """Eq. 10 branch 3: after L_d each listed tone is a static wavetable at its final frequency,
        a_j sin(2 pi f_finish/fs (i mod L_s) + theta'_j), added to the looped buffer.  L_d must be a multiple of L_s
         and the tone's move must have ended by L_d."""
        L = X_static.shape[0]
        if L_d % L:
            raise ValueError("L_d must be a positive integer multiple of L_s (PAPER.md:135)")
        X = X_static.copy()
        i = np.arange(L, dtype=np.int64).astype(LD)
        t_d = LD(L_d) / self.fs
        for k in tones:
            seg = self.segments[int(k)][-1]
            if seg.profile != PROFILE_STATIC and not (t_d - seg.t_s >= seg.T):
                raise ValueError("the tone is still moving at L_d")
            f_fin = seg.f0 if seg.profile == PROFILE_STATIC else seg.f1
            turns = _frac(self.handback_theta(int(k), L_d) + f_fin / self.fs * i).astype(np.float64)
            X += float(self.amplitude(int(k), np.array([L_d]))[0]) * np.sin(TWO_PI * turns)
        return X

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


def snap_frequency(f0: float, sample_rate: float, L_s: int) -> float:
    """Eq. 6: f_j = nint(f0 L_s / fs) fs / L_s, the closest frequency with a whole number of
    cycles in L_s samples (error below fs / (2 L_s); the paper quotes the grid spacing, "less than 534 Hz")."""
    j = np.rint(LD(f0) * LD(L_s) / LD(sample_rate))
    return float(j * LD(sample_rate) / LD(L_s))


def mux_channels(plans: Sequence["OraclePlan"], n0: int, n1: int) -> np.ndarray:
    """The paper's Wavetable Multiplexer (Fig. 4; chunk layout PAPER.md:77): the int16 codes of the
    channels' waveforms "read sequentially in groups of four": out[C i + c] = code_c[n0 + i] for C channels."""
    C = len(plans)
    out = np.empty((n1 - n0) * C, dtype=np.int16)
    for c, p in enumerate(plans):
        out[c::C] = p.codes(n0, n1)
    return out


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
