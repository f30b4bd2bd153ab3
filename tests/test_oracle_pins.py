"""Pins for the oracle (CPU only): every part of oracle/ is checked against something other
than itself -- closed forms, FFT bins, the boundary-value definition of the minimum-jerk ramp,
numerical integration of the frequency profile, 50-digit arithmetic, the paper's printed
expressions (Eq. 10 branch 2, theta', the L_d rule, the 534 Hz grid).  Citations are
PAPER.md:<line>.  A plausible mistake in the oracle (dropped term, wrong sign or index,
cycles/radians mix-up, printed-but-wrong Eq. 10 branch 1) fails at least one of these.
"""
import math
import os

import mpmath
import numpy as np
import pytest

import awg_workloads as W
import oracle
from oracle import LD, OraclePlan, PROFILE_LINEAR, PROFILE_MINJERK, PROFILE_STATIC

FS = 560e6
GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def one_tone(f0, f1=None, A=1.0, phi0=0.0, t_start=0.0, t_dur=0.0, profile=PROFILE_STATIC, fs=FS,
             chunk_len=1024, scale=0.9 * 32767.0):
    p = OraclePlan(1, fs, chunk_len, scale)
    p.set_trajectories([f0], [f0 if f1 is None else f1], [A], [phi0], [t_start], [t_dur], [profile])
    return p


# ------------------------------------------------------------------ static tones: closed forms
def test_static_quarter_rate_sequence():
    # f = fs/4, phi0 = 0, A = 1  ->  0, 1, 0, -1, ...   (Eq. 8)
    V = one_tone(FS / 4).waveform(0, 64)
    assert np.allclose(V, np.tile([0.0, 1.0, 0.0, -1.0], 16), atol=1e-12)


def test_static_eighth_rate_sequence():
    r = math.sqrt(0.5)
    V = one_tone(FS / 8, A=0.5).waveform(0, 32)
    assert np.allclose(V, 0.5 * np.tile([0, r, 1, r, 0, -r, -1, -r], 4), atol=1e-12)


def test_static_dc_with_quarter_turn_phase():
    # f = 0, phi0 = pi/2 -> constant A: phi0 is in radians and adds inside the sine (G8)
    V = one_tone(0.0, A=0.37, phi0=math.pi / 2).waveform(0, 16)
    assert np.allclose(V, 0.37, atol=1e-15)


def test_phase_offset_is_radians_and_sine_convention():
    # V[0] = A sin(phi0)
    for phi0 in (0.3, 1.0, 2.5, 6.0):
        assert one_tone(123e6, A=0.8, phi0=phi0).waveform(0, 1)[0] == pytest.approx(0.8 * math.sin(phi0), abs=1e-15)


def test_on_grid_tone_is_a_single_fft_bin():
    # f_j = j fs/L_s holds exactly j cycles in L_s samples (Eq. 5)
    L, j, A = 4096, 357, 0.7
    V = one_tone(j * FS / L, A=A, phi0=1.0).waveform(0, L)
    F = np.abs(np.fft.rfft(V))
    assert F[j] == pytest.approx(A * L / 2, rel=1e-12)
    F[j] = 0.0
    assert F.max() < 1e-9 * L
    # periodic: the next L samples repeat the buffer (this is why the paper's static buffer can loop)
    assert np.allclose(one_tone(j * FS / L, A=A, phi0=1.0).waveform(L, 2 * L), V, atol=1e-11)


def test_frequency_grid_is_534_hz():
    # "the error in this approximation is less than 534 Hz" at 560 MS/s, L_s = 2^20 (Eq. 6)
    assert FS / (1 << 20) == pytest.approx(534.06, abs=0.01)


def test_comb_matches_dirichlet_closed_form():
    # the paper's static benchmark signal a sum_j sin(2pi(f0 + j df)t), f0 = 50 MHz, df = 1 MHz
    N, n = 32, 4096
    w = W.comb_toneset(N, n)
    V = oracle.plan_from_workload(w).waveform(0, n)
    t = np.arange(n) / FS
    f_first, df = 50e6, 1e6
    num = np.sin(math.pi * N * df * t)
    den = np.sin(math.pi * df * t)
    with np.errstate(invalid="ignore", divide="ignore"):
        ratio = np.where(np.abs(den) > 1e-300, num / den, float(N))
    closed = np.sin(2 * math.pi * (f_first + (N - 1) * df / 2) * t) * ratio / N
    assert np.allclose(V, closed, atol=2e-10)


def test_coherent_sum_and_zero_phase():
    N = 16
    f = np.linspace(80e6, 120e6, N)
    A = np.linspace(0.01, 0.05, N)
    z = np.zeros(N)
    p = OraclePlan(N, FS, 1024)
    p.set_trajectories(f, f, A, np.full(N, math.pi / 2), z, z, z.astype(int))
    assert p.waveform(0, 1)[0] == pytest.approx(A.sum(), abs=1e-15)  # V[0] = sum A_k
    p.set_trajectories(f, f, A, z, z, z, z.astype(int))
    assert p.waveform(0, 1)[0] == 0.0  # sin convention: zero phases give exactly 0 at n = 0


def test_zero_amplitude_gives_zero_codes():
    w = W.config1()
    p = OraclePlan(w.n_tones, w.sample_rate, 4096)
    p.set_trajectories(w.f0, w.f1, np.zeros(w.n_tones), w.phi0, w.t_start, w.t_dur, w.profile)
    c = p.codes(0, 4096)
    assert c.dtype == np.int16 and not c.any()
    assert oracle.c_codes(p, 0, 4096).any() == False  # noqa: E712
    assert p.quantise(np.array([-0.0]))[0] == 0


# ------------------------------------------------------------------ quantiser (G9)
def test_quantiser_pins():
    p = one_tone(0.0, A=1.0, phi0=math.pi / 2)
    assert p.codes(0, 1)[0] == 29490  # rint(0.9*32767 = 29490.3)
    assert p.quantise(np.array([0.0]))[0] == 0
    q = p.quantise(np.array([2.0, -2.0, 1.2, -1.2]))
    assert q.tolist() == [32767, -32768, 32767, -32768]  # saturation, asymmetric int16 range
    # round half to even at exact ties
    p2 = OraclePlan(1, FS, 8, scale=1.0)
    assert p2.quantise(np.array([0.5, 1.5, 2.5, -0.5, -1.5])).tolist() == [0, 2, 2, 0, -2]
    v = np.linspace(-1.3, 1.3, 20001)
    assert np.all(np.diff(p.quantise(v).astype(np.int32)) >= 0)  # monotone
    # C quantiser identical
    import ctypes
    out = np.empty(v.shape[0], np.int16)
    from oracle.c_evaluator import _load
    assert _load().awg_oracle_quantise(v.ctypes.data, v.shape[0], ctypes.c_double(p.scale), out.ctypes.data) == 0
    assert np.array_equal(out, p.quantise(v))


# ------------------------------------------------------------------ chirps
F0, F1 = 100e6, 103e6
NS, NT = 2800, 11200  # move starts at sample 2800 (5 us) and lasts 11200 samples (20 us) at 560 MS/s
TS, TD = NS / FS, NT / FS


def _central_freq(p, n):
    ph = p.phase(0, np.array([n - 1, n + 1]))
    return float((ph[1] - ph[0]) * LD(FS) / LD(2))


def test_linear_chirp_slope_endpoints_and_total_phase():
    p = one_tone(F0, F1, phi0=0.7, t_start=TS, t_dur=TD, profile=PROFILE_LINEAR)
    n = np.arange(NS + 1, NS + NT - 1)
    ph = p.phase(0, np.arange(NS, NS + NT))
    d2 = (ph[2:] - 2 * ph[1:-1] + ph[:-2]).astype(np.float64)
    # quadratic phase: constant second difference = chirp rate / fs^2 = (D/T)/fs^2 cycles
    assert np.allclose(d2, (F1 - F0) / TD / FS ** 2, rtol=0, atol=1e-13)
    assert _central_freq(p, NS - 5) == pytest.approx(F0, abs=1e-3)
    assert _central_freq(p, NS + NT + 5) == pytest.approx(F1, abs=1e-3)
    assert _central_freq(p, NS + NT // 2) == pytest.approx((F0 + F1) / 2, abs=1e-3)
    ph = p.phase(0, np.array([NS, NS + NT]))
    assert float(ph[1] - ph[0]) == pytest.approx(TD * (F0 + F1) / 2, abs=1e-9)  # mean frequency (f0+f1)/2
    assert len(n) > 0


def _minjerk_from_boundary_conditions():
    """The minimum-jerk ramp is THE quintic h(s) with h(0)=0, h(1)=1, h'=h''=0 at both ends
    (PAPER.md:137 'minimum jerk trajectory', ref [53]).  Solve for it instead of retyping it."""
    rows, rhs = [], []
    for s, val in ((0.0, 0.0), (1.0, 1.0)):
        rows.append([s ** k for k in range(6)]); rhs.append(val)
        rows.append([k * s ** (k - 1) if k >= 1 else 0.0 for k in range(6)]); rhs.append(0.0)
        rows.append([k * (k - 1) * s ** (k - 2) if k >= 2 else 0.0 for k in range(6)]); rhs.append(0.0)
    c = np.linalg.solve(np.array(rows), np.array(rhs))  # ascending powers
    return np.polynomial.Polynomial(c)


def test_minjerk_boundary_value_solution_is_10_15_6():
    h = _minjerk_from_boundary_conditions()
    assert np.allclose(h.coef, [0, 0, 0, 10, -15, 6], atol=1e-9)


def test_minjerk_phase_is_integral_of_boundary_value_quintic():
    # G1: phase = closed-form time integral of the min-jerk frequency ramp (not the printed Eq. 10 branch 1)
    h = _minjerk_from_boundary_conditions()
    g = h.integ()  # g(s) = int_0^s h
    theta = 0.7 / (2 * math.pi)
    p = one_tone(F0, F1, phi0=0.7, t_start=TS, t_dur=TD, profile=PROFILE_MINJERK)
    n = np.arange(NS, NS + NT + 1, 37)
    s = (n - NS) / NT
    want = theta + F0 * (n / FS) + (F1 - F0) * TD * g(s)
    got = p.phase(0, n).astype(np.float64)
    assert np.abs(got - want).max() < 1e-9


def test_minjerk_endpoints_and_derivatives():
    p = one_tone(F0, F1, phi0=0.0, t_start=TS, t_dur=TD, profile=PROFILE_MINJERK)
    D = F1 - F0
    # instantaneous frequency from the oracle's own phase (central differences)
    assert _central_freq(p, NS - 3) == pytest.approx(F0, abs=1e-3)
    assert _central_freq(p, NS + NT + 3) == pytest.approx(F1, abs=1e-3)
    assert _central_freq(p, NS + NT // 2) == pytest.approx((F0 + F1) / 2, abs=1e-2)
    # zero first and second derivative of f at both ends: f - f0 = O(s^3) with coefficient 10
    for eps in (1e-2, 3e-2):
        k = int(round(eps * NT))
        e = k / NT
        f_a = _central_freq(p, NS + k)
        f_b = _central_freq(p, NS + NT - k)
        assert abs(f_a - F0) <= 10.5 * abs(D) * e ** 3 and abs(f_a - F0) >= 9.0 * abs(D) * e ** 3
        assert abs(f_b - F1) <= 10.5 * abs(D) * e ** 3 and abs(f_b - F1) >= 9.0 * abs(D) * e ** 3
    # inst_freq() agrees with d(phase)/dt and is symmetric: h(s) + h(1-s) = 1
    for k in (100, 3000, 5600, 9000):
        assert float(p.inst_freq(0, [NS + k])[0]) == pytest.approx(_central_freq(p, NS + k), abs=0.5)
        a = float(p.inst_freq(0, [NS + k])[0]) - F0
        b = float(p.inst_freq(0, [NS + NT - k])[0]) - F0
        assert a + b == pytest.approx(D, rel=1e-12)
    # Phi(T/2) - theta - f0 (t_s + T/2) = 5 D T/64 ; Phi(T) - Phi(0) = T (f0+f1)/2
    ph = p.phase(0, np.array([NS, NS + NT // 2, NS + NT])).astype(np.float64)
    assert ph[1] - F0 * (TS + TD / 2) == pytest.approx(5 * D * TD / 64, abs=1e-9)
    assert ph[2] - ph[0] == pytest.approx(TD * (F0 + F1) / 2, abs=1e-9)


def test_printed_eq10_branch1_is_not_what_we_compute():
    # Eq. 10 branch 1 as printed: phi = (2 pi i/fs)(f_start + p(i)).  Its slope at the
    # end of the move is f_start + 1.5 D, not f_finish -- so it cannot be the integral of a ramp that ends
    # at f_finish.  The oracle must differ from it mid-move (reading G1).
    D = F1 - F0

    def printed_cycles(i):
        s = i / NT
        return (i / FS) * (F0 + D * (2.5 * s ** 4 - 3 * s ** 5 + s ** 6))

    slope_end = (printed_cycles(NT) - printed_cycles(NT - 1e-3)) / 1e-3 * FS
    assert slope_end == pytest.approx(F0 + 1.5 * D, rel=1e-4)
    p = one_tone(F0, F1, t_start=0.0, t_dur=TD, profile=PROFILE_MINJERK)
    mid = float(p.phase(0, [NT // 2])[0])
    assert abs(mid - printed_cycles(NT // 2)) > 1.0  # > 1 cycle apart at mid-move
    # both agree at the end point (the printed phase at T matches branch 2, reading P3)
    assert float(p.phase(0, [NT])[0]) == pytest.approx(printed_cycles(NT), abs=1e-8)


@pytest.mark.parametrize("profile", [PROFILE_LINEAR, PROFILE_MINJERK])
def test_after_move_is_eq10_branch2_and_theta_prime(profile):
    # t_s = 0, theta = 0:  phi = 2 pi f_finish i/fs + pi T (f_start - f_finish) rad   (Eq. 10 branch 2)
    p = one_tone(F0, F1, t_start=0.0, t_dur=TD, profile=profile, chunk_len=1 << 14)
    for i in (NT, NT + 1, NT + 1000, 3 * NT):
        want_rad = mpmath.mpf(2) * mpmath.pi * mpmath.mpf(F1) / mpmath.mpf(FS) * i + mpmath.pi * mpmath.mpf(TD) * (mpmath.mpf(F0) - mpmath.mpf(F1))
        got = mpmath.mpf(float(p.phase(0, [i])[0])) * 2 * mpmath.pi
        assert abs(got - want_rad) < 1e-7
    # continuity across the end of the move
    a, b = p.phase(0, [NT - 1, NT + 1]).astype(np.float64)
    f_mid = (b - a) * FS / 2
    assert f_mid == pytest.approx(F1, abs=200.0 if profile == PROFILE_LINEAR else 1e-2)
    # theta'_j = 2 pi f_finish L_d/fs + pi T (f_start - f_finish) is the branch-2 phase at i = L_d
    L_s = 1 << 14
    L_d = L_s * math.ceil(TD * FS / L_s)
    theta_prime = 2 * math.pi * F1 / FS * L_d + math.pi * TD * (F0 - F1)
    assert float(p.phase(0, [L_d])[0]) * 2 * math.pi == pytest.approx(theta_prime, abs=1e-6)


def test_playback_length_rule():
    # L_d = L_s ceil(T fs / L_s): 35 ms at 560 MS/s with L_s = 2^20 -> 19 chunks
    w = W.config3(4)
    assert w.n_chunks == 19 and w.n_samples == 19 * (1 << 20) == 19_922_944


@pytest.mark.parametrize("profile", [PROFILE_LINEAR, PROFILE_MINJERK])
def test_zero_span_move_equals_static_bit_for_bit(profile):
    a = one_tone(F0, F0, phi0=1.1, t_start=TS, t_dur=TD, profile=profile)
    b = one_tone(F0, phi0=1.1)
    n1 = NS + NT + 500
    # before and during the move the D = 0 terms vanish exactly: bit-for-bit
    assert np.array_equal(a.waveform(0, NS + NT), b.waveform(0, NS + NT))
    # after it, theta + f0 t_s + f1 tau is the same number up to long-double rounding only
    assert np.abs(a.waveform(0, n1) - b.waveform(0, n1)).max() < 1e-12
    assert np.array_equal(a.codes(0, n1), b.codes(0, n1))


def test_instant_retune_T0():
    p = one_tone(F0, F1, t_start=TS, t_dur=0.0, profile=PROFILE_MINJERK)
    assert _central_freq(p, NS - 2) == pytest.approx(F0, abs=1e-3)
    assert _central_freq(p, NS + 2) == pytest.approx(F1, abs=1e-3)
    a, b = p.phase(0, [NS, NS + 1]).astype(np.float64)
    assert a == pytest.approx(F0 * TS, abs=1e-9) and b - a == pytest.approx(F1 / FS, abs=1e-12)


def test_brute_force_numerical_integration_of_frequency_profile():
    # <= 3 tones, 64 samples: integrate f(t) (before: f0, during: boundary-value quintic or linear ramp, after: f1)
    # with the trapezoid rule on a 10^6-point grid instead of using any closed form.
    h_mj = _minjerk_from_boundary_conditions()
    specs = [(90e6, 95e6, 3e-6, 10e-6, PROFILE_MINJERK, 0.3), (110e6, 108e6, 1e-6, 25e-6, PROFILE_LINEAR, 1.9),
             (120e6, 120e6, 0.0, 0.0, PROFILE_STATIC, 4.0)]
    p = OraclePlan(3, FS, 1024)
    p.set_trajectories(*[np.array(x) for x in zip(*[(a, b, 1 / 3, ph, ts, td) for a, b, ts, td, _, ph in specs])],
                       [s[4] for s in specs])
    t_end = 40e-6
    grid = np.linspace(0.0, t_end, 1_000_001)
    n = np.unique(np.random.default_rng(7).integers(0, int(t_end * FS), 64))
    for k, (f0, f1, ts, td, prof, ph0) in enumerate(specs):
        if prof == PROFILE_STATIC:
            f = np.full_like(grid, f0)
        else:
            s = np.clip((grid - ts) / td, 0.0, 1.0)
            f = f0 + (f1 - f0) * (h_mj(s) if prof == PROFILE_MINJERK else s)
        cum = np.concatenate([[0.0], np.cumsum((f[1:] + f[:-1]) * 0.5 * np.diff(grid))])
        want = ph0 / (2 * math.pi) + np.interp(n / FS, grid, cum)
        got = p.phase(k, n).astype(np.float64)
        assert np.abs(got - want).max() < 1e-7


def test_chirp_endpoints_show_up_as_fft_peaks():
    # instantaneous-frequency endpoints via the waveform itself: windows before / after the move
    L = 8192
    p = one_tone(F0, F1, A=1.0, t_start=L / FS, t_dur=4 * L / FS, profile=PROFILE_MINJERK)
    for a, f_want in ((0, F0), (5 * L, F1)):
        V = p.waveform(a, a + L) * np.hanning(L)
        j = int(np.argmax(np.abs(np.fft.rfft(V))))
        assert abs(j * FS / L - f_want) <= FS / L


def test_nyquist_folding_is_not_special_cased():
    # G16: tones above Nyquist are evaluated as given (C4 has 60-98.6 MHz at 100 MS/s): alias at |f - fs|
    fs, L = 100e6, 4096
    j = 1000
    f = fs - j * fs / L
    V = one_tone(f, fs=fs).waveform(0, L)
    F = np.abs(np.fft.rfft(V))
    assert int(np.argmax(F)) == j and F[j] == pytest.approx(L / 2, rel=1e-9)


# ------------------------------------------------------------------ precision / range reduction (Eq. 14)
def _mp_phase(seg_args, fs, n):
    """50-digit evaluation of the section-8(c) definition from the double inputs."""
    mp = mpmath.mp
    mp.dps = 50
    f0, f1, phi0, ts, T, prof = seg_args
    f0, f1, ts, T, fs = (mpmath.mpf(float(x)) for x in (f0, f1, ts, T, fs))
    theta = mpmath.mpf(float(phi0)) / (2 * mpmath.pi)
    t = mpmath.mpf(int(n)) / fs
    tau = t - ts
    if prof == PROFILE_STATIC or tau <= 0:
        return theta + f0 * t
    if tau >= T:
        return theta + f0 * ts + f1 * tau + T * (f0 - f1) / 2
    s = tau / T
    g = s ** 2 / 2 if prof == PROFILE_LINEAR else (mpmath.mpf(5) / 2 * s ** 4 - 3 * s ** 5 + s ** 6)
    return theta + f0 * t + (f1 - f0) * T * g


@pytest.mark.parametrize("cfg", ["C2", "C3"])
def test_long_phase_precision_against_50_digits(cfg):
    w = W.config2() if cfg == "C2" else W.config3(64)
    p = oracle.plan_from_workload(w)
    rng = np.random.default_rng(11)
    worst = 0.0
    for _ in range(400):
        k = int(rng.integers(0, w.n_tones))
        n = int(rng.integers(0, w.n_samples))
        ref = _mp_phase((w.f0[k], w.f1[k], w.phi0[k], w.t_start[k], w.t_dur[k], int(w.profile[k])), w.sample_rate, n)
        got = mpmath.mpf(float(p.phase(k, [n])[0] - np.floor(p.phase(k, [n])[0])))
        d = (got - (ref - mpmath.floor(ref)))
        d = abs(d - mpmath.nint(d))
        worst = max(worst, float(d))
    assert worst < 1e-9  # cycles; phases reach 5.6e6 cycles here (fp32 ulp there is 0.5 cycle)


def test_one_second_static_phase_precision():
    # C4-like: 98.6 MHz for 1 s -> 1e8 cycles; still good to 1e-9 cycle
    p = one_tone(98.6e6, phi0=2.2, fs=100e6)
    for n in (99_999_999, 100_139_007):
        ref = _mp_phase((98.6e6, 98.6e6, 2.2, 0.0, 0.0, PROFILE_STATIC), 100e6, n)
        got = float(p.phase(0, [n])[0] - np.floor(p.phase(0, [n])[0]))
        d = float(abs(mpmath.mpf(got) - (ref - mpmath.floor(ref))))
        assert min(d, 1 - d) < 1e-9


def test_range_reduction_leaves_the_sine_unchanged():
    # Eq. 14: sin(2 pi modf(phi/2pi)) = sin(phi)
    mpmath.mp.dps = 50
    p = one_tone(87.123456e6, A=1.0, phi0=0.4)
    for n in (1, 12345, 6_000_000):
        ref = _mp_phase((87.123456e6, 87.123456e6, 0.4, 0.0, 0.0, 0), FS, n)
        assert p.waveform(n, n + 1)[0] == pytest.approx(float(mpmath.sin(2 * mpmath.pi * ref)), abs=1e-9)


# ------------------------------------------------------------------ chunking and updates
def test_chunking_is_bit_identical():
    w = W.config1()
    total = 1 << 14
    ref = None
    for cl in (1 << 10, 1 << 12, 1 << 14):
        p = OraclePlan(w.n_tones, w.sample_rate, cl, w.scale)
        p.set_trajectories(w.f0, w.f1, w.A, w.phi0, w.t_start, w.t_dur, w.profile)
        got = np.concatenate([p.chunk(c) for c in range(total // cl)])
        if ref is None:
            ref = got
        assert np.array_equal(got, ref)
    assert np.array_equal(ref, oracle.plan_from_workload(w).codes(0, total))


def test_update_is_phase_and_frequency_continuous():
    cl = 4096
    p = one_tone(F0, F1, phi0=0.9, t_start=0.0, t_dur=2 * cl / FS, profile=PROFILE_MINJERK, chunk_len=cl)
    old_ph = p.phase(0, [3 * cl])[0]
    old_f = p.inst_freq(0, [3 * cl])[0]
    p.update_trajectories(3, [0], [99e6], [1.5 * cl / FS], [PROFILE_MINJERK])
    new_ph = p.phase(0, [3 * cl])[0]
    d = float((new_ph - old_ph) - np.rint(new_ph - old_ph))
    assert abs(d) < 1e-9  # same phase mod 1 at the update instant
    assert float(p.inst_freq(0, [3 * cl])[0] - old_f) == 0.0
    assert _central_freq(p, 3 * cl + 1) == pytest.approx(F1, abs=1e-2)  # (unwrapped phase is continuous only mod 1 across segments)
    assert _central_freq(p, 5 * cl) == pytest.approx(99e6, abs=1e-2)
    # samples before the update are untouched
    q = one_tone(F0, F1, phi0=0.9, t_start=0.0, t_dur=2 * cl / FS, profile=PROFILE_MINJERK, chunk_len=cl)
    assert np.array_equal(p.waveform(0, 3 * cl), q.waveform(0, 3 * cl))


def test_mid_move_update_continues_from_instantaneous_frequency():
    cl = 4096
    p = one_tone(F0, F1, t_start=0.0, t_dur=4 * cl / FS, profile=PROFILE_MINJERK, chunk_len=cl)
    f_mid = float(p.inst_freq(0, [2 * cl])[0])
    assert f_mid == pytest.approx((F0 + F1) / 2, rel=1e-12)
    ph_old = p.phase(0, [2 * cl])[0]
    p.update_trajectories(2, [0], [F0], [2 * cl / FS], [PROFILE_LINEAR])
    assert _central_freq(p, 2 * cl + 1) == pytest.approx(f_mid, abs=(F1 - F0) / (2 * cl) * 2)
    ph_new = p.phase(0, [2 * cl])[0]
    assert abs(float((ph_new - ph_old) - np.rint(ph_new - ph_old))) < 1e-9
    assert _central_freq(p, 5 * cl) == pytest.approx(F0, abs=1e-2)


def test_noop_update_leaves_waveform_unchanged():
    cl = 2048
    a = one_tone(F0, A=0.5, phi0=0.2, chunk_len=cl)
    b = one_tone(F0, A=0.5, phi0=0.2, chunk_len=cl)
    b.update_trajectories(2, [0], [F0], [3e-6], [PROFILE_MINJERK])
    assert np.abs(a.waveform(0, 6 * cl) - b.waveform(0, 6 * cl)).max() < 1e-9


def test_update_rejects_bad_orders_and_duplicates():
    p = one_tone(F0, chunk_len=1024)
    p.update_trajectories(5, [0], [F1], [1e-6], [PROFILE_MINJERK])
    with pytest.raises(ValueError):
        p.update_trajectories(4, [0], [F1], [1e-6], [PROFILE_MINJERK])
    q = OraclePlan(2, FS, 1024)
    z = np.zeros(2)
    q.set_trajectories([F0, F1], [F0, F1], [0.5, 0.5], z, z, z, [0, 0])
    with pytest.raises(ValueError):
        q.update_trajectories(1, [1, 1], [F0, F0], [1e-6, 1e-6], [2, 2])


# ------------------------------------------------------------------ two independent evaluators
@pytest.mark.parametrize("name", ["C1", "C2", "C4"])
def test_numpy_and_c_oracles_agree(name):
    w = {"C1": W.config1, "C2": W.config2, "C4": lambda: W.config4(6)}[name]()
    p = oracle.plan_from_workload(w)
    if name == "C4":
        windows = [(0, 3000), (2 * w.chunk_len - 1500, 2 * w.chunk_len + 12000), (5 * w.chunk_len, 5 * w.chunk_len + 11000)]
    elif name == "C2":
        k = int(np.argmax(w.t_dur))
        a = int(w.t_start[k] * w.sample_rate)
        windows = [(0, 4000), (a - 1000, a + 3000), (w.n_samples - 4000, w.n_samples)]
    else:
        windows = [(0, 20000), (w.n_samples - 5000, w.n_samples)]
    for a, b in windows:
        Vn, Vc = p.waveform(a, b), oracle.c_waveform(p, a, b)
        assert np.abs(Vn - Vc).max() < 1e-12
        assert np.mean(p.quantise(Vn) != oracle.c_codes(p, a, b)) <= 1e-4


# ------------------------------------------------------------------ stored values
def test_golden_c1_head_codes():
    """First 64 int16 codes of config 1, written by tests/golden/make_golden.py (which calls only oracle/):
    guards the generator's draw order and the oracle's arithmetic against accidental change."""
    path = os.path.join(GOLDEN, "c1_head_codes.txt")
    want = np.array([int(x) for x in open(path).read().split("\n") if x and not x.startswith("#")], dtype=np.int16)
    p = oracle.plan_from_workload(W.config1())
    assert np.array_equal(p.codes(0, want.shape[0]), want)
    assert np.array_equal(oracle.c_codes(p, 0, want.shape[0]), want)


def test_golden_paper_constants():
    """Numbers the paper prints (tests/golden/paper_constants.txt, each with its citation)."""
    vals = {}
    for line in open(os.path.join(GOLDEN, "paper_constants.txt")):
        if line.strip() and not line.startswith("#"):
            key, val = line.split()[:2]
            vals[key] = float(val)
    assert FS / 2 ** 20 < vals["freq_grid_error_bound_hz"] + 0.1  # "< 534 Hz"
    assert vals["chunk_samples"] == 2 ** 20 and vals["bytes_per_sample"] == 2
    assert W.config3(2).n_chunks * 2 ** 20 >= vals["playback_ms"] * 1e-3 * FS > (W.config3(2).n_chunks - 1) * 2 ** 20
    assert W.config4(1).n_tones == vals["streaming_tones_100MS"] and W.config3().n_tones == vals["playback_tones"]
    assert vals["C2_cpu_ms_per_MB"] / vals["C1_sp_ms_per_MB"] == pytest.approx(vals["speedup_sp"], abs=1.0)
    assert vals["C2_cpu_ms_per_MB"] / vals["C1_dp_ms_per_MB"] == pytest.approx(vals["speedup_dp"], abs=1.0)
