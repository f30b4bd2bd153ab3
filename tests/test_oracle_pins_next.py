"""Pins for the oracle functions of the NEXT rows: four-channel multiplexing (PAPER.md:77,
166), the static-buffer pathway (Eq. 6-9, Eq. 10 branch 3 / theta': PAPER.md:95-105, 133, 141-146) and time-varying
amplitudes (Eq. 9).  Each check is against something the paper or the mathematics fixes, not against the
oracle's own formula retyped."""
import math

import mpmath
import mpmath as mp
import numpy as np
import pytest

import oracle

STATIC, LINEAR, MINJERK = oracle.PROFILE_STATIC, oracle.PROFILE_LINEAR, oracle.PROFILE_MINJERK
FS = 560e6


def _plan(rows, L=1024, fs=FS):
    cols = list(zip(*rows))
    p = oracle.OraclePlan(len(rows), fs, L)
    p.set_trajectories(*cols)
    return p


# ------------------------------------------------------------------ Eq. 6: frequency snapping
def test_snap_frequency_grid_and_error_bound():
    L = 1 << 20
    grid = FS / L
    assert abs(grid - 534.06) < 0.005                      # "less than 534 Hz" is the grid spacing
    rng = np.random.default_rng(0)
    for f0 in rng.uniform(1e6, 270e6, 200):
        f = oracle.snap_frequency(f0, FS, L)
        j = f * L / FS
        assert abs(j - round(j)) < 1e-6                    # an integer number of cycles in L_s samples (Eq. 5/6)
        assert abs(f - f0) <= grid / 2 + 1e-6              # nearest grid point
    assert oracle.snap_frequency(7 * grid, FS, L) == pytest.approx(7 * grid, rel=0, abs=1e-6)   # grid points are fixed points
    assert oracle.snap_frequency(7.49 * grid, FS, L) == pytest.approx(7 * grid, abs=1e-6)
    assert oracle.snap_frequency(7.51 * grid, FS, L) == pytest.approx(8 * grid, abs=1e-6)


def test_snapped_tone_is_exactly_periodic_in_the_buffer_and_unsnapped_is_not():
    L = 4096
    f0 = 101.2345e6
    fsn = oracle.snap_frequency(f0, FS, L)
    p = _plan([(fsn, fsn, 0.7, 0.3, 0, 0, STATIC), (f0, f0, 0.7, 0.3, 0, 0, STATIC)], L)
    a = p.waveform(0, 3 * L, tones=[0])
    assert np.max(np.abs(a[:L] - a[L:2 * L])) < 1e-12 and np.max(np.abs(a[:L] - a[2 * L:])) < 1e-12
    b = p.waveform(0, 2 * L, tones=[1])
    assert np.max(np.abs(b[:L] - b[L:])) > 1e-3            # off the grid the looped buffer would jump: why Eq. 6 exists


# ------------------------------------------------------------------ Eq. 7-9: looped static buffer + dynamic tones
def test_static_buffer_is_one_period_of_the_direct_sum_and_single_fft_bins():
    L = 2048
    js = [37, 200, 511]
    rows = [(j * FS / L, j * FS / L, 0.1 * (i + 1), 0.4 * i, 0, 0, STATIC) for i, j in enumerate(js)]
    p = _plan(rows, L)
    X = p.static_buffer([0, 1, 2])
    assert X.shape == (L,)
    # on-grid tones: the buffer's DFT is three single bins of magnitude a L / 2 (Eq. 5)
    F = np.abs(np.fft.rfft(X))
    for i, j in enumerate(js):
        assert F[j] == pytest.approx(0.1 * (i + 1) * L / 2, rel=1e-9)
    rest = np.delete(F, js)
    assert rest.max() < 1e-8 * L
    # X[0] = sum a sin(theta) (Eq. 8 at i = 0)
    assert X[0] == pytest.approx(sum(0.1 * (i + 1) * math.sin(0.4 * i) for i in range(3)), abs=1e-14)


def test_static_pathway_equals_absolute_time_evaluation_for_snapped_tones():
    L = 4096
    rng = np.random.default_rng(3)
    rows = []
    for k in range(6):      # static set, on the grid
        f = oracle.snap_frequency(rng.uniform(60e6, 200e6), FS, L)
        rows.append((f, f, 0.1, rng.uniform(0, 6.28), 0, 0, STATIC))
    for k in range(3):      # dynamic tones: off-grid, moving
        f = rng.uniform(60e6, 200e6)
        rows.append((f, f + 3e6, 0.1, rng.uniform(0, 6.28), 2e-6, 9e-6, MINJERK))
    p = _plan(rows, L)
    X = p.static_buffer(range(6))
    n0, n1 = 3 * L - 100, 5 * L + 77       # spans two wraps of the looped buffer
    V = p.waveform_static_pathway(n0, n1, X, range(6, 9))
    assert np.max(np.abs(V - p.waveform(n0, n1))) < 1e-12
    # the looped index really is i mod L_s: the static part alone repeats with period L
    Vs = p.waveform_static_pathway(0, 3 * L, X, [])
    assert np.array_equal(Vs[:L], Vs[L:2 * L]) and np.array_equal(Vs[:L], X)


# ------------------------------------------------------------------ Eq. 10 branch 3: theta' and the hand-back
def test_handback_theta_is_the_papers_theta_prime():
    # theta' = 2 pi f_finish/fs L_d + pi T (f_start - f_finish)  [+ theta_j], t_s = 0
    mpmath.mp.dps = 50
    L = 1 << 12
    f0, f1, T, th = 100e6, 103e6, 17.3e-6, 0.77
    p = _plan([(f0, f1, 0.5, th, 0.0, T, MINJERK)], L)
    L_d = L * math.ceil(T * FS / L)
    want = (2 * mpmath.pi * mpmath.mpf(f1) / mpmath.mpf(FS) * L_d + mpmath.pi * mpmath.mpf(T) * (mpmath.mpf(f0) - mpmath.mpf(f1))
            + mpmath.mpf(th)) / (2 * mpmath.pi)
    want = want - mpmath.floor(want)
    got = mpmath.mpf(float(p.handback_theta(0, L_d)))
    d = abs(got - want)
    assert min(d, 1 - d) < 1e-9


def test_folded_buffer_continues_the_moved_tone_seamlessly():
    L = 4096
    fsn = [oracle.snap_frequency(f, FS, L) for f in (90e6, 140e6)]
    f_fin = oracle.snap_frequency(97e6, FS, L)
    T = 11.7e-6
    rows = [(fsn[0], fsn[0], 0.3, 0.2, 0, 0, STATIC), (fsn[1], fsn[1], 0.3, 1.2, 0, 0, STATIC),
            (fsn[0] + 5e6, f_fin, 0.3, 2.2, 0.0, T, MINJERK)]
    p = _plan(rows, L)
    L_d = L * math.ceil(T * FS / L)
    X = p.static_buffer([0, 1])
    X2 = p.fold_into_static_buffer(X, [2], L_d)
    # for i >= L_d the looped buffer alone is the whole waveform (Eq. 10 branch 3): sample L_d + i of the absolute-time
    # evaluation equals X2[i mod L]
    direct = p.waveform(L_d, L_d + 3 * L)
    assert np.max(np.abs(direct - np.tile(X2, 3))) < 1e-9
    # first sample after the hand-back: the moved tone's phase is theta' exactly
    assert direct[0] == pytest.approx(X[0] + 0.3 * math.sin(2 * math.pi * float(p.handback_theta(2, L_d))), abs=1e-12)
    with pytest.raises(ValueError):
        p.fold_into_static_buffer(X, [2], L_d + 8)         # L_d must be a multiple of L_s
    with pytest.raises(ValueError):
        p.fold_into_static_buffer(X, [2], 0)               # still moving


def test_unsnapped_final_frequency_would_not_loop():
    L = 4096
    T = 11.7e-6
    p = _plan([(100e6, 97.000123e6, 0.3, 2.2, 0.0, T, MINJERK)], L)
    L_d = L * math.ceil(T * FS / L)
    X2 = p.fold_into_static_buffer(np.zeros(L), [0], L_d)
    direct = p.waveform(L_d, L_d + 2 * L)
    assert np.max(np.abs(direct[:L] - X2)) < 1e-9          # the first period is right by construction of theta'
    assert np.max(np.abs(direct[L:] - X2)) > 1e-3          # the second is not: f_finish must be on the Eq. 6 grid


# ------------------------------------------------------------------ WM: four-channel multiplexing
def test_mux_channels_layout_and_bit_identity():
    L = 512
    rng = np.random.default_rng(5)
    plans = []
    for c in range(4):
        rows = [(rng.uniform(30e6, 250e6), 0, 0.3, rng.uniform(0, 6.28), 0, 0, STATIC) for _ in range(3 + c)]
        rows = [(r[0], r[0]) + r[2:] for r in rows]
        plans.append(_plan(rows, L))
    m = oracle.mux_channels(plans, 2 * L, 3 * L)
    assert m.dtype == np.int16 and m.shape == (4 * L,)
    for c in range(4):
        assert np.array_equal(m[c::4], plans[c].chunk(2))  # de-interleaved channel c = the single-channel oracle, bit for bit
    # "groups of four": element i of every channel sits in words 4 i .. 4 i + 3
    g = m.reshape(L, 4)
    assert np.array_equal(g[17], [plans[c].chunk(2)[17] for c in range(4)])
    # the paper's chunk: 2^20 samples = 4 x 2^18 = 2 MiB
    assert 4 * (1 << 18) == 1 << 20 and (1 << 20) * 2 == 2 * 1024 * 1024
    # constant channels of distinct DC levels make the layout unmistakable
    dc = [_plan([(0.0, 0.0, 0.1 * (c + 1), math.pi / 2, 0, 0, STATIC)], 8) for c in range(4)]
    md = oracle.mux_channels(dc, 0, 8)
    want = np.rint(0.9 * 32767.0 * 0.1 * np.arange(1, 5)).astype(np.int16)
    assert np.array_equal(md.reshape(8, 4), np.tile(want, (8, 1)))


# ------------------------------------------------------------------ a_j[i]: amplitude ramps
def test_amplitude_ramp_endpoints_shape_and_dc_closed_form():
    L = 4096
    Ta, ts = 5e-6, 1e-6
    # a DC "tone" (f = 0, theta = pi/2) makes V[n] = a[n]: the ramp can be read off directly
    p = _plan([(0.0, 0.0, 0.2, math.pi / 2, 0, 0, STATIC)], L)
    p.set_amplitude_ramps([0.8], [ts], [Ta], [MINJERK])
    n_s, n_e = int(round(ts * FS)), int(round((ts + Ta) * FS))
    V = p.waveform(0, L)
    assert np.allclose(V[:n_s + 1], 0.2, atol=1e-15) and np.allclose(V[n_e:], 0.8, atol=1e-12)
    mid = (n_s + n_e) // 2
    s = (mid / FS - ts) / Ta
    assert V[mid] == pytest.approx(0.2 + 0.6 * (10 * s ** 3 - 15 * s ** 4 + 6 * s ** 5), abs=1e-12)
    assert abs(V[(n_s + n_e) // 2] - 0.5) < 1e-3           # half way at half time (symmetry h(1/2) = 1/2)
    d = np.diff(V)
    assert np.all(d >= -1e-15)                             # monotone
    # minimum jerk: zero slope and curvature at both ends -> first and second differences vanish there
    assert abs(d[n_s + 1]) < 1e-6 and abs(d[n_e - 2]) < 1e-6
    dd = np.diff(V, 2)
    assert abs(dd[n_s + 1]) < 1e-8 and abs(dd[n_e - 4]) < 1e-8
    # linear ramp: constant first difference
    p.set_amplitude_ramps([0.8], [ts], [Ta], [LINEAR])
    d = np.diff(p.waveform(0, L))[n_s + 2:n_e - 2]
    assert np.ptp(d) < 1e-13 and d[0] == pytest.approx(0.6 / (Ta * FS), rel=1e-9)


def test_amplitude_ramp_multiplies_the_unramped_tone():
    L = 2048
    rows = [(80e6, 83e6, 0.5, 0.4, 0.5e-6, 2e-6, MINJERK), (120e6, 120e6, 0.25, 1.0, 0, 0, STATIC)]
    p = _plan(rows, L)
    unit = [p.waveform(0, L, tones=[k]) / p.A[k] for k in range(2)]     # sin(...) of each tone
    p.set_amplitude_ramps([0.0, 0.25], [1e-6, 0.0], [1.5e-6, 0.0], [MINJERK, STATIC])   # tone 0 fades out, tone 1 untouched
    V = p.waveform(0, L)
    a0 = p.amplitude(0, np.arange(L))
    assert np.max(np.abs(V - (a0 * unit[0] + 0.25 * unit[1]))) < 1e-15
    assert a0[0] == 0.5 and a0[-1] == 0.0
    # tone creation: A0 = 0 -> A1; before the ramp the tone is silent
    q = _plan([(80e6, 80e6, 0.0, 0.4, 0, 0, STATIC)], L)
    q.set_amplitude_ramps([0.3], [1e-6], [1e-6], [LINEAR])
    Vq = q.waveform(0, L)
    assert not Vq[:int(1e-6 * FS)].any() and np.max(np.abs(Vq[-100:])) > 0.2
    # the C evaluator follows the same ramps
    assert np.max(np.abs(oracle.c_waveform(p, 0, L) - V)) < 1e-12
    assert np.max(np.abs(oracle.c_waveform(q, 0, L) - Vq)) < 1e-12


def test_zero_duration_amplitude_step_and_static_profile():
    L = 256
    p = _plan([(0.0, 0.0, 0.2, math.pi / 2, 0, 0, STATIC)], L)
    p.set_amplitude_ramps([0.6], [99.5 / FS], [0.0], [LINEAR])   # the step falls between samples 99 and 100
    V = p.waveform(0, L)
    assert np.allclose(V[:100], 0.2) and np.allclose(V[100:], 0.6)
    p.set_amplitude_ramps([0.6], [0.0], [1e-6], [STATIC])   # STATIC profile: amplitude stays
    assert np.allclose(p.waveform(0, L), 0.2)


# ------------------------------------------------------------------ exponential chirp (PAPER.md:137 names it; reading G20)
def _exp_plan(f0=80e6, f1=120e6, T=200e-6, t_s=10e-6, phi0=0.7, fs=560e6, L=1 << 18):
    op = oracle.OraclePlan(1, fs, L)
    op.set_trajectories([f0], [f1], [1.0], [phi0], [t_s], [T], [oracle.awg_oracle.PROFILE_EXP])
    return op


def test_exp_chirp_frequency_is_geometric_and_hits_both_ends():
    """f(tau) = f0 (f1/f0)^(tau/T): f0 at the start, f1 at the end, the GEOMETRIC mean half way, log f linear in time --
    read off the oracle's own phase by central differences (the phase is what the oracle computes; the frequency law is the pin)."""
    f0, f1, T, t_s, fs = 80e6, 120e6, 200e-6, 10e-6, 560e6
    op = _exp_plan(f0, f1, T, t_s)
    def freq_at(tau):
        n = (t_s + tau) * fs
        ns = np.array([n - 0.5, n + 0.5])
        ph = oracle.awg_oracle.segment_phase(op.segments[0][0], ns.astype(np.longdouble) / np.longdouble(fs))
        return float((ph[1] - ph[0]) * fs)
    assert abs(freq_at(2e-9) - f0) < 2e3
    assert abs(freq_at(T - 2e-9) - f1) < 2e3
    assert abs(freq_at(T / 2) - math.sqrt(f0 * f1)) < 1.0          # 97.98 MHz, not the arithmetic 100 MHz
    lf = [math.log(freq_at(T * s)) for s in (0.2, 0.4, 0.6, 0.8)]
    assert abs((lf[2] - lf[1]) - (lf[1] - lf[0])) < 1e-7 and abs((lf[3] - lf[2]) - (lf[2] - lf[1])) < 1e-7
    # before the move the tone is static at f0, after it static at f1
    assert abs(freq_at(-3e-6) - f0) < 1e-3 and abs(freq_at(T + 3e-6) - f1) < 1e-3
    assert abs(float(op.inst_freq(0, np.array([int((t_s + T / 2) * fs)]))[0]) - f0 * (f1 / f0) ** ((int((t_s + T / 2) * fs) / fs - t_s) / T)) < 1e-3


def test_exp_chirp_phase_is_the_integral_of_the_geometric_frequency():
    """Closed form in 50-digit arithmetic: cycles gained over the whole move = T (f1 - f0)/ln(f1/f0) (the logarithmic mean of
    the end frequencies times T); and a brute-force trapezoid integration of f0 r^(t/T) on 10^6 points for a point mid-move."""
    mp.mp.dps = 50
    f0, f1, T, t_s, fs, phi0 = 80e6, 120e6, 200e-6, 10e-6, 560e6, 0.7
    op = _exp_plan(f0, f1, T, t_s, phi0)
    seg = op.segments[0][0]
    LD = np.longdouble
    t_end = LD(t_s) + LD(T)
    ph_end = oracle.awg_oracle.segment_phase(seg, np.array([t_end], dtype=LD))[0]
    want = mp.mpf(phi0) / (2 * mp.pi) + mp.mpf(f0) * mp.mpf(t_s) + mp.mpf(T) * (mp.mpf(f1) - mp.mpf(f0)) / mp.log(mp.mpf(f1) / mp.mpf(f0))
    assert abs(mp.mpf(float(ph_end)) - want) < mp.mpf("1e-8")
    # continuity at the end of the move and slope f1 afterwards
    ph_after = oracle.awg_oracle.segment_phase(seg, np.array([t_end + LD(1e-6)], dtype=LD))[0]
    assert abs(float(ph_after - ph_end) - f1 * 1e-6) < 1e-9
    # trapezoid integration of the frequency law up to tau = 0.37 T
    tau = 0.37 * T
    grid = np.linspace(0.0, tau, 1_000_001)
    f = f0 * (f1 / f0) ** (grid / T)
    integral = float(np.sum((f[1:] + f[:-1]) * 0.5) * (grid[1] - grid[0]))
    ph_mid = oracle.awg_oracle.segment_phase(seg, np.array([LD(t_s) + LD(tau)], dtype=LD))[0]
    assert abs(float(ph_mid) - (phi0 / (2 * math.pi) + f0 * t_s + integral)) < 1e-7
    # it is not the linear chirp between the same ends: the two differ by many cycles mid-move
    lin = oracle.OraclePlan(1, fs, 1 << 18)
    lin.set_trajectories([f0], [f1], [1.0], [phi0], [t_s], [T], [oracle.awg_oracle.PROFILE_LINEAR])
    ph_lin = oracle.awg_oracle.segment_phase(lin.segments[0][0], np.array([LD(t_s) + LD(T / 2)], dtype=LD))[0]
    ph_exp = oracle.awg_oracle.segment_phase(seg, np.array([LD(t_s) + LD(T / 2)], dtype=LD))[0]
    assert abs(float(ph_lin - ph_exp)) > 50.0


def test_exp_chirp_limits_updates_and_c_evaluator():
    """f1 -> f0: the exponential chirp tends to the static tone; a downward chirp mirrors an upward one; an update mid-move
    continues phase and frequency; the C evaluator agrees with numpy."""
    fs, L = 560e6, 1 << 16
    near = _exp_plan(90e6, 90e6 * (1 + 1e-13), 100e-6, 0.0, 0.3, fs, L)
    sta = oracle.OraclePlan(1, fs, L)
    sta.set_trajectories([90e6], [90e6], [1.0], [0.3], [0.0], [0.0], [oracle.awg_oracle.PROFILE_STATIC])
    assert np.abs(near.waveform(0, 4096) - sta.waveform(0, 4096)).max() < 1e-6
    down = _exp_plan(120e6, 80e6, 150e-6, 5e-6, 0.1, fs, L)
    n_mid = int((5e-6 + 75e-6) * fs)
    assert abs(float(down.inst_freq(0, np.array([n_mid]))[0]) - 120e6 * (80e6 / 120e6) ** ((n_mid / fs - 5e-6) / 150e-6)) < 1e-3
    # mid-move update: phase- and frequency-continuous (G12)
    op = _exp_plan(80e6, 120e6, 400e-6, 0.0, 0.2, fs, L)
    n_u = 1 * L
    f_before = float(op.inst_freq(0, np.array([n_u]))[0])
    ph_before = op.phase(0, np.array([n_u]))[0]
    op.update_trajectories(1, [0], [70e6], [100e-6], [oracle.awg_oracle.PROFILE_EXP])
    assert abs(float(op.inst_freq(0, np.array([n_u]))[0]) - f_before) < 1e-3
    d = float(op.phase(0, np.array([n_u]))[0] - ph_before)
    assert abs(d - round(d)) < 1e-9
    # numpy vs C on a window that covers the update and the end of the new move
    V_np = op.waveform(n_u - 64, n_u + 60000)
    V_c = oracle.c_waveform(op, n_u - 64, n_u + 60000)
    assert np.abs(V_np - V_c).max() < 1e-12
