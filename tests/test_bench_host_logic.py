"""Host-side arithmetic of bench.py's roofline accounting (no GPU): which pipe binds, how the algorithmic
operations are counted (DESIGN.md section 6 "Roofline": 1 multiply-add per static tone-sample, 2 inside a slow
move, 1 MUFU.SIN + 2 multiply-adds inside any other move), and that frac = roofline time / measured time."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import awg_workloads as W  # noqa: E402
import bench  # noqa: E402


def test_moving_tone_samples_counts_overlap_with_the_launch():
    w = W.config3()  # every tone moves for 35 ms from t = 0; the buffer is 19 x 2^20 samples at 560 MS/s
    n_move = int(35e-3 * 560e6)
    assert bench.moving_tone_samples(w) == w.n_tones * n_move
    w1 = W.config1()  # 4 linear chirps over the whole 2^20-sample span, 12 static tones
    assert bench.moving_tone_samples(w1) == 4 * w1.n_samples
    w2 = W.config2()
    want = 0
    for k in range(w2.n_tones):
        if w2.profile[k] != W.PROFILE_STATIC:
            a = w2.t_start[k] * 560e6
            b = min(w2.n_samples, (w2.t_start[k] + w2.t_dur[k]) * 560e6)
            want += int(b - a)
    assert bench.moving_tone_samples(w2) == want
    assert 0 < want < 0.03 * w2.tone_samples  # ~1.4 % of C2's tone-samples sit inside a move


def test_pipe_roofline_picks_the_binding_pipe_and_scales_with_time():
    sm_mhz = 1965.0
    fma_peak = 128 * 148 * sm_mhz * 1e6
    xu_peak = 16 * 148 * sm_mhz * 1e6
    w2 = W.config2()
    r = bench.pipe_roofline(w2, 0.05, "auto", sm_mhz)
    assert r["bound"] == "alu" and r["pipe"].startswith("FMA") and r["unit"] == "GFMA/s"
    n_mov = bench.moving_tone_samples(w2)
    assert r["fma_ops"] == (w2.tone_samples - n_mov) + 2 * n_mov and r["mufu_ops"] == n_mov
    assert np.isclose(r["frac"], (r["fma_ops"] / fma_peak) / 0.05e-3)
    assert np.isclose(r["achieved"] / r["peak"], r["frac"])
    assert np.isclose(bench.pipe_roofline(w2, 0.10, "auto", sm_mhz)["frac"], r["frac"] / 2)
    # every tone-sample through MUFU: the XU pipe binds (1 sine against 2 multiply-adds at an 8:1 peak ratio)
    rm = bench.pipe_roofline(w2, 0.2, "mufu", sm_mhz)
    assert rm["pipe"].startswith("XU") and rm["mufu_ops"] == w2.tone_samples
    assert np.isclose(rm["frac"], (w2.tone_samples / xu_peak) / 0.2e-3)
    # C3: every tone is a slow mover (10 MHz over 35 ms): two multiply-adds per moving tone-sample, no sine per sample
    w3 = W.config3()
    fast, slow = bench.moving_tone_samples(w3, split=True)
    assert fast == 0 and slow == w3.n_tones * int(35e-3 * 560e6)
    r3 = bench.pipe_roofline(w3, 2.25, "auto", sm_mhz)
    assert r3["pipe"].startswith("FMA") and r3["mufu_ops"] == 0
    assert np.isclose(r3["frac"], ((w3.tone_samples - slow) + 2 * slow) / fma_peak / 2.25e-3)
    # the fast moves of C2 (0.5-5 MHz in 50-500 us) are not slow movers
    assert bench.moving_tone_samples(w2, split=True)[1] == 0
    assert not bench.is_slow_mover(W.PROFILE_MINJERK, 5e6 * 200e-6, 200e-6 * 560e6)
    assert bench.is_slow_mover(W.PROFILE_MINJERK, 10e6 * 35e-3, 35e-3 * 560e6)
