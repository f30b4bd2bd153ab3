"""GPU parity for the NEXT rows of SURVEY.md section 8(f), through the C ABI, against the oracle:
NEXT-2 four-channel multiplexed output, NEXT-3 static-buffer pathway (Eq. 6-9 and the theta'
hand-back of Eq. 10 branch 3), NEXT-4 time-varying amplitudes (Eq. 9).  Same bar as test_gpu_parity.py."""
import math

import numpy as np
import pytest

import awg_workloads as W
import oracle
from parity_util import assert_codes_close, assert_f32_close

pytestmark = pytest.mark.gpu

STATIC, LINEAR, MINJERK = W.PROFILE_STATIC, W.PROFILE_LINEAR, W.PROFILE_MINJERK
FS = 560e6


@pytest.fixture(scope="module")
def torch_cuda():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    return torch


@pytest.fixture(params=["fma", "mufu"])
def eng(request, awg):
    return {"fma": awg.AWG_ENGINE_FMA, "mufu": awg.AWG_ENGINE_MUFU}[request.param]


def _np(t):
    return t.cpu().numpy()


def _pair(awg, fs, chunk_len, rows, engine=None):
    cols = list(zip(*rows))
    p = awg.Plan(len(rows), fs, chunk_len, None, engine if engine is not None else awg.AWG_ENGINE_AUTO)
    p.set_trajectories(*cols)
    op = oracle.OraclePlan(len(rows), fs, chunk_len)
    op.set_trajectories(*cols)
    return p, op


# ------------------------------------------------------------------ NEXT-2: multiplexed channels
def _channel_rows(rng, n_tones, span):
    rows = []
    for k in range(n_tones):
        f0 = rng.uniform(20e6, 250e6)
        if k % 3 == 2:
            T = rng.uniform(0.1, 0.5) * span
            rows.append((f0, f0 + rng.choice([-1, 1]) * rng.uniform(0.5e6, 5e6), 1.0 / n_tones, rng.uniform(0, 6.28),
                         rng.uniform(0, span - T), T, MINJERK))
        else:
            rows.append((f0, f0, 1.0 / n_tones, rng.uniform(0, 6.28), 0.0, 0.0, STATIC))
    return rows


def test_mux4_paper_chunk(awg, torch_cuda, eng):
    """The paper's streaming chunk: 2^20 samples = 4 channels x 2^18, 20 tones per channel (its
    560 MS/s streaming figure), groups of four."""
    L = 1 << 18
    rng = np.random.default_rng(22)
    pairs = [_pair(awg, FS, L, _channel_rows(rng, 20, 2 * L / FS), eng) for _ in range(4)]
    plans, oplans = [p for p, _ in pairs], [o for _, o in pairs]
    for c in (0, 1):
        got = _np(awg.synthesize_chunk_mux(plans, c))
        assert got.shape == (4 * L,)
        for ch in range(4):
            single = _np(plans[ch].synthesize_chunk(c))
            assert np.array_equal(got[ch::4], single), f"channel {ch} of chunk {c} differs from its single-channel synthesis"
            V = oracle.c_waveform(oplans[ch], c * L, (c + 1) * L)
            assert_codes_close(got[ch::4], oplans[ch].quantise(V), f"mux chunk {c} channel {ch}")
    # the oracle's own interleave on a window (first 4096 sample indices of chunk 1)
    want = oracle.mux_channels(oplans, L, L + 4096)
    assert_codes_close(_np(awg.synthesize_chunk_mux(plans, 1))[:4 * 4096], want, "mux vs oracle.mux_channels")
    for p in plans:
        p.close()


def test_mux_other_channel_counts_and_ragged_chunks(awg, torch_cuda, eng):
    L = 1000   # not a multiple of the 2048-sample tile: partial tiles at both chunk edges
    rng = np.random.default_rng(23)
    for C, sizes in ((2, (5, 40)), (3, (1, 33, 7)), (1, (12,))):
        pairs = [_pair(awg, FS, L, _channel_rows(rng, n, 6 * L / FS), eng) for n in sizes]
        plans, oplans = [p for p, _ in pairs], [o for _, o in pairs]
        for c in (0, 3, 5):
            got = _np(awg.synthesize_chunk_mux(plans, c))
            assert_codes_close(got, oracle.mux_channels(oplans, c * L, (c + 1) * L), f"mux C={C} chunk {c}")
            for ch in range(C):
                assert np.array_equal(got[ch::C], _np(plans[ch].synthesize_chunk(c)))
        for p in plans:
            p.close()


def test_mux_errors(awg, torch_cuda):
    torch = torch_cuda
    a = awg.Plan(2, FS, 1024)
    b = awg.Plan(2, FS, 2048)
    z = np.zeros(2)
    for p in (a, b):
        p.set_trajectories(z + 1e6, z + 1e6, z + 0.1, z, z, z, np.zeros(2, np.int32))
    buf = torch.empty(4096, dtype=torch.int16, device="cuda")
    with pytest.raises(awg.AwgError) as ei:
        awg.awg_synthesize_chunk_mux([a.handle, b.handle], 0, buf.data_ptr())
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG      # chunk_len mismatch
    with pytest.raises(awg.AwgError) as ei:
        awg.awg_synthesize_chunk_mux([a.handle, a.handle], 0, buf.data_ptr())
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG      # the same plan twice
    c = awg.Plan(2, FS, 1024)                               # no table yet
    with pytest.raises(awg.AwgError) as ei:
        awg.awg_synthesize_chunk_mux([a.handle, c.handle], 0, buf.data_ptr())
    assert ei.value.status == awg.AWG_ERR_STATE
    a.close(); b.close(); c.close()


# ------------------------------------------------------------------ NEXT-3: static-buffer pathway
def test_snap_frequency_matches_eq6(awg):
    L = 1 << 20
    assert awg.awg_snap_frequency(100e6, FS, L) == oracle.snap_frequency(100e6, FS, L)
    assert abs(awg.awg_snap_frequency(100e6, FS, L) - 100e6) <= FS / L / 2
    assert abs(FS / L - 534.06) < 0.005
    with pytest.raises(awg.AwgError):
        awg.awg_snap_frequency(100e6, -1.0, L)


def _static_rows(rng, L, n_static, n_dyn, span):
    rows = []
    for k in range(n_static):
        f = oracle.snap_frequency(rng.uniform(40e6, 240e6), FS, L)
        rows.append((f, f, 0.8 / (n_static + n_dyn), rng.uniform(0, 6.28), 0.0, 0.0, STATIC))
    for k in range(n_dyn):
        f = rng.uniform(40e6, 240e6)
        T = rng.uniform(0.1, 0.4) * span
        rows.append((f, f + rng.choice([-1, 1]) * rng.uniform(1e6, 5e6), 0.8 / (n_static + n_dyn), rng.uniform(0, 6.28),
                     rng.uniform(0, span - T), T, MINJERK if k % 2 else LINEAR))
    return rows


@pytest.mark.parametrize("L,n_static,n_dyn", [(1 << 14, 40, 5), (4096, 3, 70), (6000, 130, 2)])
def test_static_pathway_equals_per_sample_evaluation(awg, torch_cuda, eng, L, n_static, n_dyn):
    rng = np.random.default_rng(L + n_static)
    rows = _static_rows(rng, L, n_static, n_dyn, 5 * L / FS)
    p, op = _pair(awg, FS, L, rows, eng)
    chunks = (0, 1, 4, 77)
    direct = {c: (_np(p.synthesize_chunk(c)), _np(p.synthesize_chunk_f32(c))) for c in chunks}
    p.static_buffer_set(range(n_static))
    # the buffer is Eq. 8 over one period
    X = op.static_buffer(range(n_static))
    assert_f32_close(_np(p.static_buffer()), X, "X_static", tol=2e-6)
    assert p.op_counts(0, 1)[0] + sum(p.op_counts(0, 1)[1:]) == n_dyn * L      # only the dynamic tones are evaluated per sample
    for c in chunks:
        V = oracle.c_waveform(op, c * L, (c + 1) * L)                            # absolute-time definition
        Vp = op.waveform_static_pathway(c * L, (c + 1) * L, X, range(n_static, n_static + n_dyn))
        assert np.max(np.abs(V - Vp)) < 1e-9
        f = _np(p.synthesize_chunk_f32(c))
        assert_f32_close(f, V, f"static pathway f32 chunk {c}")
        got = _np(p.synthesize_chunk(c))
        assert_codes_close(got, op.quantise(V), f"static pathway chunk {c}")
        # and within rounding of the plan's own per-sample evaluation
        assert np.max(np.abs(got.astype(np.int32) - direct[c][0].astype(np.int32))) <= 1
        assert np.max(np.abs(f - direct[c][1])) < 2e-6
    # a range launch over several chunks wraps the looped index
    r = _np(p.synthesize_range(3, 3))
    assert_codes_close(r, op.quantise(oracle.c_waveform(op, 3 * L, 6 * L)), "static pathway range")
    # removing the buffer restores the per-sample evaluation bit for bit
    p.static_buffer_set([])
    assert np.array_equal(_np(p.synthesize_chunk(4)), direct[4][0])
    p.close()


def test_static_buffer_handback_theta_prime(awg, torch_cuda, eng):
    """Eq. 10 branch 3: after L_d the moved tones are looped static wavetables with theta'."""
    L = 8192
    rng = np.random.default_rng(8)
    T = 30e-6                                              # 16800 samples: L_d = 3 L
    L_d_chunks = math.ceil(T * FS / L)
    rows = []
    for k in range(10):
        f = oracle.snap_frequency(rng.uniform(40e6, 240e6), FS, L)
        rows.append((f, f, 0.05, rng.uniform(0, 6.28), 0.0, 0.0, STATIC))
    for k in range(6):   # movers that end ON the grid (they can be handed back) ...
        f1 = oracle.snap_frequency(rng.uniform(40e6, 240e6), FS, L)
        rows.append((f1 + rng.uniform(-4e6, 4e6), f1, 0.05, rng.uniform(0, 6.28), 0.0, T * rng.uniform(0.5, 1.0), MINJERK))
    rows.append((100e6, 103.000123e6, 0.05, 0.3, 0.0, T, MINJERK))   # ... and one that ends off the grid
    p, op = _pair(awg, FS, L, rows, eng)
    p.static_buffer_set(range(10))
    X = op.static_buffer(range(10))
    for c in range(L_d_chunks):                            # the dynamic phase: static buffer + movers
        V = oracle.c_waveform(op, c * L, (c + 1) * L)
        assert_f32_close(_np(p.synthesize_chunk_f32(c)), V, f"before the hand-back, chunk {c}")
    with pytest.raises(awg.AwgError) as ei:
        p.static_buffer_fold(1, [10])                      # still moving at chunk 1
    assert ei.value.status == awg.AWG_ERR_STATE
    with pytest.raises(awg.AwgError) as ei:
        p.static_buffer_fold(L_d_chunks, [16])             # ends off the Eq. 6 grid
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    p.static_buffer_fold(L_d_chunks, range(10, 16))
    X2 = op.fold_into_static_buffer(X, range(10, 16), L_d_chunks * L)
    assert_f32_close(_np(p.static_buffer()), X2, "X_static after the hand-back", tol=3e-6)
    assert sum(p.op_counts(L_d_chunks, 1)) == L            # one tone left in the per-sample evaluation
    for c in (L_d_chunks, L_d_chunks + 1, L_d_chunks + 50):
        V = oracle.c_waveform(op, c * L, (c + 1) * L)      # absolute time, every tone: the loop is seamless
        assert_f32_close(_np(p.synthesize_chunk_f32(c)), V, f"after the hand-back, chunk {c}")
        assert_codes_close(_np(p.synthesize_chunk(c)), op.quantise(V), f"after the hand-back, chunk {c}")
    with pytest.raises(awg.AwgError) as ei:
        p.synthesize_chunk(0)                              # the past is fixed, as after an update
    assert ei.value.status == awg.AWG_ERR_STATE
    with pytest.raises(awg.AwgError) as ei:
        p.update_trajectories(L_d_chunks + 1, [3], [90e6], [1e-6], [MINJERK])   # a tone in the buffer cannot move
    assert ei.value.status == awg.AWG_ERR_STATE
    p.close()


def test_static_buffer_alone_and_errors(awg, torch_cuda):
    L = 4096
    f = [oracle.snap_frequency(x, FS, L) for x in (50e6, 75e6, 111e6)]
    rows = [(f[k], f[k], 0.3, 0.5 * k, 0.0, 0.0, STATIC) for k in range(3)] + [(60.00001e6, 60.00001e6, 0.1, 0, 0, 0, STATIC)]
    p, op = _pair(awg, FS, L, rows)
    with pytest.raises(awg.AwgError) as ei:
        p.static_buffer_set([0, 3])                        # tone 3 is off the grid
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        p.static_buffer_set([0, 0])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        p.static_buffer()                                  # no buffer yet
    assert ei.value.status == awg.AWG_ERR_STATE
    p.static_buffer_set([0, 1, 2])
    # every on-grid tone in the buffer; then fold the last one too (it is static: theta' is its phase): nothing is left
    # to evaluate per sample and the output is the looped buffer, quantised
    V = oracle.c_waveform(op, 9 * L, 10 * L)
    assert_codes_close(_np(p.synthesize_chunk(9)), op.quantise(V), "three tones from the buffer")
    q, oq = _pair(awg, FS, L, rows[:3])
    q.static_buffer_set([0, 1, 2])
    assert sum(q.op_counts(0, 1)) == 0
    X = oq.static_buffer([0, 1, 2])
    for c in (0, 5):
        assert_f32_close(_np(q.synthesize_chunk_f32(c)), X, "looped buffer only", tol=2e-6)
        assert_codes_close(_np(q.synthesize_chunk(c)), oq.quantise(X), "looped buffer only")
    small = awg.Plan(1, FS, 1024)
    small.set_trajectories([FS / 8], [FS / 8], [0.5], [0.0], [0.0], [0.0], [STATIC])
    with pytest.raises(awg.AwgError) as ei:
        small.static_buffer_set([0])                       # chunk_len < 2048
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    p.close(); q.close(); small.close()


# ------------------------------------------------------------------ NEXT-4: time-varying amplitudes a_j[i]
def _ramp_pair(awg, L, rows, ramps, engine):
    p, op = _pair(awg, FS, L, rows, engine)
    cols = list(zip(*ramps))
    p.set_amplitude_ramps(*cols)
    op.set_amplitude_ramps(*cols)
    return p, op


@pytest.mark.parametrize("engine", ["fma", "mufu", "fp64"])
def test_amplitude_ramps_creation_removal_and_moving_tones(awg, torch_cuda, engine):
    """Tone creation (0 -> A), removal (A -> 0), a ramp on a moving tone, a ramp shorter than a block, an instant step,
    linear and minimum-jerk profiles; chunks before, inside and after the ramps."""
    eng = {"fma": awg.AWG_ENGINE_FMA, "mufu": awg.AWG_ENGINE_MUFU, "fp64": awg.AWG_ENGINE_FP64}[engine]
    L = 4096
    us = 1e-6
    rows = [
        (100e6, 100e6, 0.0, 0.3, 0.0, 0.0, STATIC),            # created: 0 -> 0.15 over 12 us (min-jerk)
        (85e6, 85e6, 0.15, 1.3, 0.0, 0.0, STATIC),             # removed: 0.15 -> 0 over 9 us (linear)
        (120e6, 124e6, 0.15, 2.3, 5 * us, 20 * us, MINJERK),   # moves AND fades 0.15 -> 0.05 while moving
        (140e6, 140e6, 0.10, 0.7, 0.0, 0.0, STATIC),           # 0.3 us ramp: shorter than a 512-sample block
        (60e6, 61e6, 0.10, 0.1, 2 * us, 30 * us, LINEAR),      # instant amplitude step at 10.3 us while chirping
        (200e6, 200e6, 0.15, 0.9, 0.0, 0.0, STATIC),           # untouched
        (70e6, 75e6, 0.10, 0.2, 30 * us, 8 * us, MINJERK),     # ramp long before its move
    ]
    ramps = [(0.15, 4 * us, 12 * us, MINJERK), (0.0, 7.7 * us, 9 * us, LINEAR), (0.05, 11 * us, 10 * us, MINJERK),
             (0.02, 13.1 * us, 0.3 * us, MINJERK), (0.2, 10.3 * us, 0.0, LINEAR), (0.0, 0.0, 0.0, STATIC),
             (0.15, 1 * us, 6 * us, LINEAR)]
    p, op = _ramp_pair(awg, L, rows, ramps, eng)
    n_chunks = 8                                            # 58 us: every ramp and move ends inside
    V = oracle.c_waveform(op, 0, n_chunks * L)
    gotf = np.concatenate([_np(p.synthesize_chunk_f32(c)) for c in range(n_chunks)])
    emax = assert_f32_close(gotf, V, f"amplitude ramps {engine}", tol=3e-7 if engine == "fp64" else 1e-5)
    got = np.concatenate([_np(p.synthesize_chunk(c)) for c in range(n_chunks)])
    assert_codes_close(got, op.quantise(V), f"amplitude ramps {engine}")
    # one range launch gives the same bits as the chunks
    assert np.array_equal(_np(p.synthesize_range(0, n_chunks)), got)
    # long after everything: the tones sit at their final amplitudes (the post-move tables carry A1)
    c = 500
    Vl = oracle.c_waveform(op, c * L, (c + 1) * L)
    assert_f32_close(_np(p.synthesize_chunk_f32(c)), Vl, "after the ramps")
    assert np.max(np.abs(Vl)) > 0.1
    print(f"amplitude ramps {engine}: f32 max err {emax:.2e}")
    p.close()


def test_amplitude_ramp_then_update_and_errors(awg, torch_cuda, eng):
    L = 2048
    rows = [(90e6, 90e6, 0.0, 0.4, 0.0, 0.0, STATIC), (110e6, 110e6, 0.3, 0.0, 0.0, 0.0, STATIC)]
    ramps = [(0.3, 1e-6, 4e-6, MINJERK), (0.0, 0.0, 0.0, STATIC)]
    p, op = _ramp_pair(awg, L, rows, ramps, eng)
    # chunk 3 starts after the ramp has ended (5 us = 2800 samples): a frequency update there continues at amplitude A1
    for plan in (p, op):
        plan.update_trajectories(3, [0], [93e6], [3e-6], [MINJERK])
    for c in (3, 4, 5, 9):
        V = oracle.c_waveform(op, c * L, (c + 1) * L)
        assert_f32_close(_np(p.synthesize_chunk_f32(c)), V, f"update after a ramp, chunk {c}")
        assert_codes_close(_np(p.synthesize_chunk(c)), op.quantise(V), f"update after a ramp, chunk {c}")
    with pytest.raises(awg.AwgError) as ei:
        p.set_amplitude_ramps([0.1, 0.1], [0, 0], [1e-6, 1e-6], [LINEAR, LINEAR])
    assert ei.value.status == awg.AWG_ERR_STATE            # after a per-chunk update
    q = awg.Plan(2, FS, L)
    with pytest.raises(awg.AwgError) as ei:
        q.set_amplitude_ramps([0.1, 0.1], [0, 0], [1e-6, 1e-6], [LINEAR, LINEAR])
    assert ei.value.status == awg.AWG_ERR_STATE            # no table yet
    q.set_trajectories([1e6, 2e6], [1e6, 2e6], [0.1, 0.1], [0, 0], [0, 0], [0, 0], [STATIC, STATIC])
    with pytest.raises(awg.AwgError) as ei:
        q.set_amplitude_ramps([0.1, 0.1], [0, 0], [-1e-6, 1e-6], [LINEAR, LINEAR])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        q.set_amplitude_ramps([0.1, 0.1], [0, 0], [1e-6, 1e-6], [LINEAR, 9])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    p.close(); q.close()


def test_amplitude_ramps_many_tones_bit_identical_chunkings(awg, torch_cuda, eng):
    """130 tones over two warps' batches, a third of them fading in or out: chunkings agree bit for bit."""
    N, L = 130, 1 << 14
    rng = np.random.default_rng(41)
    rows = _channel_rows(rng, N, 3 * L / FS)
    ramps = []
    for k in range(N):
        if k % 3 == 0:
            ramps.append((rows[k][2] * rng.uniform(0, 2), rng.uniform(0, 40e-6), rng.uniform(2e-6, 30e-6), MINJERK if k % 2 else LINEAR))
        else:
            ramps.append((0.0, 0.0, 0.0, STATIC))
    p, op = _ramp_pair(awg, L, rows, ramps, eng)
    ref = _np(p.synthesize_range(0, 3))
    V = oracle.c_waveform(op, 0, 3 * L)
    assert_codes_close(ref, op.quantise(V), "ramps, 130 tones")
    cols = list(zip(*rows)); rc = list(zip(*ramps))
    q = awg.Plan(N, FS, 1000, None, eng)
    q.set_trajectories(*cols)
    q.set_amplitude_ramps(*rc)
    for c in (0, 7, 16, 33, 48):
        assert np.array_equal(_np(q.synthesize_chunk(c)), ref[c * 1000:(c + 1) * 1000]), c
    p.close(); q.close()


# ------------------------------------------------------------------ the NEXT rows on large tables (leaves, cross-CTA launches)
def test_next_rows_on_a_large_table_cross_cta_and_one_cta_agree(awg, torch_cuda, eng):
    """700 tones (3 quads of leaves): amplitude ramps on a fifth of the tones, 600 on-grid static tones moved into the looped
    static buffer, the rest evaluated per sample.  A 2^21-sample chunk (1024 tiles: quads walked inside one CTA) and 2^15-sample
    launches of the same samples (16 tiles: quads spread over CTAs, int32 scratch tiles) must agree bit for bit, and match the
    oracle's static pathway."""
    N, L, l = 700, 1 << 21, 1 << 15
    rng = np.random.default_rng(77)
    f_grid = np.array([awg.awg_snap_frequency(float(f), FS, L) for f in rng.uniform(30e6, 250e6, N)])
    rows = []
    for k in range(N):
        if k < 600 and k % 5:
            rows.append((f_grid[k], f_grid[k], 1.0 / N, rng.uniform(0, 6.28), 0.0, 0.0, STATIC))
        else:
            T = rng.uniform(100e-6, 900e-6)
            rows.append((f_grid[k], f_grid[k] + rng.uniform(-3e6, 3e6), 1.0 / N, rng.uniform(0, 6.28), rng.uniform(0, 0.9e-3), T, MINJERK))
    ramps = [((rows[k][2] * rng.uniform(0, 2), rng.uniform(0, 1.2e-3), rng.uniform(20e-6, 300e-6), MINJERK if k % 2 else LINEAR)
              if (k % 5 == 0) else (0.0, 0.0, 0.0, STATIC)) for k in range(N)]
    cols, rc = list(zip(*rows)), list(zip(*ramps))
    static_idx = np.array([k for k in range(600) if k % 5], dtype=np.int32)
    # the same samples under two chunk lengths: the static buffer loops with period L, so the small plan cannot hold one;
    # the buffer pathway is checked on the large plan, the chunking identity on the per-sample evaluation
    big = awg.Plan(N, FS, L, None, eng); big.set_trajectories(*cols); big.set_amplitude_ramps(*rc)
    small = awg.Plan(N, FS, l, None, eng); small.set_trajectories(*cols); small.set_amplitude_ramps(*rc)
    ref = _np(big.synthesize_chunk(0))
    parts = np.concatenate([_np(small.synthesize_chunk(c)) for c in range(L // l)])
    assert np.array_equal(parts, ref), "ramps + large table: cross-CTA launches differ from the one-CTA launch"
    op = oracle.OraclePlan(N, FS, L)
    op.set_trajectories(*cols)
    op.set_amplitude_ramps(*rc)
    for a in (0, 5 * l, L - l):
        V = oracle.c_waveform(op, a, a + l)
        assert_codes_close(ref[a:a + l], op.quantise(V), f"large table with ramps @ {a}")
    # static-buffer pathway on the large plan: 480 tones leave the per-sample table (220 left: the lean kernel), same codes +-1
    big.static_buffer_set(static_idx)
    got = _np(big.synthesize_chunk(0))
    d = np.abs(got.astype(np.int32) - ref.astype(np.int32))
    assert d.max() <= 1, "static-buffer pathway moved a code by more than one LSB"
    big.close(); small.close()


def test_cross_cta_launches_on_two_streams_at_once(awg, torch_cuda):
    """Two 1000-tone plans launching 2^16-sample chunks (32 tiles x 4 quads: cross-CTA) on two streams at the same time:
    each stream has its own scheduler slot, arrival counters and scratch tiles, so the results equal the one-at-a-time ones."""
    torch = torch_cuda
    w1, w2 = W.config5_cell(1024, 1 << 16), W.config5_cell(4096, 1 << 16)
    p1, p2 = awg.Plan.from_workload(w1), awg.Plan.from_workload(w2)
    ref1, ref2 = _np(p1.synthesize_chunk(0)), _np(p2.synthesize_chunk(0))
    s1, s2 = torch.cuda.Stream(), torch.cuda.Stream()
    outs1, outs2 = [], []
    for _ in range(24):
        with torch.cuda.stream(s1):
            outs1.append(p1.synthesize_chunk(0))
        with torch.cuda.stream(s2):
            outs2.append(p2.synthesize_chunk(0))
    s1.synchronize(); s2.synchronize()
    assert all(np.array_equal(_np(o), ref1) for o in outs1)
    assert all(np.array_equal(_np(o), ref2) for o in outs2)
    p1.close(); p2.close()


# ------------------------------------------------------------------ NEXT-4: exponential chirps (G20)
EXP = W.PROFILE_EXP


@pytest.mark.parametrize("engine", ["fma", "mufu", "fp64"])
def test_exponential_chirps_on_three_engines(awg, torch_cuda, engine):
    """Upward, downward, octave-wide, nearly flat, very short, instant and not-yet-started exponential chirps beside
    tones of the other profiles; chunks before, inside and after the moves; chunkings agree bit for bit."""
    eng = {"fma": awg.AWG_ENGINE_FMA, "mufu": awg.AWG_ENGINE_MUFU, "fp64": awg.AWG_ENGINE_FP64}[engine]
    L = 4096
    us = 1e-6
    rows = [
        (100e6, 130e6, 0.12, 0.3, 3 * us, 25 * us, EXP),
        (90e6, 60e6, 0.12, 1.3, 0.0, 40 * us, EXP),
        (40e6, 160e6, 0.10, 2.1, 6.5 * us, 17.3 * us, EXP),           # two octaves
        (150e6, 150e6 * (1 + 1e-9), 0.08, 0.9, 1 * us, 30 * us, EXP),  # ln(f1/f0) ~ 1e-9
        (70e6, 75e6, 0.08, 0.2, 12 * us, 0.4 * us, EXP),               # shorter than a 512-sample block
        (200e6, 210e6, 0.08, 0.5, 9 * us, 0.0, EXP),                   # instant retune
        (55e6, 50e6, 0.08, 0.4, -20 * us, 35 * us, EXP),               # started before sample 0
        (120e6, 120e6, 0.08, 0.0, 2 * us, 9 * us, EXP),                # f1 = f0: a static tone
        (180e6, 185e6, 0.08, 1.7, 4 * us, 20 * us, MINJERK),
        (30e6, 30e6, 0.10, 0.6, 0.0, 0.0, STATIC),
    ]
    p, op = _pair(awg, FS, L, rows, eng)
    n_chunks = 8                                             # 58 us: every move ends inside
    V = oracle.c_waveform(op, 0, n_chunks * L)
    gotf = np.concatenate([_np(p.synthesize_chunk_f32(c)) for c in range(n_chunks)])
    emax = assert_f32_close(gotf, V, f"exponential chirps {engine}", tol=3e-7 if engine == "fp64" else 1e-5)
    got = np.concatenate([_np(p.synthesize_chunk(c)) for c in range(n_chunks)])
    assert_codes_close(got, op.quantise(V), f"exponential chirps {engine}")
    assert np.array_equal(_np(p.synthesize_range(0, n_chunks)), got)
    q = awg.Plan(len(rows), FS, 1000, None, eng)
    q.set_trajectories(*list(zip(*rows)))
    for c in (0, 3, 11, 20, 31):
        assert np.array_equal(_np(q.synthesize_chunk(c)), got[c * 1000:(c + 1) * 1000]), c
    # long after the moves: each tone sits at f1 with the phase the whole chirp left behind
    c = 3000
    Vl = oracle.c_waveform(op, c * L, (c + 1) * L)
    assert_f32_close(_np(p.synthesize_chunk_f32(c)), Vl, "after the exponential chirps")
    print(f"exponential chirps {engine}: f32 max err {emax:.2e}")
    p.close(); q.close()


def test_exponential_chirp_updates_and_errors(awg, torch_cuda, eng):
    """Per-chunk updates into and out of exponential chirps, one of them landing mid-chirp (continues phase-continuously
    from the instantaneous frequency f0 r^s); a long chirp among 300 tones (leaf path); argument checks."""
    L = 2048
    N = 300
    rng = np.random.default_rng(77)
    rows = []
    for k in range(N):
        f0 = rng.uniform(20e6, 250e6)
        if k % 5 == 0:
            rows.append((f0, f0 * rng.uniform(0.8, 1.25), 1.0 / N, rng.uniform(0, 6.28), rng.uniform(0, 20e-6), rng.uniform(5e-6, 60e-6), EXP))
        elif k % 5 == 1:
            rows.append((f0, f0 + rng.uniform(-2e6, 2e6), 1.0 / N, rng.uniform(0, 6.28), -1e-3, 30e-3, MINJERK))
        else:
            rows.append((f0, f0, 1.0 / N, rng.uniform(0, 6.28), 0.0, 0.0, STATIC))
    rows[0] = (110e6, 95e6, 1.0 / N, 0.7, 2e-6, 40e-6, EXP)   # mid-chirp at chunk 4
    p, op = _pair(awg, FS, L, rows, eng)
    n_chunks = 16
    updates = {
        # chunk 4 = 14.6 us: tone 0 is mid-chirp; tone 2 was static; tone 5 goes from an exponential chirp to minimum jerk
        4: ([0, 2, 5], [rows[0][0] * 1.1, rows[2][0] * 0.9, rows[5][0] + 1e6], [30e-6, 20e-6, 8e-6], [EXP, EXP, MINJERK]),
        # chunk 9 = 32.9 us: tone 0 is mid-chirp again and jumps back; tone 10 restarts
        9: ([0, 10], [rows[0][0], rows[10][0] * 1.05], [0.0, 10e-6], [EXP, EXP]),
    }
    gotf, got = [], []
    for c in range(n_chunks):                                # the CUDA plan takes updates in stream order with the chunks
        if c in updates:
            p.update_trajectories(c, *updates[c])
            op.update_trajectories(c, *updates[c])
        gotf.append(_np(p.synthesize_chunk_f32(c)))
        got.append(_np(p.synthesize_chunk(c)))
    V = oracle.c_waveform(op, 0, n_chunks * L)
    assert_f32_close(np.concatenate(gotf), V, "exponential chirp updates")
    assert_codes_close(np.concatenate(got), op.quantise(V), "exponential chirp updates")
    c = 2000
    assert_f32_close(_np(p.synthesize_chunk_f32(c)), oracle.c_waveform(op, c * L, (c + 1) * L), "after the updates")
    # errors: a geometric path needs two frequencies of the same sign, away from zero
    with pytest.raises(awg.AwgError) as ei:
        p.update_trajectories(20, [3], [0.0], [1e-6], [EXP])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        p.update_trajectories(20, [3], [-5e6], [1e-6], [EXP])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    q = awg.Plan(2, FS, L)
    for f0, f1 in ((0.0, 1e6), (1e6, 0.0), (1e6, -2e6)):
        with pytest.raises(awg.AwgError) as ei:
            q.set_trajectories([f0, 2e6], [f1, 2e6], [0.1, 0.1], [0, 0], [0, 0], [1e-6, 0], [EXP, STATIC])
        assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        q.set_trajectories([1e6, 2e6], [1e6, 2e6], [0.1, 0.1], [0, 0], [0, 0], [1e-6, 0], [4, STATIC])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    p.close(); q.close()


def test_exponential_chirps_in_step_across_the_polynomial_classes(awg, torch_cuda, eng):
    """96 exponential chirps that start in step off the sample grid (all their start blocks fall into one tile) and end at 24
    different times, durations 1.5 us .. 400 us and frequency ratios 0.5 .. 2: every class of classify_exp (degree 2, 4, 6 and
    the fp64 fallback) and the edge series at both ends, equal phases so that the errors of the tones can add up."""
    fs, L = 560e6, 1 << 15
    t0 = 7.123456e-6
    durs = np.geomspace(1.5e-6, 400e-6, 24)
    ratios = (0.5, 0.93, 1.07, 2.0)
    rows = []
    for i, T in enumerate(durs):
        for j, r in enumerate(ratios):
            f0 = 40e6 + 2.1e6 * (4 * i + j)
            rows.append((f0, f0 * r, 1.0 / 96, 0.3, t0, float(T), EXP))
    p, op = _pair(awg, fs, L, rows, eng)
    n_chunks = 8                                            # 468 us: every chirp ends inside
    V = oracle.c_waveform(op, 0, n_chunks * L)
    gotf = np.concatenate([_np(p.synthesize_chunk_f32(c)) for c in range(n_chunks)])
    emax = assert_f32_close(gotf, V, "exponential chirps in step")
    got = np.concatenate([_np(p.synthesize_chunk(c)) for c in range(n_chunks)])
    assert_codes_close(got, op.quantise(V), "exponential chirps in step")
    assert np.array_equal(_np(p.synthesize_range(0, n_chunks)), got)
    print(f"exponential chirps in step: f32 max err {emax:.2e} of full scale")
    p.close()
