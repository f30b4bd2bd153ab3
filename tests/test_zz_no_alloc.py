"""awg_synthesize_noalloc (include/awg.h): the one entry point that allocates nothing -- no plan, the trajectory table,
the tile scheduler's counters and the cross-CTA scratch tiles in one static __device__ array of the library.

Collected last on purpose (the suite runs with pytest -x).  The GPU test compares the entry point with the existing
path (a plan with the same trajectories) bit for bit -- the same kernels on the same table -- on calls in a row that
share the static array, and with the oracle at the bar of the other parity tests."""
import os
import re

import numpy as np
import pytest

import awg_workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
STATIC, LINEAR, MINJERK, EXP = W.PROFILE_STATIC, W.PROFILE_LINEAR, W.PROFILE_MINJERK, W.PROFILE_EXP
FS = 560e6


def _body(path, signature):
    """Text of the function that starts at `signature` (up to the closing brace in column 0)."""
    src = open(os.path.join(ROOT, path)).read()
    a = src.index(signature)
    return src[a:src.index("\n}\n", a)]


def test_the_no_alloc_path_calls_no_allocating_routine():
    """Host code of the entry point and of its launcher: no allocation, no stream or event creation; the static array's
    device address comes from cudaGetSymbolAddress (its name is not a device address in host code)."""
    entry = _body("paper_2403_15582_b200/csrc/awg_plan.cu", "awg_status awg_synthesize_noalloc(")
    launch = _body("paper_2403_15582_b200/csrc/awg_kernels.cu", "cudaError_t launch_synth_noalloc(")
    for text in (entry, launch):
        assert not re.search(r"cudaMalloc|cudaFree|cudaHostAlloc|cudaHostRegister|cudaStreamCreate|cudaEventCreate|\bnew\b|std::vector|device_state\(",
                             text)
    assert "launch_synth_noalloc(" in entry
    assert "cudaGetSymbolAddress(&ptr, g_noalloc_scratch)" in launch
    kern = open(os.path.join(ROOT, "paper_2403_15582_b200/csrc/awg_kernels.cu")).read()
    assert re.search(r"static __device__ __align__\(256\) unsigned char g_noalloc_scratch\[", kern)
    # the only uses of the name in host code: the declaration and the address lookup
    assert len(re.findall(r"\bg_noalloc_scratch\b", re.sub(r"//[^\n]*", "", kern))) == 2


def _rows_large(rng, n, span):
    """A tweezer-like table: static tones, slow and fast minimum-jerk moves, linear and exponential chirps, an instant retune."""
    rows = []
    for k in range(n):
        f0 = rng.uniform(20e6, 250e6)
        A, ph = rng.uniform(0.2, 1.0) / n, rng.uniform(0, 6.28)
        kind = k % 6
        if kind in (0, 1):
            rows.append((f0, f0, A, ph, 0.0, 0.0, STATIC))
        elif kind == 2:
            rows.append((f0, f0 + rng.uniform(-2e6, 2e6), A, ph, -1e-3, 30e-3, MINJERK))          # slow mover
        elif kind == 3:
            T = rng.uniform(0.1, 0.6) * span
            rows.append((f0, f0 + rng.uniform(-5e6, 5e6), A, ph, rng.uniform(0, span - T), T, MINJERK))   # fast mover
        elif kind == 4:
            rows.append((f0, f0 * rng.uniform(0.9, 1.1), A, ph, rng.uniform(0, 0.5 * span), rng.uniform(0.1, 0.5) * span, EXP))
        else:
            rows.append((f0, f0 + rng.uniform(-1e6, 1e6), A, ph, rng.uniform(0, span), rng.choice([0.0, 0.3 * span]), LINEAR))
    return list(zip(*rows))


def _plan_codes(awg, cols, first_sample, n_samples):
    """The existing path: a plan with 8-sample chunks, so that any range of whole 8-sample groups is a chunk range."""
    p = awg.Plan(len(cols[0]), FS, 8)
    p.set_trajectories(*cols)
    got = p.synthesize_range(first_sample // 8, n_samples // 8).cpu().numpy()
    p.close()
    return got


@pytest.mark.gpu
def test_no_alloc_entry_point_matches_the_plan_path_on_calls_in_a_row(awg):
    import torch
    import oracle
    from parity_util import assert_codes_close
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    rng = np.random.default_rng(2403)
    big = _rows_large(rng, 1000, 3 * (1 << 20) / FS)        # > 256 tones: leaves, quads of a tile on different CTAs (scratch tiles)
    small = _rows_large(rng, 40, 3 * (1 << 20) / FS)        # lean kernel, no scratch tiles; a shorter table than the call before
    calls = [
        (big, 1 << 20, 1 << 20),                            # the maximum size, tile-aligned
        (small, 3 * 2048 + 8, (1 << 18) - 16),              # ragged start and end inside tiles
        (big, (1 << 19) + 1000 * 8, 1 << 20),               # the maximum size from inside a tile: 513 tiles
        (big, 0, 4096),                                     # two tiles
    ]
    outs = [torch.full((n,), 12345, dtype=torch.int16, device="cuda") for _, _, n in calls]
    torch.cuda.synchronize()
    # the first pass also warms up module loading; free device memory must not move over the second pass
    for rep in range(2):
        free0 = torch.cuda.mem_get_info()[0]
        for (cols, first, n), out in zip(calls, outs):      # back to back on one stream, no synchronisation in between
            awg.synthesize_noalloc(FS, *cols, first, n, out)
        torch.cuda.synchronize()
        free1 = torch.cuda.mem_get_info()[0]
        got = [o.cpu().numpy().copy() for o in outs]
        for o in outs:
            o.fill_(-7)
        for i, ((cols, first, n), g) in enumerate(zip(calls, got)):
            want = _plan_codes(awg, cols, first, n)
            assert np.array_equal(g, want), f"pass {rep}, call {i}: {int(np.count_nonzero(g != want))} codes differ from the plan's"
        if rep == 1:
            assert free1 == free0, f"free device memory moved by {free0 - free1} bytes over four calls"
    # and against the oracle, at the bar of the parity tests (window of the third call)
    cols, first, n = calls[2]
    op = oracle.OraclePlan(len(cols[0]), FS, 8)
    op.set_trajectories(*cols)
    a = first + (1 << 19)
    V = oracle.c_waveform(op, a, a + 16384)
    assert_codes_close(got[2][a - first:a - first + 16384], op.quantise(V), "no-alloc entry point vs oracle")


@pytest.mark.gpu
def test_no_alloc_entry_point_rejects_sizes_beyond_its_static_scratch(awg):
    import torch
    out = torch.empty((1 << 20) + 8, dtype=torch.int16, device="cuda")
    n = 4097
    cols = [np.full(n, 1e8), np.full(n, 1e8), np.full(n, 1.0 / n), np.zeros(n), np.zeros(n), np.zeros(n), np.zeros(n, np.int32)]
    with pytest.raises(awg.AwgError) as ei:
        awg.synthesize_noalloc(FS, *cols, 0, 4096, out[:4096])
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG and "4096" in str(ei.value)
    cols = [c[:16] for c in cols]
    with pytest.raises(awg.AwgError) as ei:
        awg.synthesize_noalloc(FS, *cols, 0, (1 << 20) + 8, out)
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG and "1048576" in str(ei.value)
    for first, cnt in ((4, 4096), (0, 4100), (-8, 4096), (0, 0)):
        with pytest.raises(awg.AwgError) as ei:
            awg.awg_synthesize_noalloc(FS, 16, *cols, first, cnt, out.data_ptr())
        assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    with pytest.raises(awg.AwgError) as ei:
        awg.awg_synthesize_noalloc(FS, 16, *cols, 0, 4096, out.data_ptr() + 2)
    assert ei.value.status == awg.AWG_ERR_INVALID_ARG
    # a valid call still works after the rejected ones
    awg.synthesize_noalloc(FS, *cols, 0, 4096, out[:4096])
    torch.cuda.synchronize()
    assert np.array_equal(out[:4096].cpu().numpy(), _plan_codes(awg, cols, 0, 4096))
