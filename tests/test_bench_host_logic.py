"""Host-side arithmetic of bench.py's roofline accounting (no GPU): which pipe binds, how the algorithmic operations
are turned into a fraction (DESIGN.md section 6 "Roofline": 1 multiply-add per static tone-sample, 1.25 inside a slow
move, 1 MUFU.SIN + 2 multiply-adds inside any other move).  The counts themselves come from the LIBRARY
(awg_plan_op_counts: the classification the kernel acts on); tests/test_gpu_parity.py::test_op_counts_* checks those
against the workload definitions on the GPU box."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import bench  # noqa: E402


def test_pipe_roofline_picks_the_binding_pipe_and_scales_with_time():
    sm_mhz = 1965.0
    fma_peak = 128 * 148 * sm_mhz * 1e6
    xu_peak = 16 * 148 * sm_mhz * 1e6
    # (static, slow, fast) tone-samples of a C2-like launch: ~1.4 % inside fast moves
    counts = (552_104_905, 0, 7_895_095)
    r = bench.pipe_roofline(counts, 0.05, "auto", sm_mhz)
    assert r["bound"] == "alu" and r["pipe"].startswith("FMA") and r["unit"] == "GFMA/s"
    assert r["fma_ops"] == counts[0] + 2 * counts[2] and r["mufu_ops"] == counts[2]
    assert np.isclose(r["frac"], (r["fma_ops"] / fma_peak) / 0.05e-3)
    assert np.isclose(r["achieved"] / r["peak"], r["frac"])
    assert np.isclose(bench.pipe_roofline(counts, 0.10, "auto", sm_mhz)["frac"], r["frac"] / 2)
    # every tone-sample through MUFU: the XU pipe binds (1 sine against 2 multiply-adds at an 8:1 peak ratio)
    total = sum(counts)
    rm = bench.pipe_roofline(counts, 0.2, "mufu", sm_mhz)
    assert rm["pipe"].startswith("XU") and rm["mufu_ops"] == total
    assert np.isclose(rm["frac"], (total / xu_peak) / 0.2e-3)
    # C3-like: every tone a slow mover for 19.6e6 of 19 922 944 samples: 1.25 multiply-adds each, no sine per sample
    slow = 1000 * 19_600_000
    sta = 1000 * 19_922_944 - slow
    r3 = bench.pipe_roofline((sta, slow, 0), 2.25, "auto", sm_mhz)
    assert r3["pipe"].startswith("FMA") and r3["mufu_ops"] == 0
    assert np.isclose(r3["frac"], (sta + 1.25 * slow) / fma_peak / 2.25e-3)
    # all fast movers: XU binds (1 / 16 per clock against 2 / 128)
    rf = bench.pipe_roofline((0, 0, 10 ** 9), 1.0, "auto", sm_mhz)
    assert rf["pipe"].startswith("XU") and np.isclose(rf["frac"], 1e9 / xu_peak / 1e-3)
    f = bench.frac_of((10 ** 9, 0, 0), 1.0, sm_mhz)
    assert f["pipe"] == "FMA" and np.isclose(f["roofline_frac"], 1e9 / fma_peak / 1e-3, atol=1e-4)
