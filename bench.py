#!/usr/bin/env python
"""bench.py -- headline benchmark of the additive-synthesis hot path on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-extras]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N ... bench.py --gpus N ...

One "step" = one pass of the whole hot path (trajectory table resident -> phase re-centring -> sine ->
accumulate -> quantise -> int16 stores) over BASELINE.json config 3, the largest single-GPU configuration: 1000 tones,
every one minimum-jerk chirping over 35 ms at 560 MS/s, 19 x 2^20 = 19 922 944 samples (the paper's Playback case,
PAPER.md:246), synthesised by ONE awg_synthesize_range launch into a 39.8 MB device buffer.  Metric: tone-samples/s (G).
Rank 0 prints ONE JSON line.

  value      device-timed (CUDA events on the launch stream), inputs resident in HBM
  e2e        the same workload through the C ABI with HOST buffers: awg_set_trajectories from host arrays
             (H2D upload of the tone cores) + awg_synthesize_range_host into pinned host memory (D2H of the int16 codes)
  roofline   ALU-bound ("bound": "alu"): a tone-sample needs one fp32 multiply-add where its tone is static (angle
             addition), two inside a slow move, one MUFU.SIN + two multiply-adds inside any other move -- counted by the
             LIBRARY (awg_plan_op_counts: the classification the kernel acts on); the pipe (FMA: 128/clk/SM, XU: 16/clk/SM,
             x 148 SMs x sm_max_mhz) whose roofline time is larger binds; frac = that time / measured launch time
  cpu_baseline  the oracle (oracle/awg_oracle_c.c, as it stands) on this box's host cores, bounded sample
  extras     the other configs (C1, C2, C4 at its 382 chunks, the 20 C5 cells), a fast-mover set (every tone inside a
             468 us minimum-jerk move all the time), the static-buffer pathway, four-channel multiplexing and the
             real-time capacity search -- every line with its fraction of the binding pipe

Multi-GPU (--gpus N under torchrun): the path shards by time with no exchange (every chunk is a pure
function of the absolute sample index), so each rank synthesises its own replica of the workload --
"replicas only", weak scaling, no data-path collective; NCCL is used for the barrier and the max-over-ranks
time only.  --impl reference times the oracle on the host cores (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

import awg_workloads as W  # noqa: E402

C3_DESC = ("C3: 1000 tones, every one minimum-jerk chirping over 35 ms at 560 MS/s, 19 x 2^20 = 19 922 944 samples, "
           "precomputed pathway (BASELINE.json configs[2], seed 2; the largest single-GPU configuration)")
METRIC = "tone-samples/s"
UNIT = "Gtone-samples/s"
MUFU_PER_CLK_PER_SM = 16  # sm_100: 4 SFU lanes per SM sub-partition (measured 15.9/clk/SM, profiles/)
FMA_PER_CLK_PER_SM = 128  # sm_100: 32 fp32 lanes per SM sub-partition (measured 127/clk/SM with FFMA2, profiles/)
N_SM = 148
L2_BYTES = 126 * (1 << 20)


def read_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index: int):
        self.samples = []  # (t, sm_mhz, reasons_bitmask)
        self.max_mhz = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = float(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _reasons(self):
        nv = self.nv
        for name in ("nvmlDeviceGetCurrentClocksEventReasons", "nvmlDeviceGetCurrentClocksThrottleReasons"):
            fn = getattr(nv, name, None)
            if fn is not None:
                try:
                    return int(fn(self.h))
                except Exception:
                    pass
        return 0

    def _run(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                mhz = float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                self.samples.append((time.perf_counter(), mhz, self._reasons()))
            except Exception:
                pass
            time.sleep(0.002)

    def start(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._run, daemon=True)
            self._thr.start()

    def stop(self):
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=1.0)

    def summary(self, t0: float, t1: float):
        if self.nv is None or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml_unavailable"]}
        inside = [s for s in self.samples if t0 <= s[0] <= t1]
        if not inside:  # region shorter than the sampling period: take the nearest sample
            inside = [min(self.samples, key=lambda s: abs(s[0] - 0.5 * (t0 + t1)))]
        mask = 0
        for s in inside:
            mask |= s[2]
        names = {0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
                 0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown",
                 0x80: "hw_power_brake_slowdown", 0x100: "display_clock_setting"}
        reasons = [n for b, n in names.items() if mask & b and n != "gpu_idle"]
        return {"sm_mhz": float(np.median([s[1] for s in inside])), "sm_max_mhz": self.max_mhz,
                "reasons": reasons, "samples": len(inside)}


# --------------------------------------------------------------------------------------------------
def max_over_ranks(x: float, dist, device) -> float:
    """MAX all-reduce of a scalar over the ranks (identity when dist is None)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_per_step: int, steps: int, world: int, seconds_max_over_ranks: float) -> float:
    """Aggregate units/s of N independent replicas: every rank does the same work, the slowest rank sets the time."""
    return world * units_per_rank_per_step * steps / seconds_max_over_ranks


def oracle_rate(w, n_samples: int, repeats: int = 1):
    """tone-samples/s of the C oracle on the first n_samples of workload w, all host cores."""
    import oracle
    op = oracle.plan_from_workload(w)
    n_samples = min(n_samples, w.n_samples)
    oracle.c_waveform(op, 0, 4096)  # build + page in
    best = None
    for _ in range(repeats):
        t = time.perf_counter()
        V = oracle.c_waveform(op, 0, n_samples)
        op.quantise(V)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return w.n_tones * n_samples / best, oracle.c_num_threads(), best


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores; each step a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    w = W.config3()
    op = oracle.plan_from_workload(w)
    # warm-up doubles as a rate probe: size the per-step sample so that the K steps end within ~2 minutes
    t0 = time.perf_counter()
    for _ in range(max(1, args.warmup)):
        oracle.c_waveform(op, 0, 1 << 14)
    rate = max(1, args.warmup) * (1 << 14) * w.n_tones / (time.perf_counter() - t0)
    n = int(min(1 << 20, max(4096, rate * 120.0 / args.steps / w.n_tones)))
    n -= n % 4096
    t0 = time.perf_counter()
    for _ in range(args.steps):
        op.quantise(oracle.c_waveform(op, 0, n))
    dt = time.perf_counter() - t0
    val = w.n_tones * n * args.steps / dt / 1e9
    cores = oracle.c_num_threads()
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": C3_DESC, "sample": f"first {n} of {w.n_samples} samples per step"},
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": f"first {n} samples x {w.n_tones} tones of C3 per step, {args.steps} steps"},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


SLOW_FMA_PER_TONE_SAMPLE = 1.25   # (16 table-correction + 64 accumulate) multiply-adds per 64 tone-samples of a thread


def pipe_roofline(counts, ms, engine, sm_mhz):
    """Binding ALU roofline of launches that took `ms` in total over `counts` = (static, slow, fast) tone-samples as the
    LIBRARY classifies them (awg_plan_op_counts).

    Algorithmic work: a tone-sample of a tone that is static there needs ONE fp32 multiply-add (angle addition over a
    symmetric sample pair); inside a slow move 1.25 multiply-adds (16 to move the tone's 16 pair-table entries to the thread's
    local frequency + 64 for the thread's 64 samples);
    inside any other move one MUFU.SIN plus two multiply-adds (range multiply, amplitude accumulate).  With
    --engine mufu every tone-sample takes the MUFU path.  The roofline time is the larger of (multiply-adds / FMA-pipe
    peak) and (sines / XU-pipe peak) at sm_mhz; frac = that time / the measured time."""
    n_sta, n_slow, n_fast = (int(x) for x in counts)
    if engine == "mufu":
        n_sta, n_slow, n_fast = 0, 0, n_sta + n_slow + n_fast
    fma_ops, xu_ops = n_sta + SLOW_FMA_PER_TONE_SAMPLE * n_slow + 2 * n_fast, n_fast
    peak_fma = FMA_PER_CLK_PER_SM * N_SM * sm_mhz * 1e6
    peak_xu = MUFU_PER_CLK_PER_SM * N_SM * sm_mhz * 1e6
    t_fma, t_xu = fma_ops / peak_fma, xu_ops / peak_xu
    t = ms * 1e-3
    if t_fma >= t_xu:
        pipe, ops, peak, unit = "FMA (fp32 multiply-add)", fma_ops, peak_fma, "GFMA/s"
    else:
        pipe, ops, peak, unit = "XU (MUFU.SIN)", xu_ops, peak_xu, "Gsin/s"
    return {"bound": "alu", "pipe": pipe, "achieved": ops / t / 1e9, "peak": peak / 1e9, "unit": unit,
            "frac": max(t_fma, t_xu) / t, "static_tone_samples": n_sta, "moving_tone_samples": n_slow + n_fast,
            "slow_moving_tone_samples": n_slow, "fma_ops": int(fma_ops), "mufu_ops": int(xu_ops),
            "t_fma_us": t_fma * 1e6, "t_xu_us": t_xu * 1e6}


def frac_of(counts, ms, sm_mhz, engine="auto"):
    r = pipe_roofline(counts, ms, engine, sm_mhz)
    return {"roofline_frac": round(r["frac"], 4), "pipe": r["pipe"].split()[0]}


ENGINES = {"auto": lambda awg: awg.AWG_ENGINE_AUTO, "fma": lambda awg: awg.AWG_ENGINE_FMA,
           "mufu": lambda awg: awg.AWG_ENGINE_MUFU}


def pick_workload(name: str):
    """The timed workload: C3 (the headline: the largest single-GPU configuration, BASELINE.json configs[2]) unless
    --workload asks for another one (profiling aid: C1, C2, C5:<tones>:<log2 chunk>, CAP:<static|half|moving>:<tones>)."""
    if name == "C2":
        return W.config2(), ("C2: 100 tones at 560 MS/s for 10 ms = 5.6 M samples, 50 min-jerk movers "
                             "(BASELINE.json configs[1], seed 1)")
    if name == "C1":
        return W.config1(), "C1: 16 tones, 2^20 samples (BASELINE.json configs[0])"
    if name == "C3":
        return W.config3(), C3_DESC
    kind, *rest = name.split(":")
    if kind == "C5":
        n_t, lg = int(rest[0]), int(rest[1])
        return W.config5_cell(n_t, 1 << lg), f"C5 cell: {n_t} tones x 2^{lg} samples (BASELINE.json configs[4])"
    if kind == "CAP":
        n_t = int(rest[1])
        return (W.capacity_toneset(n_t, 560e6, 1 << 20, rest[0], n_chunks=4),
                f"capacity tone set: {n_t} tones ({rest[0]}), 4 x 2^20 samples at 560 MS/s")
    raise SystemExit(f"unknown --workload {name}")


# --------------------------------------------------------------------------------------------------
def device_time_range(torch, plan, n_chunks, bufs, steps, warmup, prequeue_ms=0.0):
    """ms per step of awg_synthesize_range, CUDA events on the launch stream, rotating output buffers.

    prequeue_ms > 0: the timed launches are queued behind a spin kernel of about that length (torch.cuda._sleep), so the
    host has submitted all of them before the first one starts and the events bracket back-to-back DEVICE execution; used
    for launches of a few microseconds, where a Python call (~10 us) would otherwise be what the events time."""
    stream = torch.cuda.current_stream()
    for i in range(warmup):
        plan.synthesize_range(0, n_chunks, out=bufs[i % len(bufs)], stream=stream)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    if prequeue_ms > 0.0:
        torch.cuda._sleep(int(prequeue_ms * 1e-3 * 1.9e9))
    a.record(stream)
    for i in range(steps):
        plan.synthesize_range(0, n_chunks, out=bufs[i % len(bufs)], stream=stream)
    b.record(stream)
    b.synchronize()
    return a.elapsed_time(b) / steps


def make_bufs(torch, n_samples):
    n_buf = max(2, -(-int(1.06 * L2_BYTES) // (2 * n_samples)))
    return [torch.empty(n_samples, dtype=torch.int16, device="cuda") for _ in range(n_buf)]


def stream_through_ring(awg, w, host_mirror, n_chunks=None, n_slots=4):
    """Runs workload w (with its per-chunk updates) through the ring as fast as it goes; the ring's virtual DAC consumes
    one chunk per chunk_len/fs and counts the chunks that were not complete when due.
    Returns (underruns, max_chunk_ms, wall_s, chunks)."""
    p = awg.Plan.from_workload(w)
    ring = awg.Ring(p, n_slots=n_slots, host_mirror=host_mirror)
    ups = w.updates_by_chunk()
    n_chunks = n_chunks or w.n_chunks
    depth = n_slots - 1
    t0 = time.perf_counter()
    for c in range(n_chunks + depth):
        if c < n_chunks:
            ring.submit(c, ups.get(c))
        if c >= depth:
            idx, _, _, _ = ring.acquire()
            ring.release(idx)
    wall = time.perf_counter() - t0
    produced, underruns, max_ms = ring.stats()
    ring.close()
    p.close()
    return underruns, max_ms, wall, produced


def device_time_chunks(torch, awg, w, n_chunks=None):
    """Device time (ms, CUDA events around every synthesis launch, table uploads outside) of the chunks of a workload with
    per-chunk updates, and the library's operation counts summed over the chunks."""
    p = awg.Plan.from_workload(w)
    ups = w.updates_by_chunk()
    n_chunks = n_chunks or w.n_chunks
    out = [torch.empty(w.chunk_len, dtype=torch.int16, device="cuda") for _ in range(4)]
    stream = torch.cuda.current_stream()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(n_chunks)]
    counts = [0, 0, 0]
    warm = torch.empty(w.chunk_len, dtype=torch.float32, device="cuda")
    for c in range(n_chunks):
        if c in ups:
            u = ups[c]
            p.update_trajectories(c, u.tone_idx, u.f1, u.t_dur, u.profile)
            p.synthesize_chunk_f32(c, out=warm, stream=stream)   # carries the table upload; not timed
        for i, v in enumerate(p.op_counts(c, 1)):
            counts[i] += v
        evs[c][0].record(stream)
        p.synthesize_chunk(c, out=out[c % 4], stream=stream)
        evs[c][1].record(stream)
    torch.cuda.synchronize()
    ms = [a.elapsed_time(b) for a, b in evs]
    p.close()
    return sum(ms), max(ms), counts


def realtime_capacity(awg, make_workload, host_mirror, lo=16, hi=65536):
    """Largest tone count that streams in real time: bisection on N; a probe streams >= 1 s of signal
    through the ring (3 slots) and is sustained when the ring's own underrun counter stays at zero."""
    def ok(n):
        w = make_workload(n)
        und, _, _, _ = stream_through_ring(awg, w, host_mirror, n_slots=3)
        return und == 0

    good, bad = None, None
    n = lo
    while n <= hi:  # exponential search for the first failing count
        if ok(n):
            good = n
            n *= 2
        else:
            bad = n
            break
    if good is None:
        return 0
    if bad is None:
        return good
    while bad - good > max(8, good // 32):
        mid = (good + bad) // 2
        if ok(mid):
            good = mid
        else:
            bad = mid
    return good


def fast_mover_capacity(torch, awg, fs, chunk_len, lo=16, hi=65536):
    """Largest count of tones that are ALL inside short minimum-jerk moves all the time (W.fast_mover_stream) whose
    every chunk is synthesised within chunk_len/fs of device time.  (The criterion here is the device time of the synthesis
    launches alone; fast_mover_ring_capacity() streams the same set through the ring, host planning included.)"""
    deadline_ms = chunk_len / fs * 1e3

    def ok(n):
        _, worst, _ = device_time_chunks(torch, awg, W.fast_mover_stream(n, fs, chunk_len, 6))
        return worst <= deadline_ms

    good, bad, n = None, None, lo
    while n <= hi:
        if ok(n):
            good, n = n, n * 2
        else:
            bad = n
            break
    if good is None:
        return 0
    if bad is None:
        return good
    while bad - good > max(8, good // 32):
        mid = (good + bad) // 2
        if ok(mid):
            good = mid
        else:
            bad = mid
    return good


def fast_mover_ring_capacity(awg, fs, chunk_len, seconds=1.0, lo=256, hi=8192):
    """Largest all-fast-mover count (W.fast_mover_stream) the RING sustains: its own underrun counter stays at zero over
    `seconds` of signal while, every chunk, the host re-plans every tone (awg_ring_submit with N updates), uploads the table
    and launches.  Beside the device-time figure: this one includes the host."""
    n_chunks = int(math.ceil(seconds * fs / chunk_len))

    def ok(n):
        und, _, _, _ = stream_through_ring(awg, W.fast_mover_stream(n, fs, chunk_len, n_chunks), False, n_slots=4)
        return und == 0

    good, bad, n = None, None, lo
    while n <= hi:
        if ok(n):
            good, n = n, n * 2
        else:
            bad = n
            break
    if good is None:
        return 0
    if bad is None:
        return good
    while bad - good > max(64, good // 16):
        mid = (good + bad) // 2
        if ok(mid):
            good = mid
        else:
            bad = mid
    return good


def run_extras(torch, awg, sm_max_mhz):
    out = {}
    # ---- per-config device throughput (range launch for C1/C2, per-cell chunk launch for C5), each with its fraction
    cfgs = {}
    for name, w in (("C1", W.config1()), ("C2", W.config2())):
        p = awg.Plan.from_workload(w)
        bufs = make_bufs(torch, w.n_samples)
        ms_host = device_time_range(torch, p, w.n_chunks, bufs, 50, 5)
        ms = device_time_range(torch, p, w.n_chunks, bufs, 50, 5, prequeue_ms=3.0)
        cfgs[name] = {"tones": w.n_tones, "samples": w.n_samples, "ms": ms, "ms_host_paced": ms_host, "gts_per_s": w.tone_samples / ms / 1e6,
                      "out_MS_per_s": w.n_samples / ms / 1e3, **frac_of(p.op_counts(0, w.n_chunks), ms, sm_max_mhz)}
        del bufs
        p.close()
    # ---- C4 at its stated length: 382 chunks = 1 s at 100 MS/s, 7 258 moves
    w4 = W.config4(382)
    ms4, worst4, counts4 = device_time_chunks(torch, awg, w4)
    cfgs["C4_device"] = {"tones": w4.n_tones, "chunks": w4.n_chunks, "ms_total": ms4, "max_chunk_ms": worst4,
                         "gts_per_s": w4.tone_samples / ms4 / 1e6, **frac_of(counts4, ms4, sm_max_mhz)}
    for mirror in (False, True):
        und, max_ms, wall, produced = stream_through_ring(awg, w4, mirror)
        cfgs["C4_ring" + ("_d2h" if mirror else "")] = {
            "tones": w4.n_tones, "chunks": produced, "underruns": und, "max_chunk_ms": max_ms,
            "deadline_ms": w4.chunk_len / w4.sample_rate * 1e3, "wall_s": wall,
            "gts_per_s": w4.n_tones * w4.chunk_len * produced / wall / 1e9,
            "realtime_margin": (w4.chunk_len / w4.sample_rate) / (wall / produced),
            "roofline_frac": cfgs["C4_device"]["roofline_frac"], "pipe": cfgs["C4_device"]["pipe"],
            "frac_note": "fraction of the synthesis launches (C4_device); the ring adds host-side update planning and table uploads"}
    # ---- fast movers: every tone inside a 468 us minimum-jerk move all the time (the MUFU pass)
    wf = W.fast_mover_stream(4096, 560e6, 1 << 18, 8)
    msf, worstf, countsf = device_time_chunks(torch, awg, wf)
    cfgs["FAST_4096"] = {"tones": wf.n_tones, "chunks": wf.n_chunks, "ms_total": msf, "max_chunk_ms": worstf,
                         "gts_per_s": wf.tone_samples / msf / 1e6, **frac_of(countsf, msf, sm_max_mhz)}
    # ---- exponential chirps (PAPER.md:137 names them; G20): 1024 tones, each 3 % up in frequency over 300 us
    # inside one 2^18-sample chunk (they start and end in step: both edge blocks of every tone fall into one tile each)
    rngx = np.random.default_rng(11)
    fx = rngx.uniform(30e6, 240e6, 1024)
    p = awg.Plan(1024, 560e6, 1 << 18)
    p.set_trajectories(fx, fx * 1.03, np.full(1024, 1.0 / 1024), rngx.uniform(0, 6.28, 1024), np.full(1024, 20e-6), np.full(1024, 300e-6),
                       np.full(1024, W.PROFILE_EXP, np.int32))
    bufs = make_bufs(torch, 1 << 18)
    ms = device_time_range(torch, p, 1, bufs, 20, 3, prequeue_ms=1.0)
    cfgs["EXP_1024"] = {"tones": 1024, "samples": 1 << 18, "ms": ms, "gts_per_s": 1024 * (1 << 18) / ms / 1e6,
                        **frac_of(p.op_counts(0, 1), ms, sm_max_mhz)}
    del bufs
    p.close()
    # ---- static set (the paper's comb), per-sample and through the looped static buffer
    ws = W.capacity_toneset(4096, 560e6, 1 << 20, "static", n_chunks=4)
    p = awg.Plan.from_workload(ws)
    bufs = make_bufs(torch, ws.n_samples)
    ms = device_time_range(torch, p, ws.n_chunks, bufs, 10, 3)
    cfgs["STATIC_4096"] = {"tones": ws.n_tones, "samples": ws.n_samples, "ms": ms, "gts_per_s": ws.tone_samples / ms / 1e6,
                           **frac_of(p.op_counts(0, ws.n_chunks), ms, sm_max_mhz)}
    del bufs
    p.close()
    # static-buffer pathway (NEXT-3): 4096 tones snapped to the fs/L_s grid live in X_static, 64 movers are evaluated
    L = 1 << 20
    rng = np.random.default_rng(9)
    fsn = [awg.awg_snap_frequency(float(f), 560e6, L) for f in rng.uniform(30e6, 250e6, 4096)]
    f0 = np.concatenate([fsn, rng.uniform(30e6, 250e6, 64)])
    n = f0.shape[0]
    prof = np.zeros(n, np.int32); prof[4096:] = W.PROFILE_MINJERK
    f1 = f0.copy(); f1[4096:] += 5e6
    tdur = np.zeros(n); tdur[4096:] = 300e-6
    p = awg.Plan(n, 560e6, L)
    p.set_trajectories(f0, f1, np.full(n, 1.0 / n), rng.uniform(0, 6.28, n), np.zeros(n), tdur, prof)
    p.static_buffer_set(np.arange(4096))
    bufs = make_bufs(torch, 4 * L)
    ms = device_time_range(torch, p, 4, bufs, 20, 3)
    cfgs["STATIC_BUFFER_4096+64"] = {
        "tones": n, "tones_per_sample": 64, "samples": 4 * L, "ms": ms, "effective_gts_per_s": n * 4 * L / ms / 1e6,
        **frac_of(p.op_counts(0, 4), ms, sm_max_mhz),
        "note": "4096 on-grid static tones come from the looped X_static (Eq. 9); the fraction counts the 64 evaluated tones only"}
    del bufs
    p.close()
    # four-channel multiplexing (NEXT-2): the paper's chunk, 4 x 2^18 samples, 20 tones per channel
    Lm = 1 << 18
    plans = [awg.Plan.from_workload(W.config5_cell(20, Lm)) for _ in range(4)]
    outm = [torch.empty(4 * Lm, dtype=torch.int16, device="cuda") for _ in range(32)]
    stream = torch.cuda.current_stream()
    for i in range(5):
        awg.synthesize_chunk_mux(plans, 0, out=outm[i], stream=stream)
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    torch.cuda._sleep(int(3e-3 * 1.9e9))   # queue pre-filled behind a 3 ms spin: the events time the device, not the Python caller
    a.record(stream)
    for i in range(32):
        awg.synthesize_chunk_mux(plans, 0, out=outm[i], stream=stream)
    b.record(stream)
    b.synchronize()
    ms = a.elapsed_time(b) / 32
    cm = [sum(x) for x in zip(*[pl.op_counts(0, 1) for pl in plans])]
    cfgs["MUX4_20x4"] = {"tones_per_channel": 20, "samples_per_channel": Lm, "ms": ms, "gts_per_s": 80 * Lm / ms / 1e6,
                         "out_MS_per_s_per_channel": Lm / ms / 1e3, "deadline_ms": Lm / 560e6 * 1e3, **frac_of(cm, ms, sm_max_mhz)}
    for pl in plans:
        pl.close()
    out["configs"] = cfgs
    # ---- C5: all 20 cells.  us = device time per launch with the queue pre-filled (launches of a few microseconds are
    # otherwise paced by the Python caller); us_host_paced = the same launches submitted back to back from Python
    sweep = {}
    for n_t, cl in W.config5_grid():
        w = W.config5_cell(n_t, cl)
        p = awg.Plan.from_workload(w)
        bufs = make_bufs(torch, cl)
        ms_host = device_time_range(torch, p, 1, bufs, 20, 3)
        ms = device_time_range(torch, p, 1, bufs, 40, 3, prequeue_ms=max(1.0, 40 * 0.03))
        sweep[f"N{n_t}_L{cl.bit_length() - 1}"] = {"gts_per_s": round(w.tone_samples / ms / 1e6, 2), "us": round(ms * 1e3, 2),
                                                   "us_host_paced": round(ms_host * 1e3, 2),
                                                   **frac_of(p.op_counts(0, 1), ms, sm_max_mhz)}
        del bufs
        p.close()
    out["C5"] = sweep
    # ---- real-time capacity: ring underruns == 0 over >= 1 s of signal
    cap = {}
    for fs, cl, tag in ((560e6, 1 << 20, "560MS"), (100e6, 1 << 18, "100MS")):
        n_chunks = int(math.ceil(1.0 * fs / cl))
        for mix, key in (("static", "static"), ("half", "half_static_half_fast"), ("moving", "all_slow_movers")):
            mk = (lambda n, fs=fs, cl=cl, mix=mix, n_chunks=n_chunks: W.capacity_toneset(n, fs, cl, mix, n_chunks=n_chunks))
            cap[f"{tag}_{key}"] = realtime_capacity(awg, mk, False)
        cap[f"{tag}_static_d2h"] = realtime_capacity(awg, (lambda n, fs=fs, cl=cl, n_chunks=n_chunks:
                                                           W.capacity_toneset(n, fs, cl, "static", n_chunks=n_chunks)), True)
    # short chunks (2^18 samples = 468 us at 560 MS/s: 128 tiles per launch, fewer than the grid has CTAs): the launches spread a
    # tile's tone quads over CTAs
    n18 = int(math.ceil(0.5 * 560e6 / (1 << 18)))
    cap["560MS_static_L18_chunks"] = realtime_capacity(awg, (lambda n: W.capacity_toneset(n, 560e6, 1 << 18, "static", n_chunks=n18)), False)
    cap["560MS_all_fast_movers_device_time"] = fast_mover_capacity(torch, awg, 560e6, 1 << 18)
    cap["100MS_all_fast_movers_device_time"] = fast_mover_capacity(torch, awg, 100e6, 1 << 15)
    cap["560MS_all_fast_movers_ring"] = fast_mover_ring_capacity(awg, 560e6, 1 << 18)
    out["max_realtime_tones"] = cap
    # fraction of the binding roofline AT each capacity: roofline time of one chunk of the N_max-tone set / the chunk's deadline
    def cap_frac(n, make, fs, cl, chunk=1):
        if not n:
            return None
        pl = awg.Plan.from_workload(make(n))
        r = pipe_roofline(pl.op_counts(chunk, 1), cl / fs * 1e3, "auto", sm_max_mhz)
        pl.close()
        return {"roofline_frac": round(r["frac"], 4), "pipe": r["pipe"].split()[0]}

    capf = {}
    for fs, cl, tag in ((560e6, 1 << 20, "560MS"), (100e6, 1 << 18, "100MS")):
        n_chunks = int(math.ceil(1.0 * fs / cl))   # the same tone sets as in the search (the slow movers' move spans the probe)
        for mix, key in (("static", "static"), ("half", "half_static_half_fast"), ("moving", "all_slow_movers"), ("static", "static_d2h")):
            capf[f"{tag}_{key}"] = cap_frac(cap[f"{tag}_{key}"], (lambda n, fs=fs, cl=cl, mix=mix, n_chunks=n_chunks:
                                                                  W.capacity_toneset(n, fs, cl, mix, n_chunks=n_chunks)), fs, cl, chunk=n_chunks // 2)
    capf["560MS_static_L18_chunks"] = cap_frac(cap["560MS_static_L18_chunks"], (lambda n: W.capacity_toneset(n, 560e6, 1 << 18, "static", n_chunks=4)), 560e6, 1 << 18)
    for fs, cl, key in ((560e6, 1 << 18, "560MS_all_fast_movers_device_time"), (100e6, 1 << 15, "100MS_all_fast_movers_device_time"),
                        (560e6, 1 << 18, "560MS_all_fast_movers_ring")):
        n = cap[key]
        if n:   # every tone-sample of such a set is inside a move: one sine each
            r = pipe_roofline((0, 0, n * cl), cl / fs * 1e3, "auto", sm_max_mhz)
            capf[key] = {"roofline_frac": round(r["frac"], 4), "pipe": r["pipe"].split()[0]}
    out["max_realtime_tones_roofline"] = capf
    out["max_realtime_tones_note"] = (
        "largest N streamed through the ring (3 slots) for >= 1 s of signal with the ring's underrun counter at zero; tone sets "
        "drawn like C5 (2^20-sample chunks at 560 MS/s, 2^18 at 100 MS/s; '_L18_chunks': 2^18-sample chunks at 560 MS/s over 0.5 s); 'all_slow_movers' = one +-5 MHz minimum-jerk move "
        "spanning the probe (the slow pass); '_d2h' = pinned-host mirror on; 'all_fast_movers_device_time' = every tone "
        "inside a one-chunk minimum-jerk move all the time (2^18-sample chunks = 468 us at 560 MS/s, 2^15 = 328 us at "
        "100 MS/s), criterion: every chunk's synthesis within chunk_len/fs of device time; 'all_fast_movers_ring' = the same "
        "set through the ring (4 slots, >= 1 s, underruns == 0): the host re-plans every tone every chunk (threaded from 2048 tones)")
    # ---- the paper's two scaling laws, re-fitted on this GPU (context, not a target)
    laws = {}
    # Eq. 12: N_streaming = (P / fs)^(1 / (1 - k)), N_streaming = tones that can be chirped indefinitely
    # (all fast movers, 2^18-sample chunks, device-time criterion) at sampling rate fs
    pts = []
    for fs in (280e6, 400e6, 560e6, 800e6, 1120e6):
        n = fast_mover_capacity(torch, awg, fs, 1 << 18)
        if n:
            pts.append((fs, n))
    if len(pts) >= 3:
        x, y = np.log([p_[0] for p_ in pts]), np.log([p_[1] for p_ in pts])
        m, c = np.polyfit(x, y, 1)                      # log N = m log fs + c,  m = -1 / (1 - k)
        k = 1.0 + 1.0 / m
        r2 = 1.0 - float(np.sum((y - (m * x + c)) ** 2) / np.sum((y - y.mean()) ** 2))
        laws["eq12_streaming"] = {"points_fs_N": [[p_[0], int(p_[1])] for p_ in pts], "k": float(k),
                                  "P_tone_samples_per_s": float(math.exp(c * (1.0 - k))), "r2": r2,
                                  "paper": {"k": 0.249, "r2": 0.9997, "hardware": "Quadro RTX 6000"},
                                  "note": "k = 0: time per chunk proportional to the tone count (compute-bound); the paper's k = 0.249 "
                                          "reflects latency hiding improving with the tone count on its hardware"}
    # Eq. 13: tau_playback = A (T fs)^a N^b (+ t_overhead N): wall-clock latency from the trajectory arrays to
    # the complete waveform in device memory (awg_set_trajectories + awg_synthesize_range + synchronize), every tone one
    # minimum-jerk move over the whole waveform
    rows = []
    for n_t in (100, 400, 1000, 4000):
        for lg in (20, 22, 24):
            w = W.capacity_toneset(n_t, 560e6, 1 << lg, "moving", n_chunks=1)
            pl = awg.Plan(w.n_tones, w.sample_rate, w.chunk_len)
            buf = torch.empty(1 << lg, dtype=torch.int16, device="cuda")
            traj = (w.f0, w.f1, w.A, w.phi0, w.t_start, w.t_dur, w.profile)
            best = float("inf")
            for _ in range(4):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                pl.set_trajectories(*traj)
                pl.synthesize_range(0, 1, out=buf)
                torch.cuda.synchronize()
                best = min(best, time.perf_counter() - t0)
            pl.close()
            del buf
            rows.append((n_t, 1 << lg, best))
    X = np.array([[1.0, math.log(r[1]), math.log(r[0])] for r in rows])
    yv = np.log([r[2] for r in rows])
    coef, *_ = np.linalg.lstsq(X, yv, rcond=None)
    r2 = 1.0 - float(np.sum((yv - X @ coef) ** 2) / np.sum((yv - yv.mean()) ** 2))
    laws["eq13_playback"] = {"points_N_samples_seconds": [[r[0], r[1], r[2]] for r in rows], "A_seconds": float(math.exp(coef[0])),
                             "a": float(coef[1]), "b": float(coef[2]), "r2": r2,
                             "paper": {"a_b": "both sub-linear, values only in its Fig. 10", "r2": 0.997},
                             "note": "log-linear least squares without the t_overhead N term"}
    out["paper_scaling_laws_on_b200"] = laws
    out["paper_context"] = {"hardware": "Quadro RTX 6000 + PCIe 2.0 DAC (PAPER.md:69)", "streaming_tones_560MS": 20,
                            "streaming_tones_100MS": 194, "playback_tones_35ms_560MS": 1000,
                            "static_fp32_gts_per_s": 79.4}
    return out


def run_ours(args):
    import torch
    import paper_2403_15582_b200 as awg

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    peaks, peaks_src = read_peaks()
    sm_max_mhz = float(peaks.get("sm_max_mhz", 1965.0))

    w, w_desc = pick_workload(args.workload)
    plan = awg.Plan.from_workload(w, engine=ENGINES[args.engine](awg))
    bufs = make_bufs(torch, w.n_samples)
    stream = torch.cuda.current_stream()
    host_out = torch.empty(w.n_samples, dtype=torch.int16, pin_memory=True)
    traj = (w.f0, w.f1, w.A, w.phi0, w.t_start, w.t_dur, w.profile)

    # ---- device-timed value -------------------------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    for i in range(max(3, args.warmup)):
        plan.synthesize_range(0, w.n_chunks, out=bufs[i % len(bufs)], stream=stream)
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    launches0 = awg.awg_kernel_launch_count()
    t_host0 = time.perf_counter()
    ev0.record(stream)
    for i in range(args.steps):
        plan.synthesize_range(0, w.n_chunks, out=bufs[i % len(bufs)], stream=stream)
    ev1.record(stream)
    barrier()
    t_host1 = time.perf_counter()
    launches = awg.awg_kernel_launch_count() - launches0
    ms_total = ev0.elapsed_time(ev1)
    sampler.stop()
    clocks = sampler.summary(t_host0, t_host1)
    ms_total_max = max_over_ranks(ms_total, dist, "cuda")
    ms_per_step = ms_total_max / args.steps
    value = whole_job_rate(w.tone_samples, args.steps, world, ms_total_max * 1e-3) / 1e9

    # ---- end to end through the C ABI with host buffers -----------------------------------------
    for _ in range(2):
        plan.set_trajectories(*traj)
        plan.synthesize_range_host(0, w.n_chunks, out=host_out)
    io0 = plan.io_bytes()
    e2e_steps = max(3, min(args.steps, 50))
    barrier()
    t0 = time.perf_counter()
    for _ in range(e2e_steps):
        plan.set_trajectories(*traj)                                  # host arrays -> table -> H2D upload
        plan.synthesize_range_host(0, w.n_chunks, out=host_out)       # synthesis + D2H of every int16 code
    torch.cuda.synchronize()
    dt = time.perf_counter() - t0
    io1 = plan.io_bytes()
    dt_max = max_over_ranks(dt, dist, "cuda")
    e2e_value = whole_job_rate(w.tone_samples, e2e_steps, world, dt_max) / 1e9
    e2e = {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": (io1[0] - io0[0]) // e2e_steps,
           "d2h_bytes_per_step": (io1[1] - io0[1]) // e2e_steps, "steps": e2e_steps,
           "ms_per_step": dt_max / e2e_steps * 1e3,
           "what": "awg_set_trajectories(host arrays) + awg_synthesize_range_host(pinned host int16)"}

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant (only) kernel ---------------------------------------------------
    ms_local = ms_total / args.steps
    traffic = None
    try:
        with open(os.path.join(ROOT, "profiles", "traffic.json")) as f:
            traffic = json.load(f).get("awg_synth_kernel_C3_dram_bytes_per_launch")
    except Exception:
        pass
    counts = plan.op_counts(0, w.n_chunks)
    roofline = pipe_roofline(counts, ms_local, args.engine, sm_max_mhz)
    roofline.update({
        "traffic": traffic,
        "peak_how": f"{FMA_PER_CLK_PER_SM} FMA (or {MUFU_PER_CLK_PER_SM} MUFU) /clk/SM x {N_SM} SMs x {sm_max_mhz:.0f} MHz "
                    f"(sm_max_mhz of MEASURED_PEAKS.json, {peaks_src}); the pipe whose roofline time is larger binds",
        "kernel": "awg_synth_kernel", "launch_ms": ms_local,
        "hbm": {"algorithmic_bytes_per_launch": 2 * w.n_samples, "achieved_gbs": 2 * w.n_samples / (ms_local * 1e-3) / 1e9,
                "peak_gbs": peaks.get("hbm_gbs"), "frac": 2 * w.n_samples / (ms_local * 1e-3) / 1e9 / float(peaks.get("hbm_gbs", 6650.0))},
    })
    if clocks.get("sm_mhz"):
        roofline["frac_at_achieved_clock"] = pipe_roofline(counts, ms_local, args.engine, clocks["sm_mhz"])["frac"]
    if args.engine != "mufu" and counts[1] > 0:
        # continuity with round 1, whose slow pass needed (and whose bench counted) 2 multiply-adds per slow tone-sample
        n_sta, n_slow, n_fast = (int(x) for x in counts)
        roofline["frac_if_slow_tone_samples_counted_as_2_fma"] = (
            (n_sta + 2 * n_slow + 2 * n_fast) / (FMA_PER_CLK_PER_SM * N_SM * sm_max_mhz * 1e6) / (ms_local * 1e-3))
        roofline["slow_fma_per_tone_sample"] = SLOW_FMA_PER_TONE_SAMPLE

    # ---- oracle on this box's host cores (bounded sample) ----------------------------------------
    n_cpu = max(1 << 16, min(1 << 22, (1 << 32) // w.n_tones // 4096 * 4096))   # ~4e9 tone-samples: ~10 s on 16 cores
    rate, cores, secs = oracle_rate(w, n_cpu)
    cpu_baseline = {"value": rate / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
                    "sample": f"first {min(n_cpu, w.n_samples)} of {w.n_samples} samples x {w.n_tones} tones of {w.name}, "
                              f"{secs:.2f} s wall"}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup),
        "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": w_desc, "engine": args.engine,
                   "tones": w.n_tones, "samples_per_step": w.n_samples, "launch": "one awg_synthesize_range per step",
                   "l2": f"output rotates over {len(bufs)} device buffers ({len(bufs) * 2 * w.n_samples / 1e6:.0f} MB > 126 MB L2); "
                         f"the only input is the {w.n_tones * 288 // 1024} KB tone table",
                   "parallelism": "replicas only (no data-path collective)" if world > 1 else "1 GPU"},
        "out_MS_per_s": world * w.n_samples / ms_per_step / 1e3,
        "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu_baseline,
        "phase_dtype": "u64 fixed-point turns + fp64 re-centring, u32/fp32 in the inner loop",
    }
    if world == 1 and not args.no_extras:
        line["extras"] = run_extras(torch, awg, sm_max_mhz)
    plan.close()
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", default="C3", help="timed workload (default C3 = the headline; others are profiling aids)")
    ap.add_argument("--engine", choices=sorted(ENGINES), default="auto", help="sine engine of the timed plan")
    ap.add_argument("--no-extras", action="store_true", help="skip the other configs and the capacity search")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
