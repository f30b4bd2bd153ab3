"""ctypes binding of include/awg.h: the same names, argument marshalling only.

Every step of the hot path runs in the CUDA library; nothing here computes.  PyTorch is used for
device memory and streams only.  There is no CPU fallback: if ``libawg_b200.so`` is missing the
import fails (build it with ``python paper_2403_15582_b200/build.py``).
"""
from __future__ import annotations

import ctypes
import os
from ctypes import POINTER, byref, c_char_p, c_double, c_int16, c_int32, c_int64, c_void_p
from typing import Optional, Sequence, Tuple

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_PKG, "libawg_b200.so")

AWG_OK = 0
AWG_ERR_INVALID_ARG = -1
AWG_ERR_ALLOC = -2
AWG_ERR_CUDA = -3
AWG_ERR_STATE = -4
AWG_ERR_UNDERRUN = -5

AWG_PROFILE_STATIC = 0
AWG_PROFILE_LINEAR = 1
AWG_PROFILE_MINJERK = 2
AWG_PROFILE_EXP = 3

AWG_ENGINE_AUTO = 0
AWG_ENGINE_MUFU = 1
AWG_ENGINE_FP64 = 2
AWG_ENGINE_FMA = 3

#: every symbol include/awg.h declares (tests check that the library exports each of them)
EXPORTED = (
    "awg_plan_create", "awg_plan_destroy", "awg_set_scale", "awg_set_engine", "awg_set_trajectories",
    "awg_set_amplitude_ramps", "awg_update_trajectories", "awg_synthesize_chunk", "awg_synthesize_chunk_f32", "awg_synthesize_range",
    "awg_synthesize_range_host", "awg_ring_create", "awg_ring_submit", "awg_ring_acquire", "awg_ring_release",
    "awg_synthesize_chunk_mux", "awg_snap_frequency", "awg_static_buffer_set", "awg_static_buffer_fold",
    "awg_static_buffer_read",
    "awg_ring_stats", "awg_ring_destroy", "awg_plan_io_bytes", "awg_plan_op_counts", "awg_plan_hot_tiles", "awg_synthesize_noalloc", "awg_kernel_launch_count",
    "awg_last_error",
)


def _load() -> ctypes.CDLL:
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: the CUDA extension has not been built "
            "(python paper_2403_15582_b200/build.py).  There is no CPU fallback.")
    lib = ctypes.CDLL(LIB_PATH)
    P, D, I32, I64 = c_void_p, c_double, c_int32, c_int64
    sig = {
        "awg_plan_create": (I32, [POINTER(P), I32, D, I64]),
        "awg_plan_destroy": (I32, [P]),
        "awg_set_scale": (I32, [P, D]),
        "awg_set_engine": (I32, [P, I32]),
        "awg_set_trajectories": (I32, [P, P, P, P, P, P, P, P]),
        "awg_set_amplitude_ramps": (I32, [P, P, P, P, P]),
        "awg_update_trajectories": (I32, [P, I64, I32, P, P, P, P]),
        "awg_synthesize_chunk": (I32, [P, I64, P, P]),
        "awg_synthesize_chunk_f32": (I32, [P, I64, P, P]),
        "awg_synthesize_range": (I32, [P, I64, I64, P, P]),
        "awg_synthesize_range_host": (I32, [P, I64, I64, P]),
        "awg_synthesize_chunk_mux": (I32, [POINTER(P), I32, I64, P, P]),
        "awg_snap_frequency": (I32, [D, D, I64, POINTER(D)]),
        "awg_static_buffer_set": (I32, [P, I32, P, P]),
        "awg_static_buffer_fold": (I32, [P, I64, I32, P, P]),
        "awg_static_buffer_read": (I32, [P, P, P]),
        "awg_ring_create": (I32, [POINTER(P), P, I32, I32]),
        "awg_ring_submit": (I32, [P, I64, I32, P, P, P, P]),
        "awg_ring_acquire": (I32, [P, POINTER(I64), POINTER(P), POINTER(P)]),
        "awg_ring_release": (I32, [P, I64]),
        "awg_ring_stats": (I32, [P, POINTER(I64), POINTER(I64), POINTER(D)]),
        "awg_ring_destroy": (I32, [P]),
        "awg_plan_io_bytes": (I32, [P, POINTER(I64), POINTER(I64)]),
        "awg_plan_op_counts": (I32, [P, I64, I64, POINTER(I64), POINTER(I64), POINTER(I64)]),
        "awg_plan_hot_tiles": (I32, [P, I64, I64, POINTER(I32), POINTER(I32)]),
        "awg_synthesize_noalloc": (I32, [D, I32, P, P, P, P, P, P, P, I64, I64, P, P]),
        "awg_kernel_launch_count": (I64, []),
        "awg_last_error": (c_char_p, []),
    }
    for name, (res, args) in sig.items():
        try:
            fn = getattr(lib, name)
        except AttributeError as e:
            raise ImportError(f"{LIB_PATH} is stale (no symbol {name}): rebuild it with "
                              "python paper_2403_15582_b200/build.py") from e
        fn.restype = res
        fn.argtypes = args
    return lib


_lib = _load()


class AwgError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(f"awg status {status}: {message}")
        self.status = status


def awg_last_error() -> str:
    return (_lib.awg_last_error() or b"").decode()


def _check(status: int, allow: Tuple[int, ...] = ()) -> int:
    if status != AWG_OK and status not in allow:
        raise AwgError(status, awg_last_error())
    return status


def _f64(a, n: Optional[int] = None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.float64)
    if n is not None and a.shape != (n,):
        raise ValueError(f"expected {n} values, got shape {a.shape}")
    return a


def _i32(a, n: Optional[int] = None) -> np.ndarray:
    a = np.ascontiguousarray(a, dtype=np.int32)
    if n is not None and a.shape != (n,):
        raise ValueError(f"expected {n} values, got shape {a.shape}")
    return a


def _stream_handle(stream) -> int:
    """cudaStream_t of a torch stream (None = torch's current stream)."""
    if isinstance(stream, int):
        return stream
    import torch
    s = torch.cuda.current_stream() if stream is None else stream
    return int(s.cuda_stream)


# ---- the C ABI, one Python function per entry point (same names) -----------------------------------
def awg_plan_create(n_tones: int, sample_rate_hz: float, chunk_len: int) -> c_void_p:
    h = c_void_p()
    _check(_lib.awg_plan_create(byref(h), n_tones, sample_rate_hz, chunk_len))
    return h


def awg_plan_destroy(plan) -> None:
    _check(_lib.awg_plan_destroy(plan))


def awg_set_scale(plan, scale: float) -> None:
    _check(_lib.awg_set_scale(plan, scale))


def awg_set_engine(plan, engine: int) -> None:
    _check(_lib.awg_set_engine(plan, engine))


def awg_set_trajectories(plan, n_tones, f0, f1, A, phi0, t_start, t_dur, profile) -> None:
    arrs = [_f64(x, n_tones) for x in (f0, f1, A, phi0, t_start, t_dur)]
    prof = _i32(profile, n_tones)
    _check(_lib.awg_set_trajectories(plan, *[a.ctypes.data for a in arrs], prof.ctypes.data))


def awg_set_amplitude_ramps(plan, n_tones, A1, t_start, t_dur, profile) -> None:
    arrs = [_f64(x, n_tones) for x in (A1, t_start, t_dur)]
    prof = _i32(profile, n_tones)
    _check(_lib.awg_set_amplitude_ramps(plan, *[a.ctypes.data for a in arrs], prof.ctypes.data))


def awg_update_trajectories(plan, chunk_idx: int, tone_idx, f1, t_dur, profile) -> None:
    idx = _i32(tone_idx)
    n = idx.shape[0]
    f1a, da, pa = _f64(f1, n), _f64(t_dur, n), _i32(profile, n)
    _check(_lib.awg_update_trajectories(plan, chunk_idx, n, idx.ctypes.data, f1a.ctypes.data, da.ctypes.data,
                                        pa.ctypes.data))


def awg_synthesize_chunk(plan, chunk_idx: int, dev_out_ptr: int, stream=None) -> None:
    _check(_lib.awg_synthesize_chunk(plan, chunk_idx, dev_out_ptr, _stream_handle(stream)))


def awg_synthesize_chunk_f32(plan, chunk_idx: int, dev_out_ptr: int, stream=None) -> None:
    _check(_lib.awg_synthesize_chunk_f32(plan, chunk_idx, dev_out_ptr, _stream_handle(stream)))


def awg_synthesize_range(plan, first_chunk: int, n_chunks: int, dev_out_ptr: int, stream=None) -> None:
    _check(_lib.awg_synthesize_range(plan, first_chunk, n_chunks, dev_out_ptr, _stream_handle(stream)))


def awg_synthesize_range_host(plan, first_chunk: int, n_chunks: int, host_out_ptr: int) -> None:
    _check(_lib.awg_synthesize_range_host(plan, first_chunk, n_chunks, host_out_ptr))


def awg_synthesize_chunk_mux(plans: Sequence, chunk_idx: int, dev_out_ptr: int, stream=None) -> None:
    arr = (c_void_p * len(plans))(*[p.value if isinstance(p, c_void_p) else p for p in plans])
    _check(_lib.awg_synthesize_chunk_mux(arr, len(plans), chunk_idx, dev_out_ptr, _stream_handle(stream)))


def awg_snap_frequency(f0_hz: float, sample_rate_hz: float, L_s: int) -> float:
    out = c_double()
    _check(_lib.awg_snap_frequency(f0_hz, sample_rate_hz, L_s, byref(out)))
    return out.value


def awg_static_buffer_set(plan, tone_idx, stream=None) -> None:
    idx = _i32(tone_idx)
    _check(_lib.awg_static_buffer_set(plan, idx.shape[0], idx.ctypes.data, _stream_handle(stream)))


def awg_static_buffer_fold(plan, chunk_idx: int, tone_idx, stream=None) -> None:
    idx = _i32(tone_idx)
    _check(_lib.awg_static_buffer_fold(plan, chunk_idx, idx.shape[0], idx.ctypes.data, _stream_handle(stream)))


def awg_static_buffer_read(plan, dev_out_ptr: int, stream=None) -> None:
    _check(_lib.awg_static_buffer_read(plan, dev_out_ptr, _stream_handle(stream)))


def awg_ring_create(plan, n_slots: int, host_mirror: bool) -> c_void_p:
    h = c_void_p()
    _check(_lib.awg_ring_create(byref(h), plan, n_slots, 1 if host_mirror else 0))
    return h


def awg_ring_submit(ring, chunk_idx: int, tone_idx=(), f1=(), t_dur=(), profile=()) -> None:
    idx = _i32(tone_idx)
    n = idx.shape[0]
    f1a, da, pa = _f64(f1, n), _f64(t_dur, n), _i32(profile, n)
    _check(_lib.awg_ring_submit(ring, chunk_idx, n, idx.ctypes.data, f1a.ctypes.data, da.ctypes.data, pa.ctypes.data))


def awg_ring_acquire(ring) -> Tuple[int, int, int, bool]:
    """-> (chunk_idx, device pointer, host pointer or 0, on_time)."""
    c, d, h = c_int64(), c_void_p(), c_void_p()
    st = _check(_lib.awg_ring_acquire(ring, byref(c), byref(d), byref(h)), allow=(AWG_ERR_UNDERRUN,))
    return c.value, d.value or 0, h.value or 0, st == AWG_OK


def awg_ring_release(ring, chunk_idx: int) -> None:
    _check(_lib.awg_ring_release(ring, chunk_idx))


def awg_ring_stats(ring) -> Tuple[int, int, float]:
    a, b, m = c_int64(), c_int64(), c_double()
    _check(_lib.awg_ring_stats(ring, byref(a), byref(b), byref(m)))
    return a.value, b.value, m.value


def awg_ring_destroy(ring) -> None:
    _check(_lib.awg_ring_destroy(ring))


def awg_plan_io_bytes(plan) -> Tuple[int, int]:
    a, b = c_int64(), c_int64()
    _check(_lib.awg_plan_io_bytes(plan, byref(a), byref(b)))
    return a.value, b.value


def awg_synthesize_noalloc(sample_rate_hz: float, n_tones: int, f0, f1, A, phi0, t_start, t_dur, profile,
                           first_sample: int, n_samples: int, dev_out_ptr: int, stream=None) -> None:
    arrs = [_f64(x, n_tones) for x in (f0, f1, A, phi0, t_start, t_dur)]
    prof = _i32(profile, n_tones)
    _check(_lib.awg_synthesize_noalloc(sample_rate_hz, n_tones, *[a.ctypes.data for a in arrs], prof.ctypes.data,
                                       first_sample, n_samples, dev_out_ptr, _stream_handle(stream)))


def awg_plan_hot_tiles(plan, first_chunk: int, n_chunks: int) -> Tuple[int, int]:
    a, b = ctypes.c_int32(0), ctypes.c_int32(0)
    _check(_lib.awg_plan_hot_tiles(plan, first_chunk, n_chunks, byref(a), byref(b)))
    return a.value, b.value


def awg_plan_op_counts(plan, first_chunk: int, n_chunks: int) -> Tuple[int, int, int]:
    """-> (static, slow-moving, fast-moving) tone-samples of the current table over the chunk range."""
    a, b, c = c_int64(), c_int64(), c_int64()
    _check(_lib.awg_plan_op_counts(plan, first_chunk, n_chunks, byref(a), byref(b), byref(c)))
    return a.value, b.value, c.value


def awg_kernel_launch_count() -> int:
    return int(_lib.awg_kernel_launch_count())


# ---- convenience wrappers (still marshalling only) ---------------------------------------------------
class Plan:
    """Owns one awg_plan.  Output tensors are torch CUDA tensors (int16 codes or fp32 sums)."""

    def __init__(self, n_tones: int, sample_rate_hz: float, chunk_len: int, scale: Optional[float] = None,
                 engine: int = AWG_ENGINE_AUTO):
        self.n_tones, self.sample_rate, self.chunk_len = int(n_tones), float(sample_rate_hz), int(chunk_len)
        self._h = awg_plan_create(self.n_tones, self.sample_rate, self.chunk_len)
        if scale is not None:
            awg_set_scale(self._h, scale)
        if engine != AWG_ENGINE_AUTO:
            awg_set_engine(self._h, engine)

    @classmethod
    def from_workload(cls, w, engine: int = AWG_ENGINE_AUTO, chunk_len: Optional[int] = None) -> "Plan":
        p = cls(w.n_tones, w.sample_rate, chunk_len or w.chunk_len, w.scale, engine)
        p.set_trajectories(w.f0, w.f1, w.A, w.phi0, w.t_start, w.t_dur, w.profile)
        return p

    @property
    def handle(self):
        return self._h

    def set_scale(self, scale: float) -> None:
        awg_set_scale(self._h, scale)

    def set_engine(self, engine: int) -> None:
        awg_set_engine(self._h, engine)

    def set_trajectories(self, f0, f1, A, phi0, t_start, t_dur, profile) -> None:
        awg_set_trajectories(self._h, self.n_tones, f0, f1, A, phi0, t_start, t_dur, profile)

    def set_amplitude_ramps(self, A1, t_start, t_dur, profile) -> None:
        awg_set_amplitude_ramps(self._h, self.n_tones, A1, t_start, t_dur, profile)

    def update_trajectories(self, chunk_idx: int, tone_idx, f1, t_dur, profile) -> None:
        awg_update_trajectories(self._h, chunk_idx, tone_idx, f1, t_dur, profile)

    def _out(self, n: int, dtype, out):
        import torch
        if out is None:
            out = torch.empty(n, dtype=dtype, device="cuda")
        if out.dtype != dtype or out.numel() != n or not out.is_cuda or not out.is_contiguous():
            raise ValueError("output tensor has the wrong dtype, size or device")
        return out

    def synthesize_chunk(self, chunk_idx: int, out=None, stream=None):
        import torch
        out = self._out(self.chunk_len, torch.int16, out)
        awg_synthesize_chunk(self._h, chunk_idx, out.data_ptr(), stream)
        return out

    def synthesize_chunk_f32(self, chunk_idx: int, out=None, stream=None):
        import torch
        out = self._out(self.chunk_len, torch.float32, out)
        awg_synthesize_chunk_f32(self._h, chunk_idx, out.data_ptr(), stream)
        return out

    def synthesize_range(self, first_chunk: int, n_chunks: int, out=None, stream=None):
        import torch
        out = self._out(self.chunk_len * n_chunks, torch.int16, out)
        awg_synthesize_range(self._h, first_chunk, n_chunks, out.data_ptr(), stream)
        return out

    def synthesize_range_host(self, first_chunk: int, n_chunks: int, out=None):
        """Synchronous; ``out`` is a CPU int16 tensor (pinned for copy/compute overlap)."""
        import torch
        n = self.chunk_len * n_chunks
        if out is None:
            out = torch.empty(n, dtype=torch.int16, pin_memory=True)
        if out.dtype != torch.int16 or out.numel() != n or out.is_cuda or not out.is_contiguous():
            raise ValueError("host output tensor has the wrong dtype, size or device")
        awg_synthesize_range_host(self._h, first_chunk, n_chunks, out.data_ptr())
        return out

    def static_buffer_set(self, tone_idx, stream=None) -> None:
        awg_static_buffer_set(self._h, tone_idx, stream)

    def static_buffer_fold(self, chunk_idx: int, tone_idx, stream=None) -> None:
        awg_static_buffer_fold(self._h, chunk_idx, tone_idx, stream)

    def static_buffer(self, out=None, stream=None):
        import torch
        out = self._out(self.chunk_len, torch.float32, out)
        awg_static_buffer_read(self._h, out.data_ptr(), stream)
        return out

    def io_bytes(self) -> Tuple[int, int]:
        return awg_plan_io_bytes(self._h)

    def hot_tiles(self, first_chunk: int, n_chunks: int) -> Tuple[int, int]:
        """(tiles of the range where many slow moves start or end at once, how many of them the launch serves first)"""
        return awg_plan_hot_tiles(self._h, first_chunk, n_chunks)

    def op_counts(self, first_chunk: int, n_chunks: int) -> Tuple[int, int, int]:
        return awg_plan_op_counts(self._h, first_chunk, n_chunks)

    def close(self) -> None:
        if self._h is not None:
            h, self._h = self._h, None
            awg_plan_destroy(h)

    def __enter__(self):
        return self

    def __exit__(self, *exc):
        self.close()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def synthesize_chunk_mux(plans: Sequence[Plan], chunk_idx: int, out=None, stream=None):
    """Interleaved int16 codes of the channels' plans: out[C i + c] (torch CUDA tensor of C*chunk_len int16)."""
    import torch
    n = plans[0].chunk_len * len(plans)
    if out is None:
        out = torch.empty(n, dtype=torch.int16, device="cuda")
    if out.dtype != torch.int16 or out.numel() != n or not out.is_cuda or not out.is_contiguous():
        raise ValueError("output tensor has the wrong dtype, size or device")
    awg_synthesize_chunk_mux([p.handle for p in plans], chunk_idx, out.data_ptr(), stream)
    return out


def synthesize_noalloc(sample_rate_hz: float, f0, f1, A, phi0, t_start, t_dur, profile, first_sample: int, n_samples: int,
                       out, stream=None):
    """awg_synthesize_noalloc into ``out`` (a caller-owned torch CUDA tensor of n_samples int16): no plan, no device
    allocation anywhere (<= 4096 tones, <= 2^20 samples per call; calls that overlap on the GPU race)."""
    import torch
    if out.dtype != torch.int16 or out.numel() != n_samples or not out.is_cuda or not out.is_contiguous():
        raise ValueError("output tensor has the wrong dtype, size or device")
    awg_synthesize_noalloc(sample_rate_hz, len(np.atleast_1d(f0)), f0, f1, A, phi0, t_start, t_dur, profile, first_sample,
                           n_samples, out.data_ptr(), stream)
    return out


class Ring:
    """Streaming ring bound to a Plan (DAC-FIFO stand-in)."""

    def __init__(self, plan: Plan, n_slots: int = 3, host_mirror: bool = False):
        self.plan = plan
        self.host_mirror = bool(host_mirror)
        self._h = awg_ring_create(plan.handle, n_slots, host_mirror)

    def submit(self, chunk_idx: int, update=None) -> None:
        if update is None:
            awg_ring_submit(self._h, chunk_idx)
        else:
            awg_ring_submit(self._h, chunk_idx, update.tone_idx, update.f1, update.t_dur, update.profile)

    def acquire(self):
        return awg_ring_acquire(self._h)

    def release(self, chunk_idx: int) -> None:
        awg_ring_release(self._h, chunk_idx)

    def stats(self):
        return awg_ring_stats(self._h)

    def host_view(self, host_ptr: int) -> np.ndarray:
        """numpy view (no copy) of an acquired pinned-host slot."""
        n = self.plan.chunk_len
        buf = (c_int16 * n).from_address(host_ptr)
        return np.frombuffer(buf, dtype=np.int16, count=n)

    def close(self) -> None:
        if self._h is not None:
            h, self._h = self._h, None
            awg_ring_destroy(h)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
