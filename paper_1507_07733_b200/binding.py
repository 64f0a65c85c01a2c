"""ctypes binding of libaera_unfold.so -- argument marshalling only.

Function names and argument order mirror include/aera_unfold.h. torch is used for device
memory and streams, nothing else: every step of the path runs in the library's kernels.
Raises ImportError if the library cannot be built/loaded (no fallback of any kind).
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

AERA_F32, AERA_F64 = 0, 1
AERA_OP_UNFOLD, AERA_OP_SCAN, AERA_OP_FOLD, AERA_OP_RECONSTRUCT = 0, 1, 2, 3
STATUS = {0: "AERA_OK", 1: "AERA_ERR_INVALID_ARG", 2: "AERA_ERR_UNSUPPORTED_N", 3: "AERA_ERR_DTYPE_MISMATCH",
          4: "AERA_ERR_WORKSPACE", 5: "AERA_ERR_ALLOC", 6: "AERA_ERR_CUDA", 7: "AERA_ERR_BAND"}

EXPORTS = ("aera_pattern_upload", "aera_pattern_free", "aera_band", "aera_workspace_bytes", "aera_unfold_batch",
           "aera_scan_directions", "aera_unfold_batch_host", "aera_reconstruct_batch", "aera_fold_batch", "aera_pattern_set_band_filter", "aera_set_kernel_variant", "aera_launch_count",
           "aera_last_error", "aera_version", "aera_profile_enable", "aera_profile_read", "aera_measure_alu_peak", "aera_last_kernel", "aera_unfold_batch_multi", "aera_unfold_batch_i16",
           "aera_unfold_batch_upsampled", "aera_workspace_bytes_ex", "aera_reconstruct_convergence",
           "aera_unfold_batch_static", "aera_pattern_prepare", "aera_static_scratch_bytes", "aera_set_long_trace_l2_persist",
           "aera_unfold_batch_host_i16")


class AeraError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS.get(status, status)}: {msg}")
        self.status = status


class PatternDesc(C.Structure):
    _fields_ = [
        ("dtype", C.c_int),
        ("n_zenith", C.c_int), ("zenith0_deg", C.c_double), ("dzenith_deg", C.c_double),
        ("n_azimuth", C.c_int), ("azimuth0_deg", C.c_double), ("dazimuth_deg", C.c_double),
        ("azimuth_periodic", C.c_int),
        ("n_freq", C.c_int), ("freq0_hz", C.c_double), ("dfreq_hz", C.c_double),
    ]


def _load():
    try:
        path = _build.build()
    except Exception as e:  # no nvcc and no prebuilt library
        if os.path.exists(_build.LIB):
            path = _build.LIB
        else:
            raise ImportError(f"libaera_unfold.so is missing and could not be built: {e}") from e
    try:
        lib = C.CDLL(path)
    except OSError as e:
        raise ImportError(f"cannot load {path}: {e}") from e
    vp, ip, dp = C.c_void_p, C.POINTER(C.c_int), C.c_void_p
    lib.aera_pattern_upload.argtypes = [C.POINTER(PatternDesc), vp, C.c_int, vp, C.POINTER(vp)]
    lib.aera_pattern_upload.restype = C.c_int
    lib.aera_pattern_free.argtypes = [vp]
    lib.aera_pattern_free.restype = C.c_int
    lib.aera_band.argtypes = [vp, C.c_int, C.c_double, ip, ip]
    lib.aera_band.restype = C.c_int
    lib.aera_workspace_bytes.argtypes = [C.c_int, vp, C.c_int, C.c_long, C.c_int, C.c_int, C.c_double]
    lib.aera_workspace_bytes.restype = C.c_size_t
    lib.aera_unfold_batch.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.aera_unfold_batch.restype = C.c_int
    lib.aera_scan_directions.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, vp, C.c_long, dp, vp, vp, vp, C.c_size_t, vp]
    lib.aera_scan_directions.restype = C.c_int
    lib.aera_unfold_batch_host.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, vp, vp, vp]
    lib.aera_unfold_batch_host.restype = C.c_int
    lib.aera_unfold_batch_host_i16.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, vp, C.POINTER(C.c_double), dp, vp, vp, vp]
    lib.aera_unfold_batch_host_i16.restype = C.c_int
    lib.aera_reconstruct_batch.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, C.c_int, dp, vp, vp, vp, vp, vp,
                                           vp, C.c_size_t, vp]
    lib.aera_reconstruct_batch.restype = C.c_int
    lib.aera_fold_batch.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, vp, vp, C.c_size_t, vp]
    lib.aera_fold_batch.restype = C.c_int
    lib.aera_pattern_set_band_filter.argtypes = [vp, C.c_int, C.c_double, dp, C.c_int, vp]
    lib.aera_pattern_set_band_filter.restype = C.c_int
    lib.aera_set_kernel_variant.argtypes = [C.c_int]
    lib.aera_set_kernel_variant.restype = C.c_int
    lib.aera_launch_count.restype = C.c_ulonglong
    lib.aera_set_long_trace_l2_persist.argtypes = [C.c_int]
    lib.aera_set_long_trace_l2_persist.restype = C.c_int
    lib.aera_profile_enable.argtypes = [C.c_int]
    lib.aera_profile_enable.restype = C.c_int
    lib.aera_profile_read.argtypes = [C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_long)]
    lib.aera_profile_read.restype = C.c_int
    lib.aera_last_error.restype = C.c_char_p
    lib.aera_unfold_batch_multi.argtypes = [C.POINTER(vp), C.c_int, vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.aera_unfold_batch_multi.restype = C.c_int
    lib.aera_unfold_batch_i16.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_double, vp, C.POINTER(C.c_double), dp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.aera_unfold_batch_i16.restype = C.c_int
    lib.aera_unfold_batch_upsampled.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, C.c_int, vp, dp, vp, vp, vp, vp, C.c_size_t, vp]
    lib.aera_unfold_batch_upsampled.restype = C.c_int
    lib.aera_workspace_bytes_ex.argtypes = [C.c_int, vp, C.c_int, C.c_long, C.c_int, C.c_int, C.c_double, C.c_int, C.c_int]
    lib.aera_workspace_bytes_ex.restype = C.c_size_t
    lib.aera_reconstruct_convergence.argtypes = [dp, C.c_int, C.c_int, C.c_double, vp, vp]
    lib.aera_reconstruct_convergence.restype = C.c_int
    lib.aera_last_kernel.restype = C.c_char_p
    lib.aera_unfold_batch_static.argtypes = [vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_double, vp, dp, vp, vp, vp, vp]
    lib.aera_unfold_batch_static.restype = C.c_int
    lib.aera_pattern_prepare.argtypes = [vp, C.c_int, C.c_double, vp]
    lib.aera_pattern_prepare.restype = C.c_int
    lib.aera_static_scratch_bytes.restype = C.c_size_t
    lib.aera_measure_alu_peak.argtypes = [C.c_int, C.c_int, C.POINTER(C.c_double), ip, ip]
    lib.aera_measure_alu_peak.restype = C.c_int
    lib.aera_version.restype = C.c_char_p
    return lib, path


_lib, LIBRARY_PATH = _load()


def _check(st):
    if st != 0:
        raise AeraError(st, _lib.aera_last_error().decode())


def _dtype_code(t: torch.dtype) -> int:
    if t in (torch.float32, torch.complex64):
        return AERA_F32
    if t in (torch.float64, torch.complex128):
        return AERA_F64
    raise TypeError(f"unsupported dtype {t}")


def _stream_ptr(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


class Pattern:
    """Owner of an aera_pattern_t handle."""

    def __init__(self, handle, desc: PatternDesc):
        self.handle = handle
        self.desc = desc
        self.dtype = desc.dtype

    def free(self):
        if self.handle:
            _lib.aera_pattern_free(self.handle)
            self.handle = None

    def __del__(self):
        try:
            self.free()
        except Exception:
            pass


def make_desc(grid, dtype_code: int) -> PatternDesc:
    """grid: any object with the PatternGrid attribute names of aera_inputs."""
    return PatternDesc(dtype_code, grid.n_zenith, grid.zenith0_deg, grid.dzenith_deg, grid.n_azimuth, grid.azimuth0_deg,
                       grid.dazimuth_deg, 1 if grid.azimuth_periodic else 0, grid.n_freq, grid.freq0_hz, grid.dfreq_hz)


def aera_version() -> str:
    return _lib.aera_version().decode()


def aera_launch_count() -> int:
    return int(_lib.aera_launch_count())


def aera_set_kernel_variant(variant: int) -> int:
    return int(_lib.aera_set_kernel_variant(int(variant)))


def aera_set_long_trace_l2_persist(megabytes: int) -> int:
    """Opt-in: let the N = 65536 kernel set the device's persisting-L2 carve-out (MB, clipped to the device maximum;
    negative = leave the device's limit alone, the default). Returns the previous request."""
    return int(_lib.aera_set_long_trace_l2_persist(int(megabytes)))


def aera_last_kernel() -> str:
    """Kernel family the most recent unfold / fold / scan / reconstruct call of this thread dispatched to."""
    return _lib.aera_last_kernel().decode()


ALU_KINDS = {"f32x2": 0, "f32": 1, "f64": 2}


def aera_measure_alu_peak(kind: int, warps_per_sm: int = 16):
    """-> dict(lane_fma_per_s, sm_count, sm_clock_khz): measured FMA issue peak of the current device."""
    v, n, khz = C.c_double(), C.c_int(), C.c_int()
    _check(_lib.aera_measure_alu_peak(int(kind), int(warps_per_sm), C.byref(v), C.byref(n), C.byref(khz)))
    return dict(lane_fma_per_s=v.value, sm_count=n.value, sm_clock_khz=khz.value)


KERNEL_IDS = {"repack": 0, "minv": 1, "unfold": 2, "scan_fwd": 3, "scan_inv": 4, "timing": 5, "planefit": 6}


def aera_profile_enable(on: bool) -> int:
    return int(_lib.aera_profile_enable(1 if on else 0))


def aera_profile_read(kernel_id: int):
    """-> (total_ms, launches) of one kernel since aera_profile_enable(True)."""
    ms, n = C.c_double(), C.c_long()
    _check(_lib.aera_profile_read(kernel_id, C.byref(ms), C.byref(n)))
    return ms.value, n.value


def aera_pattern_upload(desc: PatternDesc, H, stream=None) -> Pattern:
    """H: numpy complex array (host) or torch CUDA complex tensor, shape [2][2][n_z][n_a][n_f]."""
    shape = (2, 2, desc.n_zenith, desc.n_azimuth, desc.n_freq)
    want = np.complex64 if desc.dtype == AERA_F32 else np.complex128
    handle = C.c_void_p()
    if isinstance(H, torch.Tensor):
        if tuple(H.shape) != shape or _dtype_code(H.dtype) != desc.dtype or not H.is_contiguous():
            raise ValueError("H must be a contiguous tensor of shape [2][2][n_z][n_a][n_f] in the descriptor's dtype")
        on_dev = 1 if H.is_cuda else 0
        st = _lib.aera_pattern_upload(C.byref(desc), _ptr(H), on_dev, _stream_ptr(stream), C.byref(handle))
    else:
        Hn = np.ascontiguousarray(H)
        if Hn.shape != shape or Hn.dtype != want:
            raise ValueError(f"H must have shape {shape} and dtype {want}")
        st = _lib.aera_pattern_upload(C.byref(desc), C.c_void_p(Hn.ctypes.data), 0, _stream_ptr(stream), C.byref(handle))
    _check(st)
    return Pattern(handle, desc)


def aera_pattern_free(p: Pattern):
    p.free()


def aera_band(p: Pattern, n_samples: int, fs_hz: float):
    lo, hi = C.c_int(), C.c_int()
    _check(_lib.aera_band(p.handle, n_samples, fs_hz, C.byref(lo), C.byref(hi)))
    return lo.value, hi.value


def aera_workspace_bytes(op: int, p: Pattern, dtype: int, n_events_or_dirs: int, n_stations: int, n_samples: int, fs_hz: float) -> int:
    n = int(_lib.aera_workspace_bytes(op, p.handle, dtype, n_events_or_dirs, n_stations, n_samples, fs_hz))
    if n == 0:
        raise AeraError(1, _lib.aera_last_error().decode())
    return n


def aera_workspace_bytes_ex(op: int, p: Pattern, dtype: int, n_events_or_dirs: int, n_stations: int, n_samples: int, fs_hz: float,
                            n_patterns: int = 1, upsample: int = 1) -> int:
    n = int(_lib.aera_workspace_bytes_ex(op, p.handle, dtype, n_events_or_dirs, n_stations, n_samples, fs_hz, n_patterns, upsample))
    if n == 0:
        raise AeraError(1, _lib.aera_last_error().decode())
    return n


def alloc_workspace(nbytes: int, device="cuda") -> torch.Tensor:
    return torch.empty(nbytes, dtype=torch.uint8, device=device)


def aera_unfold_batch(p: Pattern, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float, efield=None, peak_amp=None,
                      peak_idx=None, workspace=None, stream=None, want_efield=True):
    """traces [E][S][2][N] CUDA real tensor, dirs [E][2] CUDA float64. Returns (efield|None, peak_amp, peak_idx)."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    dt = _dtype_code(traces.dtype)
    if efield is None and want_efield:
        efield = torch.empty_like(traces)
    if peak_amp is None:
        peak_amp = torch.empty((E, S), dtype=traces.dtype, device=traces.device)
    if peak_idx is None:
        peak_idx = torch.empty((E, S), dtype=torch.int32, device=traces.device)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes(AERA_OP_UNFOLD, p, dt, E, S, N, fs_hz) if E > 0 else 256, traces.device)
    _check(_lib.aera_unfold_batch(p.handle, dt, E, S, N, fs_hz, _ptr(traces), _ptr(dirs), _ptr(efield), _ptr(peak_amp),
                                  _ptr(peak_idx), _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return efield, peak_amp, peak_idx


def aera_static_scratch_bytes() -> int:
    """Size of the scratch array built into the library (the limit of aera_unfold_batch_static)."""
    return int(_lib.aera_static_scratch_bytes())


def aera_pattern_prepare(p: Pattern, n_samples: int, fs_hz: float, stream=None):
    """Set-up: build the plan of (n_samples, fs_hz) now (allocates, synchronises) so that later calls do not."""
    _check(_lib.aera_pattern_prepare(p.handle, int(n_samples), float(fs_hz), _stream_ptr(stream)))


def aera_unfold_batch_static(p: Pattern, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float, efield, peak_amp, peak_idx, stream=None):
    """aera_unfold_batch on the library's built-in scratch array, for callers that may not allocate device memory:
    no workspace argument, and EVERY output is the caller's (efield may be None for peaks only) -- this wrapper
    allocates nothing either. Needs aera_pattern_prepare(p, N, fs_hz) beforehand; batches whose scratch exceeds
    aera_static_scratch_bytes() raise AeraError (AERA_ERR_WORKSPACE). Calls that overlap on the GPU race on the array."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    assert peak_amp is not None and peak_idx is not None and tuple(peak_amp.shape) == (E, S) and tuple(peak_idx.shape) == (E, S)
    assert peak_amp.dtype == traces.dtype and peak_idx.dtype == torch.int32 and peak_amp.is_contiguous() and peak_idx.is_contiguous()
    assert efield is None or (efield.shape == traces.shape and efield.dtype == traces.dtype and efield.is_contiguous())
    _check(_lib.aera_unfold_batch_static(p.handle, _dtype_code(traces.dtype), E, S, N, fs_hz, _ptr(traces), _ptr(dirs), _ptr(efield),
                                         _ptr(peak_amp), _ptr(peak_idx), _stream_ptr(stream)))
    return efield, peak_amp, peak_idx


def _outputs(traces, E, S, n_out, efield, peak_amp, peak_idx, want_efield, out_dtype):
    if efield is None and want_efield:
        efield = torch.empty((E, S, 2, n_out), dtype=out_dtype, device=traces.device)
    if peak_amp is None:
        peak_amp = torch.empty((E, S), dtype=out_dtype, device=traces.device)
    if peak_idx is None:
        peak_idx = torch.empty((E, S), dtype=torch.int32, device=traces.device)
    return efield, peak_amp, peak_idx


def aera_unfold_batch_multi(patterns, pattern_id: torch.Tensor, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float,
                            efield=None, peak_amp=None, peak_idx=None, workspace=None, stream=None, want_efield=True):
    """patterns: list of Pattern; pattern_id [S] CUDA int32 (antenna type per station); otherwise as aera_unfold_batch."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    assert pattern_id.is_cuda and pattern_id.dtype == torch.int32 and tuple(pattern_id.shape) == (S,) and pattern_id.is_contiguous()
    dt = _dtype_code(traces.dtype)
    efield, peak_amp, peak_idx = _outputs(traces, E, S, N, efield, peak_amp, peak_idx, want_efield, traces.dtype)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes_ex(AERA_OP_UNFOLD, patterns[0], dt, E, S, N, fs_hz, len(patterns), 1) if E > 0 else 256, traces.device)
    handles = (C.c_void_p * len(patterns))(*[p.handle for p in patterns])
    _check(_lib.aera_unfold_batch_multi(handles, len(patterns), _ptr(pattern_id), dt, E, S, N, fs_hz, _ptr(traces), _ptr(dirs), _ptr(efield),
                                        _ptr(peak_amp), _ptr(peak_idx), _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return efield, peak_amp, peak_idx


def aera_unfold_batch_i16(p: Pattern, traces: torch.Tensor, counts_to_volts, dirs: torch.Tensor, fs_hz: float, efield=None,
                          peak_amp=None, peak_idx=None, workspace=None, stream=None, want_efield=True):
    """traces [E][S][2][N] CUDA int16 ADC counts, counts_to_volts (g0, g1). Returns fp32 (efield|None, peak_amp, peak_idx)."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous() and traces.dtype == torch.int16
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    efield, peak_amp, peak_idx = _outputs(traces, E, S, N, efield, peak_amp, peak_idx, want_efield, torch.float32)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes(AERA_OP_UNFOLD, p, AERA_F32, E, S, N, fs_hz) if E > 0 else 256, traces.device)
    g = (C.c_double * 2)(float(counts_to_volts[0]), float(counts_to_volts[1]))
    _check(_lib.aera_unfold_batch_i16(p.handle, E, S, N, fs_hz, _ptr(traces), g, _ptr(dirs), _ptr(efield), _ptr(peak_amp), _ptr(peak_idx),
                                      _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return efield, peak_amp, peak_idx


def aera_unfold_batch_upsampled(p: Pattern, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float, upsample: int, efield=None,
                                peak_amp=None, peak_idx=None, workspace=None, stream=None, want_efield=True):
    """As aera_unfold_batch with the outputs on a grid `upsample` times finer: efield [E][S][2][upsample N]."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    dt = _dtype_code(traces.dtype)
    efield, peak_amp, peak_idx = _outputs(traces, E, S, N * upsample, efield, peak_amp, peak_idx, want_efield, traces.dtype)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes_ex(AERA_OP_UNFOLD, p, dt, E, S, N, fs_hz, 1, upsample) if E > 0 else 256, traces.device)
    _check(_lib.aera_unfold_batch_upsampled(p.handle, dt, E, S, N, fs_hz, upsample, _ptr(traces), _ptr(dirs), _ptr(efield), _ptr(peak_amp),
                                            _ptr(peak_idx), _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return efield, peak_amp, peak_idx


def aera_scan_directions(p: Pattern, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float, peak_amp=None, peak_idx=None,
                         workspace=None, stream=None):
    """traces [S][2][N] CUDA, dirs [D][2] CUDA float64. Returns (peak_amp [D][S], peak_idx [D][S])."""
    S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    D = dirs.shape[0]
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (D, 2) and dirs.is_contiguous()
    dt = _dtype_code(traces.dtype)
    if peak_amp is None:
        peak_amp = torch.empty((D, S), dtype=traces.dtype, device=traces.device)
    if peak_idx is None:
        peak_idx = torch.empty((D, S), dtype=torch.int32, device=traces.device)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes(AERA_OP_SCAN, p, dt, D, S, N, fs_hz) if D > 0 else 256, traces.device)
    _check(_lib.aera_scan_directions(p.handle, dt, S, N, fs_hz, _ptr(traces), D, _ptr(dirs), _ptr(peak_amp), _ptr(peak_idx),
                                     _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return peak_amp, peak_idx


def aera_pattern_set_band_filter(p: Pattern, n_samples: int, fs_hz: float, weights, stream=None):
    """weights: 1-D array-like of length K (host) or None to remove the filter."""
    if weights is None:
        _check(_lib.aera_pattern_set_band_filter(p.handle, n_samples, fs_hz, None, 0, _stream_ptr(stream)))
        return
    w = np.ascontiguousarray(weights, dtype=np.float64)
    _check(_lib.aera_pattern_set_band_filter(p.handle, n_samples, fs_hz, w.ctypes.data_as(C.c_void_p), int(w.size), _stream_ptr(stream)))


def aera_fold_batch(p: Pattern, efield: torch.Tensor, dirs: torch.Tensor, fs_hz: float, traces=None, workspace=None, stream=None):
    """efield [E][S][2 (theta, phi)][N] CUDA, dirs [E][2] CUDA float64 -> voltage traces [E][S][2][N] (forward model)."""
    E, S, two, N = efield.shape
    assert two == 2 and efield.is_cuda and efield.is_contiguous()
    assert dirs.is_cuda and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    dt = _dtype_code(efield.dtype)
    if traces is None:
        traces = torch.empty_like(efield)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes(AERA_OP_FOLD, p, dt, E, S, N, fs_hz) if E > 0 else 256, efield.device)
    _check(_lib.aera_fold_batch(p.handle, dt, E, S, N, fs_hz, _ptr(efield), _ptr(dirs), _ptr(traces), _ptr(workspace),
                                workspace.numel(), _stream_ptr(stream)))
    return traces


def aera_reconstruct_batch(p: Pattern, traces: torch.Tensor, positions: torch.Tensor, fs_hz: float, n_iter: int,
                           efield=None, want_efield=True, workspace=None, stream=None):
    """traces [E][S][2][N] CUDA, positions [S][2] CUDA float64 (metres). Returns a dict with dirs_hist
    [n_iter][E][2], efield (or None), amp_hist / idx_hist [n_iter][E][S], idx0 / w0 [E][S]."""
    E, S, two, N = traces.shape
    assert two == 2 and traces.is_cuda and traces.is_contiguous()
    assert positions.is_cuda and positions.dtype == torch.float64 and tuple(positions.shape) == (S, 2) and positions.is_contiguous()
    dt = _dtype_code(traces.dtype)
    dev = traces.device
    if efield is None and want_efield:
        efield = torch.empty_like(traces)
    dirs_hist = torch.empty((n_iter, E, 2), dtype=torch.float64, device=dev)
    amp_hist = torch.empty((n_iter, E, S), dtype=traces.dtype, device=dev)
    idx_hist = torch.empty((n_iter, E, S), dtype=torch.int32, device=dev)
    idx0 = torch.empty((E, S), dtype=torch.int32, device=dev)
    w0 = torch.empty((E, S), dtype=traces.dtype, device=dev)
    if workspace is None:
        workspace = alloc_workspace(aera_workspace_bytes(AERA_OP_RECONSTRUCT, p, dt, E, S, N, fs_hz) if E > 0 else 256, dev)
    _check(_lib.aera_reconstruct_batch(p.handle, dt, E, S, N, fs_hz, _ptr(traces), _ptr(positions), n_iter, _ptr(dirs_hist),
                                       _ptr(efield) if efield is not None else None, _ptr(amp_hist), _ptr(idx_hist), _ptr(idx0), _ptr(w0),
                                       _ptr(workspace), workspace.numel(), _stream_ptr(stream)))
    return dict(dirs_hist=dirs_hist, efield=efield, amp_hist=amp_hist, idx_hist=idx_hist, idx0=idx0, w0=w0)


def aera_reconstruct_convergence(dirs_hist: torch.Tensor, tol_deg: float, stream=None) -> torch.Tensor:
    """dirs_hist [n_iter][E][2] CUDA float64 -> conv_iter [E] int32 (first iteration within tol_deg of its predecessor, else -1)."""
    n_iter, E, two = dirs_hist.shape
    assert two == 2 and dirs_hist.is_cuda and dirs_hist.dtype == torch.float64 and dirs_hist.is_contiguous()
    out = torch.empty((E,), dtype=torch.int32, device=dirs_hist.device)
    _check(_lib.aera_reconstruct_convergence(_ptr(dirs_hist), n_iter, E, float(tol_deg), _ptr(out), _stream_ptr(stream)))
    return out


def aera_unfold_batch_host(p: Pattern, traces: torch.Tensor, dirs: torch.Tensor, fs_hz: float, efield=None, peak_amp=None,
                           peak_idx=None, want_efield=True):
    """HOST tensors (pinned for full speed). Synchronous. Returns (efield|None, peak_amp, peak_idx) on the host."""
    E, S, two, N = traces.shape
    assert two == 2 and (not traces.is_cuda) and traces.is_contiguous()
    assert (not dirs.is_cuda) and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    dt = _dtype_code(traces.dtype)
    pin = traces.is_pinned()
    if efield is None and want_efield:
        efield = torch.empty(traces.shape, dtype=traces.dtype, pin_memory=pin)
    if peak_amp is None:
        peak_amp = torch.empty((E, S), dtype=traces.dtype, pin_memory=pin)
    if peak_idx is None:
        peak_idx = torch.empty((E, S), dtype=torch.int32, pin_memory=pin)
    _check(_lib.aera_unfold_batch_host(p.handle, dt, E, S, N, fs_hz, _ptr(traces), _ptr(dirs), _ptr(efield), _ptr(peak_amp), _ptr(peak_idx)))
    return efield, peak_amp, peak_idx


def aera_unfold_batch_host_i16(p: Pattern, traces: torch.Tensor, counts_to_volts, dirs: torch.Tensor, fs_hz: float, efield=None,
                               peak_amp=None, peak_idx=None, want_efield=True):
    """HOST int16 ADC counts [E][S][2][N] (pinned for full speed). Synchronous. Returns fp32 (efield|None, peak_amp,
    peak_idx) on the host; want_efield=False moves the peaks only."""
    E, S, two, N = traces.shape
    assert two == 2 and (not traces.is_cuda) and traces.is_contiguous() and traces.dtype == torch.int16
    assert (not dirs.is_cuda) and dirs.dtype == torch.float64 and tuple(dirs.shape) == (E, 2) and dirs.is_contiguous()
    pin = traces.is_pinned()
    if efield is None and want_efield:
        efield = torch.empty(traces.shape, dtype=torch.float32, pin_memory=pin)
    if peak_amp is None:
        peak_amp = torch.empty((E, S), dtype=torch.float32, pin_memory=pin)
    if peak_idx is None:
        peak_idx = torch.empty((E, S), dtype=torch.int32, pin_memory=pin)
    g = (C.c_double * 2)(float(counts_to_volts[0]), float(counts_to_volts[1]))
    _check(_lib.aera_unfold_batch_host_i16(p.handle, E, S, N, fs_hz, _ptr(traces), g, _ptr(dirs), _ptr(efield), _ptr(peak_amp), _ptr(peak_idx)))
    return efield, peak_amp, peak_idx
