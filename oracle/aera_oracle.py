"""ctypes marshalling for oracle/aera_oracle.c (see that file's header for citations).

No arithmetic of the method happens here: arrays are converted to float64 /
complex128 (exactly representable for float32 / complex64 inputs), handed to the C
functions, and the outputs are returned as numpy arrays.
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

_lib = C.CDLL(_build.build())


class _Grid(C.Structure):
    _fields_ = [
        ("n_zenith", C.c_int), ("zenith0_deg", C.c_double), ("dzenith_deg", C.c_double),
        ("n_azimuth", C.c_int), ("azimuth0_deg", C.c_double), ("dazimuth_deg", C.c_double),
        ("azimuth_periodic", C.c_int),
        ("n_freq", C.c_int), ("freq0_hz", C.c_double), ("dfreq_hz", C.c_double),
    ]


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_long)


def _d(a):
    return a.ctypes.data_as(_dp) if a is not None else None


def _grid(g) -> _Grid:
    return _Grid(g.n_zenith, g.zenith0_deg, g.dzenith_deg, g.n_azimuth, g.azimuth0_deg,
                 g.dazimuth_deg, 1 if g.azimuth_periodic else 0, g.n_freq, g.freq0_hz, g.dfreq_hz)


def _table(g, H):
    H = np.ascontiguousarray(np.asarray(H).astype(np.complex128))
    assert H.shape == (2, 2, g.n_zenith, g.n_azimuth, g.n_freq), H.shape
    return H


_lib.oracle_num_threads.restype = C.c_int
_lib.oracle_unfold_batch.restype = C.c_long
_lib.oracle_unfold_station_spectra.restype = C.c_long
_lib.oracle_scan.restype = C.c_long
_lib.oracle_fold_station.restype = C.c_long
_lib.oracle_solve2x2.restype = C.c_int


def num_threads() -> int:
    return int(_lib.oracle_num_threads())


def twiddles(N: int):
    wr = np.empty(N); wi = np.empty(N)
    _lib.oracle_twiddles(C.c_int(N), _d(wr), _d(wi))
    return wr + 1j * wi


def band(N: int, fs_hz: float, n_freq: int, freq0_hz: float, dfreq_hz: float):
    lo = C.c_long(); hi = C.c_long()
    _lib.oracle_band(C.c_int(N), C.c_double(fs_hz), C.c_int(n_freq), C.c_double(freq0_hz),
                     C.c_double(dfreq_hz), C.byref(lo), C.byref(hi))
    return int(lo.value), int(hi.value)


def dft_band(x, k_lo: int, k_hi: int):
    x = np.ascontiguousarray(x, dtype=np.float64)
    N = x.shape[0]
    W = twiddles(N)
    wr = np.ascontiguousarray(W.real); wi = np.ascontiguousarray(W.imag)
    K = k_hi - k_lo + 1
    xr = np.empty(K); xi = np.empty(K)
    _lib.oracle_dft_band(_d(x), C.c_int(N), C.c_long(k_lo), C.c_long(k_hi), _d(wr), _d(wi), _d(xr), _d(xi))
    return xr + 1j * xi


def analytic_from_band(E, N: int, k_lo: int, k_hi: int):
    E = np.asarray(E, dtype=np.complex128)
    er = np.ascontiguousarray(E.real); ei = np.ascontiguousarray(E.imag)
    W = twiddles(N)
    wr = np.ascontiguousarray(W.real); wi = np.ascontiguousarray(W.imag)
    zr = np.empty(N); zi = np.empty(N)
    _lib.oracle_analytic_from_band(_d(er), _d(ei), C.c_int(N), C.c_long(k_lo), C.c_long(k_hi),
                                   _d(wr), _d(wi), _d(zr), _d(zi))
    return zr + 1j * zi


def pattern_eval(grid, H, theta_deg: float, phi_deg: float, f_hz: float):
    """-> complex128 [2][2] (channel, pol)."""
    H = _table(grid, H)
    out = np.empty(8)
    g = _grid(grid)
    _lib.oracle_pattern_eval(C.byref(g), _d(H.view(np.float64)), C.c_double(theta_deg),
                             C.c_double(phi_deg), C.c_double(f_hz), _d(out))
    return (out[0::2] + 1j * out[1::2]).reshape(2, 2)


def solve2x2(h, v):
    h = np.asarray(h, dtype=np.complex128).reshape(4)
    v = np.asarray(v, dtype=np.complex128).reshape(2)
    hh = np.ascontiguousarray(np.stack([h.real, h.imag], axis=1).ravel())
    vv = np.ascontiguousarray(np.stack([v.real, v.imag], axis=1).ravel())
    e = np.empty(4)
    ok = _lib.oracle_solve2x2(_d(hh), _d(vv), _d(e))
    return np.array([e[0] + 1j * e[1], e[2] + 1j * e[3]]), bool(ok)


def peak(zt, zp):
    zt = np.asarray(zt, dtype=np.complex128); zp = np.asarray(zp, dtype=np.complex128)
    N = zt.shape[0]
    a = [np.ascontiguousarray(x) for x in (zt.real, zt.imag, zp.real, zp.imag)]
    env2 = np.empty(N); amp = C.c_double(); idx = C.c_int32()
    _lib.oracle_peak(_d(a[0]), _d(a[1]), _d(a[2]), _d(a[3]), C.c_int(N), _d(env2), C.byref(amp), C.byref(idx))
    return env2, float(amp.value), int(idx.value)


def unfold_batch(grid, H, fs_hz: float, traces, dirs, want_efield=True, want_env2=False):
    """traces [U][2][N] (any real dtype), dirs [U][2] degrees (one row per unit).

    -> dict(efield [U][2][N] | None, env2 [U][N] | None, amp [U], idx [U] int32, K)
    """
    H = _table(grid, H)
    tr = np.ascontiguousarray(traces, dtype=np.float64)
    U, two, N = tr.shape
    assert two == 2
    dd = np.ascontiguousarray(dirs, dtype=np.float64)
    assert dd.shape == (U, 2)
    ef = np.empty((U, 2, N)) if want_efield else None
    e2 = np.empty((U, N)) if want_env2 else None
    amp = np.empty(U); idx = np.empty(U, dtype=np.int32)
    g = _grid(grid)
    K = _lib.oracle_unfold_batch(C.byref(g), _d(H.view(np.float64)), C.c_long(U), C.c_int(N),
                                 C.c_double(fs_hz), _d(tr), _d(dd), _d(ef), _d(e2), _d(amp),
                                 idx.ctypes.data_as(_ip))
    return dict(efield=ef, env2=e2, amp=amp, idx=idx, K=int(K))


def unfold_station_spectra(grid, H, fs_hz: float, v, theta_deg: float, phi_deg: float):
    """One station; also returns band spectra V0, V1, Et, Ep (each [K] complex128)."""
    H = _table(grid, H)
    v = np.ascontiguousarray(v, dtype=np.float64)
    two, N = v.shape
    k_lo, k_hi = band(N, fs_hz, grid.n_freq, grid.freq0_hz, grid.dfreq_hz)
    K = max(k_hi - k_lo + 1, 0)
    ef = np.empty((2, N)); e2 = np.empty(N); amp = C.c_double(); idx = C.c_int32()
    spec = np.zeros((4, max(K, 1), 2))
    g = _grid(grid)
    _lib.oracle_unfold_station_spectra(C.byref(g), _d(H.view(np.float64)), C.c_int(N), C.c_double(fs_hz),
                                       _d(v), C.c_double(theta_deg), C.c_double(phi_deg), _d(ef), _d(e2),
                                       C.byref(amp), C.byref(idx), _d(spec))
    sp = (spec[..., 0] + 1j * spec[..., 1])[:, :K]
    return dict(efield=ef, env2=e2, amp=float(amp.value), idx=int(idx.value), k_lo=k_lo, k_hi=k_hi,
                V0=sp[0], V1=sp[1], Et=sp[2], Ep=sp[3])


def scan(grid, H, fs_hz: float, traces, dirs, want_env2=False):
    """traces [S][2][N], dirs [D][2] -> amp [D][S], idx [D][S] int32 (and env2 [D][S][N] with want_env2)."""
    H = _table(grid, H)
    tr = np.ascontiguousarray(traces, dtype=np.float64)
    S, two, N = tr.shape
    dd = np.ascontiguousarray(dirs, dtype=np.float64)
    D = dd.shape[0]
    amp = np.empty((D, S)); idx = np.empty((D, S), dtype=np.int32)
    e2 = np.empty((D, S, N)) if want_env2 else None
    g = _grid(grid)
    _lib.oracle_scan(C.byref(g), _d(H.view(np.float64)), C.c_int(S), C.c_int(N), C.c_double(fs_hz),
                     _d(tr), C.c_long(D), _d(dd), _d(amp), idx.ctypes.data_as(_ip), _d(e2))
    return (amp, idx, e2) if want_env2 else (amp, idx)


def fold_station(grid, H, N: int, fs_hz: float, Et, Ep, theta_deg: float, phi_deg: float):
    """Band spectra Et, Ep [K] complex -> voltage traces v [2][N] (forward model, test helper)."""
    H = _table(grid, H)
    Et = np.asarray(Et, dtype=np.complex128); Ep = np.asarray(Ep, dtype=np.complex128)
    et = np.ascontiguousarray(np.stack([Et.real, Et.imag], axis=1))
    ep = np.ascontiguousarray(np.stack([Ep.real, Ep.imag], axis=1))
    v = np.empty((2, N))
    g = _grid(grid)
    _lib.oracle_fold_station(C.byref(g), _d(H.view(np.float64)), C.c_int(N), C.c_double(fs_hz),
                             _d(et), _d(ep), C.c_double(theta_deg), C.c_double(phi_deg), _d(v))
    return v
