"""Oracle of the remaining "next" rows of SURVEY.md 8(f) -- TEST INFRASTRUCTURE ONLY (see oracle/__init__.py).

Plain compositions of the C oracle's pinned steps (aera_oracle.c), one function per feature:

  row 2  several pattern tables, one antenna type per station (section 3: "The patterns for all
         antennas used in AERA can be stored simultaneously on the device"; L43: "For each antenna, the VEL is
         known ..."): every station is unfolded with ITS OWN table; nothing else changes.
  row 4  int16 ADC-count input (the voltage traces "are read out" by the station electronics as ADC
         counts; the paper does not give the conversion): v_c[n] = counts_to_volts[c] * counts_c[n], exactly, in
         double; then the unfolding as it stands.
  row 4  spectral up-sampling by zero-padding ("noise filtering and signal enhancing", unspecified;
         DESIGN.md reading R23): the unfolded band spectrum E[k] is unchanged, the analytic signal is evaluated on a
         grid u times finer,  z_p[n] = (2/N) sum_{k in band} E_p[k] exp(+2 pi i n k / (u N)),  n = 0 .. uN-1,
         so z_up[u n] = z[n]; E-field, envelope and its peak are taken on the fine grid (peak index in fine samples).
"""
from __future__ import annotations

import numpy as np

from . import aera_oracle as _o


def unfold_batch_multi(grid, tables, pattern_id, fs_hz: float, traces, dirs, want_env2=False):
    """traces [E][S][2][N], dirs [E][2], tables = list of H[2][2][n_z][n_a][n_f] on the same grid,
    pattern_id [S] ints (antenna type of each station). -> dict as oracle.unfold_batch over the E*S units."""
    tr = np.asarray(traces)
    E, S, _, N = tr.shape
    pid = np.asarray(pattern_id, dtype=np.int64)
    assert pid.shape == (S,) and pid.min() >= 0 and pid.max() < len(tables)
    ef = np.empty((E * S, 2, N)); amp = np.empty(E * S); idx = np.empty(E * S, dtype=np.int32)
    e2 = np.empty((E * S, N)) if want_env2 else None
    dd = np.asarray(dirs, dtype=np.float64)
    for p, H in enumerate(tables):
        st = np.nonzero(pid == p)[0]
        if st.size == 0:
            continue
        units = (np.arange(E)[:, None] * S + st[None, :]).ravel()
        r = _o.unfold_batch(grid, H, fs_hz, tr[:, st].reshape(-1, 2, N), np.repeat(dd, st.size, axis=0), want_env2=want_env2)
        ef[units] = r["efield"]; amp[units] = r["amp"]; idx[units] = r["idx"]
        if want_env2:
            e2[units] = r["env2"]
    return dict(efield=ef, env2=e2, amp=amp, idx=idx)


def unfold_batch_i16(grid, H, fs_hz: float, counts, counts_to_volts, dirs, want_env2=False):
    """counts [U][2][N] int16, counts_to_volts [2] (per channel), dirs [U][2] -> dict as oracle.unfold_batch."""
    c = np.asarray(counts)
    assert c.dtype == np.int16
    g = np.asarray(counts_to_volts, dtype=np.float64).reshape(2)
    v = c.astype(np.float64) * g[None, :, None]
    return _o.unfold_batch(grid, H, fs_hz, v, dirs, want_env2=want_env2)


def unfold_station_upsampled(grid, H, fs_hz: float, v, theta_deg: float, phi_deg: float, upsample: int, weights=None):
    """One station, analytic signal on a grid `upsample` times finer. -> dict(efield [2][uN], env2 [uN], amp, idx).
    weights (optional, [K] real): the pre-filter of oracle/aera_filter.py, E'[k] = w[k - k_lo] E[k], applied to the band
    spectra before the fine-grid transform (the band, hence the weights, do not depend on the up-sampling factor)."""
    u = int(upsample)
    assert u >= 1
    r = _o.unfold_station_spectra(grid, H, fs_hz, v, theta_deg, phi_deg)       # O1-O4: the band spectra E_theta, E_phi
    if weights is not None:
        w = np.asarray(weights, dtype=np.float64)
        assert w.shape == r["Et"].shape
        r = dict(r, Et=r["Et"] * w, Ep=r["Ep"] * w)
    N = np.asarray(v).shape[-1]
    M = u * N
    # O5 on the fine grid: oracle.analytic_from_band(E, M, ...) = (2/M) sum_k E[k] exp(+2 pi i n k / M); times u gives 2/N
    zt = u * _o.analytic_from_band(r["Et"], M, r["k_lo"], r["k_hi"])
    zp = u * _o.analytic_from_band(r["Ep"], M, r["k_lo"], r["k_hi"])
    env2, amp, idx = _o.peak(zt, zp)                                             # O7
    return dict(efield=np.stack([zt.real, zp.real]), env2=env2, amp=amp, idx=idx)


def unfold_batch_upsampled(grid, H, fs_hz: float, traces, dirs, upsample: int, weights=None):
    """traces [U][2][N], dirs [U][2] -> dict(efield [U][2][uN], env2 [U][uN], amp [U], idx [U])."""
    rs = [unfold_station_upsampled(grid, H, fs_hz, traces[i], dirs[i][0], dirs[i][1], upsample, weights) for i in range(len(traces))]
    return dict(efield=np.stack([r["efield"] for r in rs]), env2=np.stack([r["env2"] for r in rs]),
                amp=np.array([r["amp"] for r in rs]), idx=np.array([r["idx"] for r in rs], dtype=np.int32))
