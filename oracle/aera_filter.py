"""Oracle of the fused pre-filter (SURVEY.md 8f "next" row 4; "noise filtering and signal
enhancing", unspecified in the paper; reading R22): one real weight per in-band bin applied to
the unfolded spectra, E'[k] = w[k - k_lo] E[k], then the analytic signal, E-field and envelope peak exactly
as in the unfiltered path. TEST INFRASTRUCTURE ONLY. Plain composition of the C oracle's steps: the
unfiltered band spectra E (O1-O4), the weights, then O5-O7."""
from __future__ import annotations

import numpy as np

from . import aera_oracle as _o


def unfold_station_filtered(grid, H, fs_hz: float, v, theta_deg: float, phi_deg: float, weights):
    r = _o.unfold_station_spectra(grid, H, fs_hz, v, theta_deg, phi_deg)
    w = np.asarray(weights, dtype=np.float64)
    assert w.shape == r["Et"].shape
    N = np.asarray(v).shape[-1]
    zt = _o.analytic_from_band(r["Et"] * w, N, r["k_lo"], r["k_hi"])
    zp = _o.analytic_from_band(r["Ep"] * w, N, r["k_lo"], r["k_hi"])
    env2, amp, idx = _o.peak(zt, zp)
    return dict(efield=np.stack([zt.real, zp.real]), env2=env2, amp=amp, idx=idx)


def unfold_batch_filtered(grid, H, fs_hz: float, traces, dirs, weights):
    """traces [U][2][N], dirs [U][2] -> dict(efield [U][2][N], env2 [U][N], amp [U], idx [U])."""
    rs = [unfold_station_filtered(grid, H, fs_hz, traces[u], dirs[u][0], dirs[u][1], weights) for u in range(len(traces))]
    return dict(efield=np.stack([r["efield"] for r in rs]), env2=np.stack([r["env2"] for r in rs]),
                amp=np.array([r["amp"] for r in rs]), idx=np.array([r["idx"] for r in rs], dtype=np.int32))
