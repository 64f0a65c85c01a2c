"""Oracle of the device-resident reconstruction loop (SURVEY.md 8f "next" row 1; Fig. 1:
"First, as an initial estimate of the event timing in each station, the maxima of the voltage traces is
used. Second, from the timing information of the individual stations, the direction of the shower is obtained
by triangulation. Third, the antenna pattern for this direction is evaluated, and the E-field trace at each
station reconstructed from the voltage traces. Finally, the maximum of the envelope of the E-field trace is
used as updated timing information for a new iteration of the procedure."; L83 names keeping the data on the GPU as the remedy for copy-dominated run time).

TEST INFRASTRUCTURE ONLY (see oracle/__init__.py): plain numpy in float64, one step per function, in
the paper's order. The per-station unfolding inside the loop is oracle.unfold_batch (aera_oracle.c).

Readings where the paper is silent (R19-R21):
  R19 timing from voltages : n_i = lowest n maximising v0[n]^2 + v1[n]^2 (both channels of a station)
  R20 triangulation        : flat array, plane wave from direction (theta, phi):
                             c n_i / fs = c t0 - (u x_i + v y_i), (u, v) = sin(theta) (cos(phi), sin(phi)),
                             weighted linear least squares for (c t0, u, v) with weights w_i = (peak
                             amplitude of station i)^2; theta = asin(min(1, |(u, v)|)), phi = atan2(v, u) in [0, 360)
  R21 iteration            : a fixed number of iterations (the convergence test is the caller's)
"""
from __future__ import annotations

import numpy as np

from . import aera_oracle as _o

C_LIGHT_M_PER_S = 299792458.0


def timing_from_voltages(traces):
    """traces [S][2][N] -> (idx [S] int32, w [S] float64): R19."""
    v = np.asarray(traces, dtype=np.float64)
    p = v[:, 0, :] ** 2 + v[:, 1, :] ** 2
    idx = np.argmax(p, axis=1).astype(np.int32)          # numpy returns the first (lowest) maximum
    return idx, p[np.arange(p.shape[0]), idx]


def planewave_fit(positions, n_samples_idx, weights, fs_hz: float):
    """R20. positions [S][2] metres, arrival samples [S], weights [S] >= 0 -> (theta_deg, phi_deg)."""
    xy = np.asarray(positions, dtype=np.float64)
    b = C_LIGHT_M_PER_S * np.asarray(n_samples_idx, dtype=np.float64) / fs_hz
    w = np.asarray(weights, dtype=np.float64)
    if not np.any(w > 0):
        return 0.0, 0.0
    A = np.stack([np.ones(len(b)), -xy[:, 0], -xy[:, 1]], axis=1)
    sw = np.sqrt(w)
    sol, *_ = np.linalg.lstsq(A * sw[:, None], b * sw, rcond=None)
    u, v = float(sol[1]), float(sol[2])
    s = np.hypot(u, v)
    theta = np.degrees(np.arcsin(min(s, 1.0)))
    phi = np.degrees(np.arctan2(v, u))
    if phi < 0:
        phi += 360.0
    return float(theta), float(phi)


def reconstruct_event(grid, H, fs_hz: float, traces, positions, n_iter: int):
    """One event. traces [S][2][N]. Returns dict(idx0, w0, dirs [n_iter][2], amp [n_iter][S], idx [n_iter][S],
    efield [S][2][N] of the last iteration)."""
    S = traces.shape[0]
    idx0, w0 = timing_from_voltages(traces)
    t, w = idx0.astype(np.float64), w0
    dirs, amps, idxs, last = [], [], [], None
    for _ in range(n_iter):
        th, ph = planewave_fit(positions, t, w, fs_hz)
        dirs.append((th, ph))
        last = _o.unfold_batch(grid, H, fs_hz, traces, np.tile([th, ph], (S, 1)))
        amps.append(last["amp"].copy()); idxs.append(last["idx"].copy())
        t, w = last["idx"].astype(np.float64), last["amp"] ** 2
    return dict(idx0=idx0, w0=w0, dirs=np.array(dirs), amp=np.array(amps), idx=np.array(idxs),
                efield=last["efield"] if last is not None else None)


def angular_distance_deg(d0, d1):
    """Angle between two arrival directions (theta, phi in degrees) on the unit sphere, in degrees."""
    t0, p0, t1, p1 = np.radians([d0[0], d0[1], d1[0], d1[1]])
    a = np.array([np.sin(t0) * np.cos(p0), np.sin(t0) * np.sin(p0), np.cos(t0)])
    b = np.array([np.sin(t1) * np.cos(p1), np.sin(t1) * np.sin(p1), np.cos(t1)])
    return float(np.degrees(np.arctan2(np.linalg.norm(np.cross(a, b)), np.dot(a, b))))


def convergence_iteration(dirs, tol_deg: float) -> int:
    """"On convergence, the timing information yields the incident direction ...". The paper gives no
    criterion (reading R21): the loop has converged at the first iteration it >= 1 whose fitted direction lies
    within tol_deg (angle on the sphere) of the previous iteration's; -1 if none does. dirs [n_iter][2] degrees."""
    d = np.asarray(dirs, dtype=np.float64)
    for it in range(1, len(d)):
        if angular_distance_deg(d[it - 1], d[it]) < tol_deg:
            return it
    return -1
