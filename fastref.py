"""Harness-side O(N log N) float64 reference of the unfolding path -- the SECONDARY full-coverage check of
SURVEY.md 8(c)-B, and the "fairer" CPU figure of 8(d-4) (the closest analogue of the paper's FFTW baseline,
PAPER.md L31, L59).

It is NOT the oracle and NOT the product: harness code beside aera_inputs.py (used by tests/ and by bench.py's
cpu_baseline leg), it imports neither oracle/ nor the CUDA package, and
is trusted only because tests/test_fastref_vs_oracle.py pins it to the naive-DFT oracle (<= 1e-12 relative) on
a subsample. Its job is coverage: the oracle costs O(N K) per unit and can only sample the big batches; this
pipeline (numpy.fft in float64) checks EVERY unit of configs 1, 3 and 4 against the CUDA output and counts
exact / near-tie / ambiguous peak indices.

Steps, per unit (same definition as include/aera_unfold.h):
  V_c = rfft(v_c); H(theta, phi, f_k) by 8-corner trilinear interpolation (Re and Im independently, azimuth
  periodic, zenith clamped); E = H^-1 V on the in-band bins (0 elsewhere, DC and Nyquist too; det == 0 -> 0);
  z_p = ifft of the one-sided spectrum 2 E_p; e_p = Re z_p; env2 = |z_theta|^2 + |z_phi|^2; first argmax.
"""
from __future__ import annotations

import os
from concurrent.futures import ThreadPoolExecutor
from fractions import Fraction

import numpy as np


def band_limits(N: int, fs_hz: float, grid) -> tuple[int, int]:
    """Inclusive in-band bins with f0 <= k fs / N <= f0 + (n_f - 1) df, 0 < k < N/2, in exact rationals."""
    fs, f0, df = Fraction(fs_hz), Fraction(grid.freq0_hz), Fraction(grid.dfreq_hz)
    f_hi = f0 + (grid.n_freq - 1) * df
    lo = -((-f0 * N) // fs)          # ceil
    hi = (f_hi * N) // fs            # floor
    return max(int(lo), 1), min(int(hi), N // 2 - 1)


def _cell(u, n):
    i = np.minimum(np.floor(u).astype(np.int64), n - 2)
    i = np.maximum(i, 0)
    return i, u - i


def response(grid, H, theta_deg: float, phi_deg: float, f_hz):
    """Trilinear H[2][2][K] complex128 at one direction and the frequencies f_hz [K]."""
    H = np.asarray(H)
    zmax = grid.zenith0_deg + (grid.n_zenith - 1) * grid.dzenith_deg
    th = min(max(theta_deg, grid.zenith0_deg), zmax)
    iz, tz = _cell(np.float64((th - grid.zenith0_deg) / grid.dzenith_deg), grid.n_zenith)
    if grid.azimuth_periodic:
        P = (grid.n_azimuth - 1) * grid.dazimuth_deg
        pw = phi_deg - P * np.floor((phi_deg - grid.azimuth0_deg) / P)
        ua = (pw - grid.azimuth0_deg) / grid.dazimuth_deg
        ia = int(np.floor(ua)); ta = ua - ia
        ia %= (grid.n_azimuth - 1)
        ia1 = (ia + 1) % (grid.n_azimuth - 1)
    else:
        amax = grid.azimuth0_deg + (grid.n_azimuth - 1) * grid.dazimuth_deg
        ph = min(max(phi_deg, grid.azimuth0_deg), amax)
        ia, ta = _cell(np.float64((ph - grid.azimuth0_deg) / grid.dazimuth_deg), grid.n_azimuth)
        ia = int(ia); ia1 = ia + 1
    iz = int(iz)
    jf, tf = _cell((np.asarray(f_hz, dtype=np.float64) - grid.freq0_hz) / grid.dfreq_hz, grid.n_freq)
    out = np.zeros((2, 2, len(jf)), dtype=np.complex128)
    for dz, wz in ((0, 1.0 - tz), (1, tz)):
        for a, wa in ((ia, 1.0 - ta), (ia1, ta)):
            row = H[:, :, iz + dz, a, :].astype(np.complex128)       # [2][2][n_f]
            out += (wz * wa) * ((1.0 - tf) * row[:, :, jf] + tf * row[:, :, jf + 1])
    return out


def unfold_units(grid, H, fs_hz: float, traces, dirs):
    """traces [U][2][N] (any real dtype), dirs [U][2] degrees -> dict(efield [U][2][N], env2 [U][N], amp, idx).
    Units that share a direction (the stations of an event) share one pattern evaluation."""
    tr = np.asarray(traces, dtype=np.float64)
    U, _, N = tr.shape
    k_lo, k_hi = band_limits(N, fs_hz, grid)
    k = np.arange(k_lo, k_hi + 1)
    V = np.fft.rfft(tr, axis=-1)[:, :, k_lo:k_hi + 1]                  # [U][2][K]
    dd = np.asarray(dirs, dtype=np.float64)
    E = np.zeros((U, 2, len(k)), dtype=np.complex128)
    uniq, inv = np.unique(dd, axis=0, return_inverse=True)
    inv = np.asarray(inv).ravel()
    for j, (th, ph) in enumerate(uniq):
        sel = np.nonzero(inv == j)[0]
        Hk = response(grid, H, float(th), float(ph), k * (fs_hz / N))
        det = Hk[0, 0] * Hk[1, 1] - Hk[0, 1] * Hk[1, 0]
        ok = det != 0
        inv_det = np.where(ok, 1.0 / np.where(ok, det, 1.0), 0.0)
        V0, V1 = V[sel, 0], V[sel, 1]
        E[sel, 0] = (Hk[1, 1] * V0 - Hk[0, 1] * V1) * inv_det
        E[sel, 1] = (Hk[0, 0] * V1 - Hk[1, 0] * V0) * inv_det
    Z = np.zeros((U, 2, N), dtype=np.complex128)
    Z[:, :, k_lo:k_hi + 1] = 2.0 * E
    z = np.fft.ifft(Z, axis=-1)
    env2 = z[:, 0].real ** 2 + z[:, 0].imag ** 2 + z[:, 1].real ** 2 + z[:, 1].imag ** 2
    idx = np.argmax(env2, axis=-1).astype(np.int32)                    # first occurrence of the maximum
    amp = np.sqrt(env2[np.arange(U), idx])
    return dict(efield=np.ascontiguousarray(z.real), env2=env2, amp=amp, idx=idx)


def check_all_units(grid, H, fs_hz, traces, dirs, gpu_efield, gpu_amp, gpu_idx, tol, threads: int | None = None):
    """Every unit of a batch against this pipeline. traces / gpu_efield [E][S][2][N] (numpy, any real dtype),
    dirs [E][2], gpu_amp / gpu_idx [E][S]. Events are processed by a thread pool (numpy's FFT and ufuncs release
    the GIL). Returns dict(n, max_l2, max_amp, exact, tie_pm1, ambiguous, miss, bad[list of (event, station, ref idx,
    gpu idx, gap)]) with the index rule of BASELINE north_star (exact, or +-1 when the reference envelope at the
    GPU's index is within tol["tie"] of the reference maximum)."""
    E, S = traces.shape[:2]
    threads = threads or min(32, os.cpu_count() or 1)

    def one(e):
        ref = unfold_units(grid, H, fs_hz, traces[e], np.repeat(np.asarray(dirs[e])[None], S, axis=0))
        out = dict(l2=0.0, amp=0.0, exact=0, tie=0, amb=0, miss=0, bad=[])
        if gpu_efield is not None:
            d = gpu_efield[e].astype(np.float64) - ref["efield"]
            l2 = np.sqrt((d ** 2).sum(axis=(1, 2)) / (ref["efield"] ** 2).sum(axis=(1, 2)))
            out["l2"] = float(l2.max())
        out["amp"] = float(np.max(np.abs(gpu_amp[e].astype(np.float64) - ref["amp"]) / ref["amp"]))
        gi = np.asarray(gpu_idx[e]).astype(np.int64); ri = ref["idx"].astype(np.int64)
        out["exact"] = int(np.sum(gi == ri))
        for s in np.nonzero(gi != ri)[0]:
            e2 = ref["env2"][s]
            gap = 1.0 - float(np.sqrt(e2[gi[s]] / e2[ri[s]])) if 0 <= gi[s] < len(e2) else 1.0
            if gap < tol["tie"] and abs(int(gi[s]) - int(ri[s])) <= 1:
                out["tie"] += 1
            else:
                out["amb" if gap < tol["tie"] else "miss"] += 1
                out["bad"].append((int(e), int(s), int(ri[s]), int(gi[s]), gap))
        return out

    with ThreadPoolExecutor(max_workers=threads) as ex:
        parts = list(ex.map(one, range(E)))
    return dict(n=E * S, max_l2=max(p["l2"] for p in parts), max_amp=max(p["amp"] for p in parts),
                exact=sum(p["exact"] for p in parts), tie_pm1=sum(p["tie"] for p in parts),
                ambiguous=sum(p["amb"] for p in parts), miss=sum(p["miss"] for p in parts),
                bad=[b for p in parts for b in p["bad"]])
