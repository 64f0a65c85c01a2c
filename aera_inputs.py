"""Seeded synthetic inputs for the AERA E-field unfolding path (arXiv 1507.07733).

This module is the ONLY code shared by the CPU oracle's tests and the CUDA
path's tests/bench.  It holds none of the method's arithmetic: no DFT of the
method, no table interpolation, no 2x2 solve, no envelope.  It only *makes
inputs*:

  * the tabulated antenna response H[channel][pol][zenith][azimuth][freq]
    (BASELINE.json configs[0]: analytic dipole-like response times a seeded
    10 % perturbation; stands in for the measured/simulated VEL tables of
    PAPER.md L43-45, which are not available),
  * per-event shower directions (one per event),
  * per-station two-channel voltage traces: a band-limited E-field pulse
    pushed through the *analytic* (unperturbed, un-interpolated) antenna
    response at the event direction with numpy's irfft, plus Gaussian noise.

Using the analytic response for the synthesis (instead of interpolating the
perturbed table) keeps the method's interpolation out of this module; the
consequence is that an unfolded pulse differs from the injected one by the
table's ~5 % perturbation, like a real antenna-model uncertainty would
(reading R16).

Everything is a pure function of (config id, event index) through
`numpy.random.default_rng([7733, config, event])`, so any event can be
regenerated alone for the oracle subsample.
"""
from __future__ import annotations

from dataclasses import dataclass

import numpy as np

PATTERN_SEED = 1507
EVENT_SEED = 7733


@dataclass(frozen=True)
class PatternGrid:
    """Uniform (zenith, azimuth, frequency) node grid; angles in degrees, f in Hz."""

    n_zenith: int
    zenith0_deg: float
    dzenith_deg: float
    n_azimuth: int
    azimuth0_deg: float
    dazimuth_deg: float
    n_freq: int
    freq0_hz: float
    dfreq_hz: float
    azimuth_periodic: bool = True

    @property
    def shape(self):
        return (2, 2, self.n_zenith, self.n_azimuth, self.n_freq)

    @property
    def zenith_deg(self):
        return self.zenith0_deg + self.dzenith_deg * np.arange(self.n_zenith)

    @property
    def azimuth_deg(self):
        return self.azimuth0_deg + self.dazimuth_deg * np.arange(self.n_azimuth)

    @property
    def freq_hz(self):
        return self.freq0_hz + self.dfreq_hz * np.arange(self.n_freq)

    def nbytes(self, complex_itemsize: int) -> int:
        return int(np.prod(self.shape)) * complex_itemsize


@dataclass(frozen=True)
class Workload:
    """One BASELINE.json config."""

    config: int
    name: str
    n_events: int
    n_stations: int
    n_samples: int
    fs_hz: float
    dtype: str  # "f32" | "f64"
    grid: PatternGrid
    zenith_max_deg: float
    arrival_lo: float
    arrival_hi: float
    noise_sigma: float
    scan: bool = False

    @property
    def real_dtype(self):
        return np.float32 if self.dtype == "f32" else np.float64

    @property
    def complex_dtype(self):
        return np.complex64 if self.dtype == "f32" else np.complex128

    @property
    def n_units(self):
        return self.n_events * self.n_stations


_GRID_5DEG = PatternGrid(19, 0.0, 5.0, 73, 0.0, 5.0, 41, 30e6, 1.25e6)
_GRID_1DEG = PatternGrid(91, 0.0, 1.0, 361, 0.0, 1.0, 101, 30e6, 0.5e6)
_GRID_LONG = PatternGrid(19, 0.0, 5.0, 73, 0.0, 5.0, 181, 20e6, 1.0e6)

WORKLOADS = {
    0: Workload(0, "tiny-pr1", 1, 7, 256, 200e6, "f32", _GRID_5DEG, 60.0, 64, 192, 5.0),
    1: Workload(1, "aera-batch", 1000, 124, 2048, 180e6, "f32", _GRID_5DEG, 75.0, 512, 1536, 5.0),
    2: Workload(2, "direction-scan", 1, 124, 2048, 180e6, "f32", _GRID_5DEG, 75.0, 512, 1536, 5.0, scan=True),
    3: Workload(3, "fp64-batch", 10000, 40, 4096, 200e6, "f64", _GRID_1DEG, 75.0, 512, 1536, 2.0),
    4: Workload(4, "long-trace", 100, 124, 65536, 1e9, "f32", _GRID_LONG, 75.0, 16384, 49152, 5.0),
}

PULSE_F_LO_HZ = 30e6
PULSE_F_HI_HZ = 80e6
PULSE_F_C_HZ = 55e6
PULSE_SIGMA_HZ = 12.5e6


def antenna_L(f_hz):
    """Band-pass-like frequency response L(f)=1/(1+3i(f/55-55/f)), f in MHz (configs[0])."""
    f = np.asarray(f_hz, dtype=np.float64) / 1e6
    return 1.0 / (1.0 + 3.0j * (f / 55.0 - 55.0 / f))


def analytic_response(theta_deg, phi_deg, f_hz):
    """Unperturbed analytic H[c][p] at arbitrary (theta, phi, f). Returns [2][2][...] complex128."""
    th = np.deg2rad(np.asarray(theta_deg, dtype=np.float64))
    ph = np.deg2rad(np.asarray(phi_deg, dtype=np.float64))
    L = antenna_L(f_hz)
    th, ph, L = np.broadcast_arrays(th, ph, L)
    H = np.empty((2, 2) + L.shape, dtype=np.complex128)
    H[0, 0] = L * np.cos(th) * np.cos(ph)
    H[0, 1] = -L * np.sin(ph)
    H[1, 0] = L * np.cos(th) * np.sin(ph)
    H[1, 1] = L * np.cos(ph)
    return H


def pattern_table(grid: PatternGrid, complex_dtype=np.complex64, seed: int = PATTERN_SEED):
    """Tabulated H[2][2][n_z][n_a][n_f]: analytic values x (1 + 0.1 (a + i b)), a,b ~ U(-0.5,0.5).

    Generated in double, azimuth node n_a-1 overwritten with node 0 AFTER the
    perturbation when the axis is periodic, rounded once to the
    requested complex dtype.
    """
    z = grid.zenith_deg[:, None, None]
    a = grid.azimuth_deg[None, :, None]
    f = grid.freq_hz[None, None, :]
    H = analytic_response(z, a, f)
    rng = np.random.default_rng(seed)
    ab = rng.uniform(-0.5, 0.5, size=H.shape + (2,))
    H *= 1.0 + 0.1 * (ab[..., 0] + 1j * ab[..., 1])
    if grid.azimuth_periodic:
        H[:, :, :, grid.n_azimuth - 1, :] = H[:, :, :, 0, :]
    return np.ascontiguousarray(H.astype(complex_dtype))


def scan_directions(theta_max_deg=80.0, step_deg=2.0):
    """configs[2]: theta = 0,2,...,80 (41) x phi = 0,2,...,358 (180), theta-major. [D][2] float64."""
    th = np.arange(0.0, theta_max_deg + 0.5 * step_deg, step_deg)
    ph = np.arange(0.0, 360.0 - 0.5 * step_deg, step_deg)
    T, P = np.meshgrid(th, ph, indexing="ij")
    return np.ascontiguousarray(np.stack([T.ravel(), P.ravel()], axis=1))


@dataclass
class Event:
    direction_deg: np.ndarray  # [2] (zenith, azimuth)
    traces: np.ndarray  # [n_stations][2][N] real dtype
    amplitude: np.ndarray  # [n_stations] injected envelope peak A
    arrival: np.ndarray  # [n_stations] injected (real-valued) arrival sample n0
    pol_angle: np.ndarray  # [n_stations]


C_LIGHT_M_PER_S = 299792458.0


def station_positions(n_stations: int = 124, spacing_m: float = 125.0, seed: int = 23) -> np.ndarray:
    """[S][2] (x, y) in metres: a jittered square grid centred on the origin (stand-in for the AERA
    layout of PAPER.md L23: 124 stations; the real positions are not available). With 125 m spacing the
    array spans ~1.4 km, so at fs = 180 MHz a plane wave at 75 deg zenith spreads the arrival samples by
    about +-400 around the trace centre."""
    side = int(np.ceil(np.sqrt(n_stations)))
    rng = np.random.default_rng([PATTERN_SEED, seed])
    ij = np.stack(np.meshgrid(np.arange(side), np.arange(side), indexing="ij"), axis=-1).reshape(-1, 2)[:n_stations]
    xy = (ij - (side - 1) / 2.0) * spacing_m + rng.uniform(-0.25, 0.25, size=(n_stations, 2)) * spacing_m
    return np.ascontiguousarray(xy, dtype=np.float64)


def plane_wave_arrival(wl: Workload, theta_deg: float, phi_deg: float, positions: np.ndarray) -> np.ndarray:
    """Arrival sample of a plane wave coming FROM direction (theta, phi) at each station of a flat array:
    n0_i = N/2 - fs (u x_i + v y_i) / c, (u, v) = sin(theta) (cos(phi), sin(phi)). Pure geometry of the inputs;
    the method's own direction fit lives in the oracle and in the CUDA library."""
    th, ph = np.deg2rad(theta_deg), np.deg2rad(phi_deg)
    u, v = np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph)
    return wl.n_samples / 2.0 - wl.fs_hz * (u * positions[:, 0] + v * positions[:, 1]) / C_LIGHT_M_PER_S


def make_event(wl: Workload, event: int, n_stations: int | None = None, positions: np.ndarray | None = None) -> Event:
    """Generate one event of workload `wl` (seed [7733, config, event]). With `positions` [S][2] the pulse
    arrival samples follow a plane wave from the event direction (reconstruction-loop inputs) instead of
    being drawn uniformly."""
    S = wl.n_stations if n_stations is None else n_stations
    N = wl.n_samples
    # config 2 is "one event drawn by the config-1 generator"
    seed_cfg = 1 if wl.config == 2 else wl.config
    rng = np.random.default_rng([EVENT_SEED, seed_cfg, event])
    theta = rng.uniform(0.0, wl.zenith_max_deg)
    phi = rng.uniform(0.0, 360.0)
    A = np.exp(rng.uniform(np.log(10.0), np.log(1000.0), size=S))
    n0 = rng.uniform(wl.arrival_lo, wl.arrival_hi, size=S)
    if positions is not None:
        n0 = plane_wave_arrival(wl, theta, phi, np.asarray(positions)[:S])
    psi = rng.uniform(0.0, 2 * np.pi, size=S)
    alpha = rng.uniform(0.0, 2 * np.pi, size=S)

    k = np.arange(N // 2 + 1)
    f = k * (wl.fs_hz / N)
    inband = (f >= PULSE_F_LO_HZ) & (f <= PULSE_F_HI_HZ) & (k > 0) & (k < N // 2)
    w = np.where(inband, np.exp(-0.5 * ((f - PULSE_F_C_HZ) / PULSE_SIGMA_HZ) ** 2), 0.0)
    c = N / (2.0 * w.sum())
    kb = k[inband]
    Hb = analytic_response(theta, phi, f[inband])  # [2][2][Kb]
    # E spectrum of each station on the pulse band
    ph = np.exp(-2j * np.pi * np.outer(n0, kb) / N + 1j * psi[:, None])  # [S][Kb]
    Eh = (A[:, None] * c) * w[inband][None, :] * ph
    Eth = Eh * np.cos(alpha)[:, None]
    Eph = Eh * np.sin(alpha)[:, None]
    V = np.zeros((S, 2, N // 2 + 1), dtype=np.complex128)
    V[:, 0, inband] = Hb[0, 0][None, :] * Eth + Hb[0, 1][None, :] * Eph
    V[:, 1, inband] = Hb[1, 0][None, :] * Eth + Hb[1, 1][None, :] * Eph
    v = np.fft.irfft(V, n=N, axis=-1)
    v += wl.noise_sigma * rng.standard_normal(size=v.shape)
    return Event(
        direction_deg=np.array([theta, phi], dtype=np.float64),
        traces=np.ascontiguousarray(v.astype(wl.real_dtype)),
        amplitude=A,
        arrival=n0,
        pol_angle=alpha,
    )


def make_batch(wl: Workload, events, n_stations: int | None = None):
    """Stack events -> (traces [E][S][2][N], dirs [E][2] float64, amplitude [E][S], arrival [E][S])."""
    evs = [make_event(wl, int(e), n_stations) for e in events]
    traces = np.stack([e.traces for e in evs])
    dirs = np.stack([e.direction_deg for e in evs])
    amp = np.stack([e.amplitude for e in evs])
    arr = np.stack([e.arrival for e in evs])
    return traces, dirs, amp, arr


def _event_worker(args):
    cfg, ev, n_st = args
    e = make_event(WORKLOADS[cfg], ev, n_st)
    return e.traces, e.direction_deg, e.amplitude, e.arrival


def make_batch_parallel(wl: Workload, events, n_stations: int | None = None, workers: int | None = None,
                        out_traces=None):
    """make_batch with a process pool (input synthesis only). `out_traces` may be a preallocated
    [E][S][2][N] array (e.g. a view of pinned memory) that receives the traces."""
    import concurrent.futures as cf
    import os

    events = [int(e) for e in events]
    S = wl.n_stations if n_stations is None else n_stations
    if out_traces is None:
        out_traces = np.empty((len(events), S, 2, wl.n_samples), dtype=wl.real_dtype)
    dirs = np.empty((len(events), 2)); amp = np.empty((len(events), S)); arr = np.empty((len(events), S))
    workers = workers or min(32, os.cpu_count() or 1)
    if workers <= 1 or len(events) < 4:
        for i, e in enumerate(events):
            out_traces[i], dirs[i], amp[i], arr[i] = _event_worker((wl.config, e, n_stations))
        return out_traces, dirs, amp, arr
    with cf.ProcessPoolExecutor(max_workers=workers) as ex:
        for i, r in enumerate(ex.map(_event_worker, [(wl.config, e, n_stations) for e in events], chunksize=8)):
            out_traces[i], dirs[i], amp[i], arr[i] = r
    return out_traces, dirs, amp, arr
