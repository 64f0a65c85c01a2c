"""Pins of the reconstruction-loop oracle (oracle/aera_loop.py) against what geometry and the mathematics
fix -- not against itself: exact plane-wave times, invariances, a brute-force grid search, and an end-to-end
recovery of the injected direction from synthetic traces."""
import numpy as np
import pytest

import aera_inputs as ai
from oracle import aera_loop as ol

FS = 180e6


def _times(theta, phi, pos, t0=1000.0):
    th, ph = np.deg2rad(theta), np.deg2rad(phi)
    u, v = np.sin(th) * np.cos(ph), np.sin(th) * np.sin(ph)
    return t0 - FS * (u * pos[:, 0] + v * pos[:, 1]) / ol.C_LIGHT_M_PER_S


@pytest.mark.parametrize("theta,phi", [(0.0, 0.0), (10.0, 0.0), (35.0, 125.0), (74.9, 359.0), (60.0, 180.0), (20.0, 270.0)])
def test_exact_plane_wave_is_recovered(theta, phi):
    pos = ai.station_positions(31)
    th, ph = ol.planewave_fit(pos, _times(theta, phi, pos), np.ones(31), FS)
    assert abs(th - theta) < 1e-9
    if theta > 0:
        assert abs((ph - phi + 180.0) % 360.0 - 180.0) < 1e-8


def test_fit_is_invariant_under_time_offset_and_weight_scale_and_translation():
    pos = ai.station_positions(40)
    rng = np.random.default_rng(5)
    t = _times(42.0, 77.0, pos) + rng.normal(0, 0.7, size=40)      # noisy times
    w = rng.uniform(0.1, 3.0, size=40)
    a = ol.planewave_fit(pos, t, w, FS)
    assert np.allclose(a, ol.planewave_fit(pos, t + 123.0, w, FS), atol=1e-9)          # t0 absorbs a common delay
    assert np.allclose(a, ol.planewave_fit(pos, t, 17.0 * w, FS), atol=1e-9)           # only relative weights matter
    assert np.allclose(a, ol.planewave_fit(pos + [250.0, -90.0], t, w, FS), atol=1e-9) # array origin is arbitrary


def test_zero_weight_stations_are_ignored_and_no_weights_gives_zenith():
    pos = ai.station_positions(30)
    t = _times(30.0, 200.0, pos)
    w = np.ones(30); w[[3, 7, 19]] = 0.0
    t_bad = t.copy(); t_bad[[3, 7, 19]] += 500.0                    # outliers with zero weight
    th, ph = ol.planewave_fit(pos, t_bad, w, FS)
    assert abs(th - 30.0) < 1e-9 and abs(ph - 200.0) < 1e-8
    assert ol.planewave_fit(pos, t, np.zeros(30), FS) == (0.0, 0.0)


def test_fit_matches_brute_force_minimum_of_the_weighted_residual():
    """The fitted (u, v) minimises sum w (c t/fs - c t0 + u x + v y)^2 with t0 profiled out: compare with a
    dense grid search around it."""
    pos = ai.station_positions(25)
    rng = np.random.default_rng(9)
    t = _times(50.0, 310.0, pos) + rng.normal(0, 2.0, size=25)
    w = rng.uniform(0.2, 2.0, size=25)
    th, ph = ol.planewave_fit(pos, t, w, FS)
    b = ol.C_LIGHT_M_PER_S * t / FS

    def cost(u, v):
        r = b + u * pos[:, 0] + v * pos[:, 1]
        r = r - np.sum(w * r) / np.sum(w)
        return np.sum(w * r * r)
    u0, v0 = np.sin(np.deg2rad(th)) * np.cos(np.deg2rad(ph)), np.sin(np.deg2rad(th)) * np.sin(np.deg2rad(ph))
    c0 = cost(u0, v0)
    for du in np.linspace(-2e-3, 2e-3, 9):
        for dv in np.linspace(-2e-3, 2e-3, 9):
            assert cost(u0 + du, v0 + dv) >= c0 - 1e-9 * abs(c0)


def test_super_luminal_times_are_clamped_to_the_horizon():
    pos = ai.station_positions(20)
    t = 1000.0 - FS * 1.3 * pos[:, 0] / ol.C_LIGHT_M_PER_S          # |(u, v)| = 1.3 > 1
    th, ph = ol.planewave_fit(pos, t, np.ones(20), FS)
    assert abs(th - 90.0) < 1e-12 and abs((ph + 180.0) % 360.0 - 180.0) < 1e-7


def test_timing_from_voltages_lowest_index_and_both_channels():
    tr = np.zeros((3, 2, 64), dtype=np.float32)
    tr[0, 0, 10] = 3.0; tr[0, 1, 10] = 4.0; tr[0, 0, 40] = 4.9           # 25 at n = 10 beats 24.01 at n = 40
    tr[1, 1, 5] = -2.0; tr[1, 0, 50] = 2.0                                # tie: lowest index wins
    tr[2, 0, 63] = 1.0
    idx, w = ol.timing_from_voltages(tr)
    assert idx.tolist() == [10, 5, 63] and np.allclose(w, [25.0, 4.0, 1.0])


def test_loop_recovers_the_injected_direction_from_synthetic_traces(small_table):
    """End to end on configs[1]-shaped inputs with plane-wave arrivals: the direction after the E-field
    iterations lands within 1 degree of the injected one (the table's 5 % perturbation and the noise are
    the residual)."""
    wl = ai.WORKLOADS[1]
    pos = ai.station_positions(40)
    ev = ai.make_event(wl, 3, n_stations=40, positions=pos)
    r = ol.reconstruct_event(wl.grid, small_table, wl.fs_hz, ev.traces, pos, n_iter=2)
    th, ph = r["dirs"][-1]
    th0, ph0 = ev.direction_deg
    assert abs(th - th0) < 1.0 and abs((ph - ph0 + 180.0) % 360.0 - 180.0) < 2.0 / max(np.sin(np.deg2rad(th0)), 0.2)
    assert r["idx"].shape == (2, 40) and r["efield"].shape == (40, 2, wl.n_samples)


def test_convergence_iteration_closed_forms():
    """The angular distance is the great-circle angle (pole: azimuth irrelevant; equator: azimuth difference) and the
    criterion picks the first iteration within tolerance of its predecessor."""
    assert abs(ol.angular_distance_deg((0.0, 10.0), (0.0, 200.0))) < 1e-12            # both at the zenith
    assert abs(ol.angular_distance_deg((90.0, 10.0), (90.0, 40.0)) - 30.0) < 1e-12    # along the horizon
    assert abs(ol.angular_distance_deg((30.0, 77.0), (50.0, 77.0)) - 20.0) < 1e-12    # along a meridian
    assert abs(ol.angular_distance_deg((30.0, 359.9), (30.0, 0.1)) - 0.2 * np.sin(np.radians(30.0))) < 1e-6
    dirs = [(40.0, 100.0), (42.0, 101.0), (42.05, 101.0), (42.05, 101.0)]
    assert ol.convergence_iteration(dirs, 0.1) == 2 and ol.convergence_iteration(dirs, 1e-9) == 3
    assert ol.convergence_iteration(dirs[:2], 0.1) == -1 and ol.convergence_iteration(dirs, 5.0) == 1
