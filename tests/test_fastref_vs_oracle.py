"""Pins the harness-side numpy float64 pipeline (fastref.py, SURVEY.md 8c-B "secondary full-coverage
check") to the naive-DFT oracle on a subsample: E-field and amplitude <= 1e-12 relative, peak index equal,
band limits equal. Only then may the GPU tests use it to cover EVERY unit of the big configs."""
import numpy as np
import pytest

import aera_inputs as ai
import fastref
import oracle


@pytest.mark.parametrize("cfg,events,n_st", [(0, [0, 1, 2], None), (1, [0, 7], 6), (3, [3], 3)])
def test_fastref_matches_oracle(cfg, events, n_st):
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, events, n_stations=n_st)
    E, S = tr.shape[:2]
    trf = tr.reshape(E * S, 2, -1); dd = np.repeat(dirs, S, axis=0)
    ref = oracle.unfold_batch(wl.grid, H, wl.fs_hz, trf, dd, want_env2=True)
    got = fastref.unfold_units(wl.grid, H, wl.fs_hz, trf, dd)
    assert fastref.band_limits(wl.n_samples, wl.fs_hz, wl.grid) == oracle.band(wl.n_samples, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    for u in range(E * S):
        l2 = np.linalg.norm(got["efield"][u] - ref["efield"][u]) / np.linalg.norm(ref["efield"][u])
        assert l2 <= 1e-12, (cfg, u, l2)
    assert np.max(np.abs(got["amp"] - ref["amp"]) / ref["amp"]) <= 1e-12
    assert np.max(np.abs(got["env2"] - ref["env2"])) <= 1e-12 * np.max(ref["env2"])
    assert np.array_equal(got["idx"], ref["idx"])


def test_fastref_directions_wrap_clamp_and_nodes(small_grid, small_table):
    wl = ai.WORKLOADS[0]
    tr, _, _, _ = ai.make_batch(wl, range(8))
    dirs = np.array([[35.0, 125.0], [12.3, 359.9], [12.3, -10.0], [45.0, 725.0], [0.0, 0.0], [60.0, 360.0], [89.0, 200.0], [-5.0, 10.0]])
    trf = tr[:, 0]
    ref = oracle.unfold_batch(small_grid, small_table, wl.fs_hz, trf, dirs)
    got = fastref.unfold_units(small_grid, small_table, wl.fs_hz, trf, dirs)
    for u in range(len(dirs)):
        assert np.linalg.norm(got["efield"][u] - ref["efield"][u]) <= 1e-12 * np.linalg.norm(ref["efield"][u]), u
    assert np.array_equal(got["idx"], ref["idx"])


def test_check_all_units_counts_and_flags():
    """The all-unit checker classifies a correct output as exact and a shifted index as a miss."""
    wl = ai.WORKLOADS[0]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(3))
    E, S = tr.shape[:2]
    ref = fastref.unfold_units(wl.grid, H, wl.fs_hz, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0))
    ef = ref["efield"].reshape(E, S, 2, -1).astype(np.float32)
    amp = ref["amp"].reshape(E, S).astype(np.float32); idx = ref["idx"].reshape(E, S).copy()
    tol = dict(l2=1e-4, amp=1e-4, tie=1e-5)
    r = fastref.check_all_units(wl.grid, H, wl.fs_hz, tr, dirs, ef, amp, idx, tol, threads=2)
    assert r["n"] == E * S and r["exact"] == E * S and r["miss"] == 0 and r["max_l2"] < 1e-6 and r["max_amp"] < 1e-6
    idx[1, 2] += 7
    r = fastref.check_all_units(wl.grid, H, wl.fs_hz, tr, dirs, ef, amp, idx, tol, threads=2)
    assert r["exact"] == E * S - 1 and r["miss"] + r["ambiguous"] == 1 and r["bad"][0][:2] == (1, 2)
