"""Pins of the pre-filter oracle (oracle/aera_filter.py): unit weights reproduce the unfiltered oracle, a
notch removes exactly the cosine sitting on that bin, the filter is linear in the weights, and with H = identity
it equals numpy's rfft -> weights -> irfft (a library routine)."""
import numpy as np

import aera_inputs as ai
import oracle
from oracle import aera_filter as of


def _setup():
    wl = ai.WORKLOADS[0]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    ev = ai.make_event(wl, 0)
    k_lo, k_hi = oracle.band(wl.n_samples, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    return wl, H, ev, k_lo, k_hi


def test_unit_weights_reproduce_the_unfiltered_oracle():
    wl, H, ev, k_lo, k_hi = _setup()
    th, ph = ev.direction_deg
    ref = oracle.unfold_batch(wl.grid, H, wl.fs_hz, ev.traces[:3], np.tile([th, ph], (3, 1)))
    got = of.unfold_batch_filtered(wl.grid, H, wl.fs_hz, ev.traces[:3], np.tile([th, ph], (3, 1)), np.ones(k_hi - k_lo + 1))
    assert np.allclose(got["efield"], ref["efield"], rtol=0, atol=1e-12 * np.abs(ref["efield"]).max())
    assert np.array_equal(got["idx"], ref["idx"]) and np.allclose(got["amp"], ref["amp"], rtol=1e-13)


def test_identity_response_equals_rfft_weights_irfft():
    wl, _, ev, k_lo, k_hi = _setup()
    Hid = np.zeros(wl.grid.shape, dtype=np.complex128); Hid[0, 0] = 1.0; Hid[1, 1] = 1.0
    rng = np.random.default_rng(3)
    w = rng.uniform(0.0, 1.0, k_hi - k_lo + 1); w[5] = 0.0
    v = ev.traces[0].astype(np.float64)
    got = of.unfold_station_filtered(wl.grid, Hid, wl.fs_hz, v, 20.0, 100.0, w)
    X = np.fft.rfft(v, axis=-1); Y = np.zeros_like(X); Y[:, k_lo:k_hi + 1] = X[:, k_lo:k_hi + 1] * w
    ref = np.fft.irfft(Y, n=wl.n_samples, axis=-1)
    assert np.allclose(got["efield"], ref, atol=1e-10 * np.abs(ref).max())


def test_notch_removes_a_cosine_on_that_bin_and_weights_act_linearly():
    wl, _, ev, k_lo, k_hi = _setup()
    Hid = np.zeros(wl.grid.shape, dtype=np.complex128); Hid[0, 0] = 1.0; Hid[1, 1] = 1.0
    N = wl.n_samples; m = k_lo + 11
    n = np.arange(N)
    v = np.stack([3.0 * np.cos(2 * np.pi * m * n / N + 0.4), 2.0 * np.sin(2 * np.pi * m * n / N)])
    w = np.ones(k_hi - k_lo + 1)
    full = of.unfold_station_filtered(wl.grid, Hid, wl.fs_hz, v, 10.0, 10.0, w)
    assert abs(full["amp"] - np.hypot(3.0, 2.0)) < 1e-10          # envelope of a pure in-band cosine pair is constant
    w[11] = 0.0
    assert np.abs(of.unfold_station_filtered(wl.grid, Hid, wl.fs_hz, v, 10.0, 10.0, w)["efield"]).max() < 1e-10
    w[11] = 0.25
    assert np.allclose(of.unfold_station_filtered(wl.grid, Hid, wl.fs_hz, v, 10.0, 10.0, w)["efield"], 0.25 * full["efield"], atol=1e-12)
