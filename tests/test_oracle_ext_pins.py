"""Pins of oracle/aera_ext.py: per-station pattern tables, int16 ADC input, spectral
up-sampling. Each is pinned against something other than itself: the single-table oracle (bit for bit), exactly
representable count scales, closed forms (constant envelope of a cosine, half-sample pulse arrival) and
scipy.signal.resample (a library routine) for the zero-padded spectrum."""
import numpy as np
import scipy.signal

import aera_inputs as ai
import oracle
from oracle import aera_ext as ox


def _setup(n_events=2):
    wl = ai.WORKLOADS[0]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(n_events))
    return wl, H, tr, dirs


# ---------------------------------------------------------------- row 2: several tables
def test_identical_tables_give_the_single_table_result_bit_for_bit():
    wl, H, tr, dirs = _setup()
    E, S = tr.shape[:2]
    single = oracle.unfold_batch(wl.grid, H, wl.fs_hz, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0))
    multi = ox.unfold_batch_multi(wl.grid, [H, H.copy(), H.copy()], np.arange(S) % 3, wl.fs_hz, tr, dirs)
    assert np.array_equal(multi["efield"], single["efield"]) and np.array_equal(multi["amp"], single["amp"])
    assert np.array_equal(multi["idx"], single["idx"])


def test_each_station_is_unfolded_with_its_own_table():
    wl, H, tr, dirs = _setup()
    E, S = tr.shape[:2]
    H2 = ai.pattern_table(wl.grid, wl.complex_dtype, seed=99)           # another antenna type: other perturbation
    Hid = np.zeros(wl.grid.shape, dtype=np.complex64); Hid[0, 0] = 1.0; Hid[1, 1] = 1.0   # identity response
    pid = np.array([0, 1, 2, 1, 0, 2, 1])
    multi = ox.unfold_batch_multi(wl.grid, [H, H2, Hid], pid, wl.fs_hz, tr, dirs)
    k_lo, k_hi = oracle.band(wl.n_samples, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    for e in range(E):
        for s in range(S):
            tab = [H, H2, Hid][pid[s]]
            ref = oracle.unfold_batch(wl.grid, tab, wl.fs_hz, tr[e, s][None], dirs[e][None])
            assert np.array_equal(multi["efield"][e * S + s], ref["efield"][0])
            if pid[s] == 2:     # identity response: the unfolding is a brick-wall band-pass (numpy rfft / irfft)
                X = np.fft.rfft(tr[e, s].astype(np.float64), axis=-1); Y = np.zeros_like(X); Y[:, k_lo:k_hi + 1] = X[:, k_lo:k_hi + 1]
                bp = np.fft.irfft(Y, n=wl.n_samples, axis=-1)
                assert np.allclose(multi["efield"][e * S + s], bp, atol=1e-10 * np.abs(bp).max())
    assert not np.allclose(multi["efield"][1], oracle.unfold_batch(wl.grid, H, wl.fs_hz, tr[0, 1][None], dirs[0][None])["efield"][0], rtol=1e-3)


# ---------------------------------------------------------------- row 4: int16 input
def test_int16_counts_with_a_power_of_two_scale_equal_the_float_path_exactly():
    wl, H, tr, dirs = _setup(1)
    counts = np.clip(np.round(tr[0] * 8.0), -32768, 32767).astype(np.int16)      # 1/8 microvolt per count
    g = [0.125, 0.125]
    got = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, counts, g, np.repeat(dirs, 7, axis=0))
    ref = oracle.unfold_batch(wl.grid, H, wl.fs_hz, counts.astype(np.float64) * 0.125, np.repeat(dirs, 7, axis=0))
    assert np.array_equal(got["efield"], ref["efield"]) and np.array_equal(got["idx"], ref["idx"])


def test_int16_per_channel_scale_is_linear():
    wl, H, tr, dirs = _setup(1)
    counts = np.clip(np.round(tr[0] * 4.0), -32768, 32767).astype(np.int16)
    dd = np.repeat(dirs, 7, axis=0)
    a = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, counts, [0.25, 0.25], dd)
    b = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, counts, [0.5, 0.5], dd)
    assert np.allclose(b["efield"], 2.0 * a["efield"], rtol=1e-13) and np.array_equal(a["idx"], b["idx"])
    zero1 = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, counts, [0.25, 0.0], dd)     # channel 1 switched off
    c0 = counts.copy(); c0[:, 1] = 0
    assert np.array_equal(zero1["efield"], ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, c0, [0.25, 0.25], dd)["efield"])


# ---------------------------------------------------------------- row 4: spectral up-sampling
def test_upsampled_grid_contains_the_original_samples_and_matches_scipy_resample():
    wl, H, tr, dirs = _setup(1)
    th, ph = dirs[0]
    base = oracle.unfold_batch(wl.grid, H, wl.fs_hz, tr[0, :2], np.tile(dirs[0], (2, 1)), want_env2=True)
    for u in (1, 2, 4):
        up = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr[0, :2], np.tile(dirs[0], (2, 1)), u)
        assert up["efield"].shape == (2, 2, u * wl.n_samples)
        scale = np.abs(base["efield"]).max()
        assert np.max(np.abs(up["efield"][:, :, ::u] - base["efield"])) <= 1e-12 * scale       # z_up[u n] = z[n]
        assert np.max(np.abs(up["env2"][:, ::u] - base["env2"])) <= 1e-12 * base["env2"].max()
        ref = scipy.signal.resample(base["efield"], u * wl.n_samples, axis=-1)                   # FFT zero-padding (library)
        assert np.max(np.abs(up["efield"] - ref)) <= 1e-11 * scale
        assert np.all(up["amp"] >= base["amp"] * (1 - 1e-12))                                     # the fine grid can only find a higher peak


def test_filtered_upsampled_contains_the_filtered_samples_and_matches_scipy_resample():
    """The optional pre-filter weights of the up-sampling oracle: the fine grid through the filtered coarse samples
    (oracle/aera_filter.py, pinned on its own), scipy's FFT resampling of them, and weights of one = no weights."""
    from oracle import aera_filter as of
    wl, H, tr, dirs = _setup(1)
    dd = np.tile(dirs[0], (2, 1))
    k_lo, k_hi = oracle.band(wl.n_samples, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    rng = np.random.default_rng(11)
    w = 0.2 + 0.8 * rng.uniform(size=k_hi - k_lo + 1); w[[3, len(w) // 3, len(w) - 5]] = 0.0
    base = of.unfold_batch_filtered(wl.grid, H, wl.fs_hz, tr[0, :2], dd, w)
    plain = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr[0, :2], dd, 4)
    ones = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr[0, :2], dd, 4, np.ones_like(w))
    assert np.array_equal(plain["efield"], ones["efield"]) and np.array_equal(plain["idx"], ones["idx"])
    up = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr[0, :2], dd, 4, w)
    scale = np.abs(base["efield"]).max()
    assert np.max(np.abs(up["efield"] - plain["efield"])) > 1e-3 * scale                         # the weights do something
    assert np.max(np.abs(up["efield"][:, :, ::4] - base["efield"])) <= 1e-12 * scale
    assert np.max(np.abs(up["env2"][:, ::4] - base["env2"])) <= 1e-12 * base["env2"].max()
    ref = scipy.signal.resample(base["efield"], 4 * wl.n_samples, axis=-1)
    assert np.max(np.abs(up["efield"] - ref)) <= 1e-11 * scale


def test_upsampled_cosine_has_constant_envelope_and_half_sample_pulse_is_found():
    wl = ai.WORKLOADS[0]
    Hid = np.zeros(wl.grid.shape, dtype=np.complex128); Hid[0, 0] = 1.0; Hid[1, 1] = 1.0
    N = wl.n_samples; n = np.arange(N)
    k_lo, k_hi = oracle.band(N, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    m = k_lo + 7
    v = np.stack([3.0 * np.cos(2 * np.pi * m * n / N + 0.3), 4.0 * np.cos(2 * np.pi * m * n / N - 1.0)])
    up = ox.unfold_station_upsampled(wl.grid, Hid, wl.fs_hz, v, 10.0, 20.0, 4)
    assert np.max(np.abs(np.sqrt(up["env2"]) - 5.0)) < 1e-11
    # a band-limited pulse arriving at the half sample n0 = 100.5: on the 2x grid its envelope peaks at 201 with amplitude A
    k = np.arange(k_lo, k_hi + 1); w = np.exp(-0.5 * ((k - 70.0) / 9.0) ** 2); A = 250.0; n0 = 100.5
    Eb = A * (N / (2.0 * w.sum())) * w * np.exp(-2j * np.pi * k * n0 / N + 0.7j)
    X = np.zeros(N // 2 + 1, dtype=complex); X[k_lo:k_hi + 1] = Eb
    v = np.stack([np.fft.irfft(X, n=N), np.zeros(N)])
    up = ox.unfold_station_upsampled(wl.grid, Hid, wl.fs_hz, v, 10.0, 20.0, 2)
    assert up["idx"] == 201 and abs(up["amp"] - A) < 1e-9 * A
    coarse = ox.unfold_station_upsampled(wl.grid, Hid, wl.fs_hz, v, 10.0, 20.0, 1)
    assert coarse["idx"] in (100, 101) and coarse["amp"] < A
