"""Pins for the CPU oracle (oracle/aera_oracle.c) against facts that are not the oracle itself:
library routines (numpy.fft, scipy.signal.hilbert, scipy RegularGridInterpolator,
numpy.linalg.solve), closed forms, invariants and the paper's printed numbers.
Citations: PAPER.md L29, L43-45, L59-63, L71; SURVEY.md section 8(c)-B.
"""
import os

import numpy as np
import pytest
import scipy.interpolate
import scipy.signal

import aera_inputs as ai
import oracle

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


# ---------------------------------------------------------------- O1: forward DFT
@pytest.mark.parametrize("N", [8, 16, 60, 64, 256])
def test_dft_matches_library_fft(N):
    rng = np.random.default_rng(N)
    x = rng.standard_normal(N)
    X = oracle.dft_band(x, 0, N - 1)
    ref = np.fft.fft(x)
    assert np.max(np.abs(X - ref)) <= 1e-12 * np.max(np.abs(ref))


def test_dft_delta_and_cosine_closed_forms():
    N = 64
    for m in (0, 1, 5, 63):
        x = np.zeros(N); x[m] = 1.0
        X = oracle.dft_band(x, 0, N - 1)
        k = np.arange(N)
        # delta[n-m] -> exp(-2 pi i m k / N): sign and index convention (FFTW forward)
        assert np.max(np.abs(X - np.exp(-2j * np.pi * ((m * k) % N) / N))) < 1e-14
    m = 7
    x = np.cos(2 * np.pi * m * np.arange(N) / N)
    X = oracle.dft_band(x, 0, N - 1)
    assert abs(X[m] - N / 2) < 1e-12 and abs(X[N - m] - N / 2) < 1e-12
    X[m] = 0; X[N - m] = 0
    assert np.max(np.abs(X)) < 1e-12
    # a sine lands on -i N/2: fixes the sign of the imaginary part
    x = np.sin(2 * np.pi * m * np.arange(N) / N)
    assert abs(oracle.dft_band(x, m, m)[0] - (-0.5j * N)) < 1e-12


def test_dft_parseval_and_linearity():
    N = 128
    rng = np.random.default_rng(1)
    x = rng.standard_normal(N); y = rng.standard_normal(N)
    X = oracle.dft_band(x, 0, N // 2)
    lhs = np.sum(x * x)
    rhs = (abs(X[0]) ** 2 + 2 * np.sum(abs(X[1:N // 2]) ** 2) + abs(X[N // 2]) ** 2) / N
    assert abs(lhs - rhs) < 1e-11 * lhs
    Z = oracle.dft_band(2.0 * x - 3.0 * y, 3, 40)
    assert np.max(np.abs(Z - (2.0 * oracle.dft_band(x, 3, 40) - 3.0 * oracle.dft_band(y, 3, 40)))) < 1e-11


def test_twiddle_table_is_accurate_and_unit_modulus():
    N = 65536
    W = oracle.twiddles(N)
    assert np.max(np.abs(np.abs(W) - 1.0)) < 3e-16
    # exact values at the octants
    assert W[0] == 1.0 and abs(W[N // 4] - (-1j)) < 1e-16 and abs(W[N // 2] + 1.0) < 1e-16
    assert abs(W[N // 8] - (1 - 1j) / np.sqrt(2)) < 2e-16


# ---------------------------------------------------------------- O2: band
def test_band_limits_golden():
    rows = [l.split() for l in open(os.path.join(GOLDEN, "band_limits.txt")) if l.strip() and not l.startswith("#")]
    assert len(rows) == 5
    for cfg, N, fs, nf, f0, df, klo, khi, K in rows:
        lo, hi = oracle.band(int(N), float(fs), int(nf), float(f0), float(df))
        assert (lo, hi) == (int(klo), int(khi)), cfg
        assert hi - lo + 1 == int(K)
        wl = ai.WORKLOADS[int(cfg)]
        assert (wl.n_samples, wl.fs_hz, wl.grid.n_freq) == (int(N), float(fs), int(nf))


def test_band_edges_inclusive_and_dc_nyquist_excluded():
    # bins exactly on both edges: fs=64, N=64 -> f_k = k; table 4..10 Hz
    assert oracle.band(64, 64.0, 7, 4.0, 1.0) == (4, 10)
    # a table reaching DC / Nyquist never yields k=0 or k=N/2 (convention R4: parity unpinned)
    assert oracle.band(64, 64.0, 33, 0.0, 1.0) == (1, 31)
    # empty band
    lo, hi = oracle.band(64, 64.0, 2, 100.0, 1.0)
    assert hi < lo


# ---------------------------------------------------------------- O3: pattern interpolation
def test_interp_reproduces_grid_nodes_exactly(small_grid, small_table):
    g, H = small_grid, small_table
    rng = np.random.default_rng(2)
    for _ in range(50):
        iz = rng.integers(0, g.n_zenith); ia = rng.integers(0, g.n_azimuth); jf = rng.integers(0, g.n_freq)
        got = oracle.pattern_eval(g, H, g.zenith_deg[iz], g.azimuth_deg[ia], g.freq_hz[jf])
        want = H[:, :, iz, ia, jf].astype(np.complex128)
        assert np.array_equal(got, want)  # bit-exact: weights are exactly 1 and 0


def _multilinear_table(g):
    z = g.zenith_deg[:, None, None]; a = g.azimuth_deg[None, :, None]; f = g.freq_hz[None, None, :] / 1e6
    H = np.empty(g.shape, dtype=np.complex128)
    coef = np.random.default_rng(3).standard_normal((4, 8, 2))
    fn = []
    for cp in range(4):
        c = coef[cp, :, 0] + 1j * coef[cp, :, 1]
        def F(z, a, f, c=c):
            return (c[0] + c[1] * z + c[2] * a + c[3] * f + c[4] * z * a + c[5] * z * f + c[6] * a * f + c[7] * z * a * f)
        fn.append(F)
        H[cp // 2, cp % 2] = F(z, a, f)
    return H, fn


def test_interp_reproduces_multilinear_function():
    g = ai.PatternGrid(19, 0.0, 5.0, 73, 0.0, 5.0, 41, 30e6, 1.25e6, azimuth_periodic=False)
    H, fn = _multilinear_table(g)
    rng = np.random.default_rng(4)
    for _ in range(200):
        th = rng.uniform(0, 90); ph = rng.uniform(0, 360); f = rng.uniform(30e6, 80e6)
        got = oracle.pattern_eval(g, H, th, ph, f).ravel()
        want = np.array([F(th, ph, f / 1e6) for F in fn])
        assert np.max(np.abs(got - want)) <= 1e-12 * np.max(np.abs(want))


def test_interp_cell_centre_is_mean_of_corners(small_grid, small_table):
    g, H = small_grid, small_table
    iz, ia, jf = 3, 71, 10  # ia=71: upper azimuth neighbour is node 72 == node 0 (periodic)
    got = oracle.pattern_eval(g, H, g.zenith_deg[iz] + 2.5, g.azimuth_deg[ia] + 2.5, g.freq_hz[jf] + 0.625e6)
    corners = H[:, :, iz:iz + 2, [71, 0], jf:jf + 2].astype(np.complex128)
    assert np.max(np.abs(got - corners.mean(axis=(2, 3, 4)))) < 1e-15


def test_interp_azimuth_periodic_and_zenith_clamped(small_grid, small_table):
    g, H = small_grid, small_table
    a = oracle.pattern_eval(g, H, 33.3, 123.4, 51e6)
    for shift in (-720.0, -360.0, 360.0, 720.0):
        b = oracle.pattern_eval(g, H, 33.3, 123.4 + shift, 51e6)
        assert np.max(np.abs(a - b)) < 1e-13
    assert np.array_equal(oracle.pattern_eval(g, H, 20.0, 360.0, 40e6), oracle.pattern_eval(g, H, 20.0, 0.0, 40e6))
    # crossing 360: continuous, and 358 deg uses nodes 355 and 0
    got = oracle.pattern_eval(g, H, 10.0, 358.0, 30e6)
    want = 0.4 * H[:, :, 2, 71, 0].astype(np.complex128) + 0.6 * H[:, :, 2, 0, 0].astype(np.complex128)
    assert np.max(np.abs(got - want)) < 1e-15
    # zenith outside the table clamps (convention R12: parity unpinned)
    assert np.array_equal(oracle.pattern_eval(g, H, 95.0, 10.0, 40e6), oracle.pattern_eval(g, H, 90.0, 10.0, 40e6))
    assert np.array_equal(oracle.pattern_eval(g, H, -3.0, 10.0, 40e6), oracle.pattern_eval(g, H, 0.0, 10.0, 40e6))


def test_interp_matches_scipy_regular_grid(small_grid, small_table):
    g, H = small_grid, small_table
    Hd = H.astype(np.complex128)
    rgi = [scipy.interpolate.RegularGridInterpolator((g.zenith_deg, g.azimuth_deg, g.freq_hz), Hd[c, p], method="linear")
           for c in range(2) for p in range(2)]
    rng = np.random.default_rng(5)
    for _ in range(100):
        th = rng.uniform(0, 90); ph = rng.uniform(0, 360); f = rng.uniform(30e6, 80e6)
        got = oracle.pattern_eval(g, H, th, ph, f).ravel()
        want = np.array([r([[th, ph, f]])[0] for r in rgi])
        assert np.max(np.abs(got - want)) <= 1e-13


def test_paper_table_size_and_error_estimate():
    facts = {}
    for l in open(os.path.join(GOLDEN, "paper_facts.txt")):
        if l.strip() and not l.startswith("#"):
            k, v = l.split("#")[0].split()
            facts[k] = float(v)
    g = ai.PatternGrid(31, 0.0, 3.0, 49, 0.0, 7.5, 98, 30e6, 0.5e6)
    # one antenna = one channel: [pol 2][n_z][n_a][n_f] complex64
    assert int(np.prod(g.shape[2:])) == int(facts["largest_pattern_nodes"])
    mb = g.nbytes(8) / 2 / 1e6
    assert abs(mb - facts["largest_pattern_mb_fp32"]) < 0.05
    assert abs(21 * 2.0 ** -23 * 100 - facts["fp32_interp_rel_error_percent"]) < 0.01e-4


# ---------------------------------------------------------------- O4: solve
def test_solve_matches_linalg():
    rng = np.random.default_rng(6)
    for _ in range(100):
        Hm = rng.standard_normal((2, 2)) + 1j * rng.standard_normal((2, 2))
        v = rng.standard_normal(2) + 1j * rng.standard_normal(2)
        e, ok = oracle.solve2x2(Hm, v)
        assert ok
        assert np.max(np.abs(e - np.linalg.solve(Hm, v))) < 1e-12 * np.max(np.abs(e))
    e, ok = oracle.solve2x2(np.array([[1, 2], [2, 4]], dtype=complex), np.array([1, 1], dtype=complex))
    assert not ok and np.all(e == 0)  # convention R8: parity unpinned


# ---------------------------------------------------------------- O4+O5: fold -> unfold round trip
@pytest.mark.parametrize("direction", [(35.0, 125.0), (0.0, 0.0), (37.3, 201.7), (74.9, 359.2)])
def test_fold_unfold_round_trip(small_grid, small_table, direction):
    g, H = small_grid, small_table
    N, fs = 256, 200e6
    k_lo, k_hi = oracle.band(N, fs, g.n_freq, g.freq0_hz, g.dfreq_hz)
    K = k_hi - k_lo + 1
    rng = np.random.default_rng(7)
    Et = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    Ep = rng.standard_normal(K) + 1j * rng.standard_normal(K)
    v = oracle.fold_station(g, H, N, fs, Et, Ep, *direction)
    r = oracle.unfold_station_spectra(g, H, fs, v, *direction)
    assert np.max(np.abs(r["Et"] - Et)) <= 1e-10 * np.max(np.abs(Et))
    assert np.max(np.abs(r["Ep"] - Ep)) <= 1e-10 * np.max(np.abs(Ep))
    # time domain: e_p = irfft of the band spectrum (library routine)
    full = np.zeros(N // 2 + 1, dtype=complex); full[k_lo:k_hi + 1] = Et
    et = np.fft.irfft(full, n=N)
    assert np.linalg.norm(r["efield"][0] - et) <= 1e-10 * np.linalg.norm(et)


# ---------------------------------------------------------------- whole pipeline, H == identity
def test_identity_pattern_reduces_to_bandpass_hilbert():
    g = ai.PatternGrid(3, 0.0, 45.0, 5, 0.0, 90.0, 41, 30e6, 1.25e6)
    H = np.zeros(g.shape, dtype=np.complex128)
    H[0, 0] = 1.0; H[1, 1] = 1.0
    N, fs = 512, 200e6
    rng = np.random.default_rng(8)
    v = rng.standard_normal((3, 2, N))
    dirs = np.array([[10.0, 20.0], [50.0, 300.0], [0.0, 0.0]])
    r = oracle.unfold_batch(g, H, fs, v, dirs, want_env2=True)
    k_lo, k_hi = oracle.band(N, fs, g.n_freq, g.freq0_hz, g.dfreq_hz)
    for u in range(3):
        V = np.fft.rfft(v[u], axis=-1)
        V[:, :k_lo] = 0; V[:, k_hi + 1:] = 0
        e = np.fft.irfft(V, n=N, axis=-1)
        z = scipy.signal.hilbert(e, axis=-1)
        env2 = np.sum(np.abs(z) ** 2, axis=0)
        assert np.linalg.norm(r["efield"][u] - e) <= 1e-12 * np.linalg.norm(e)
        assert np.max(np.abs(r["env2"][u] - env2)) <= 1e-12 * env2.max()
        assert r["idx"][u] == int(np.argmax(env2))
        assert abs(r["amp"][u] - np.sqrt(env2.max())) <= 1e-12 * r["amp"][u]


# ---------------------------------------------------------------- O5-O7: envelope
def test_cosine_envelope_is_constant():
    g = ai.PatternGrid(3, 0.0, 45.0, 5, 0.0, 90.0, 41, 30e6, 1.25e6)
    H = np.zeros(g.shape, dtype=np.complex128); H[0, 0] = 1.0; H[1, 1] = 1.0
    N, fs = 256, 200e6
    n = np.arange(N)
    A, m, psi = 3.0, 60, 0.7  # bin 60 = 46.9 MHz, in band
    v = np.stack([A * np.cos(2 * np.pi * m * n / N + psi), np.zeros(N)])[None]
    r = oracle.unfold_batch(g, H, fs, v, np.array([[0.0, 0.0]]), want_env2=True)
    assert np.max(np.abs(np.sqrt(r["env2"][0]) - A)) < 1e-12
    assert abs(r["amp"][0] - A) < 1e-12


def test_pulse_peak_amplitude_and_index():
    g = ai.PatternGrid(3, 0.0, 45.0, 5, 0.0, 90.0, 41, 30e6, 1.25e6)
    H = np.zeros(g.shape, dtype=np.complex128); H[0, 0] = 1.0; H[1, 1] = 1.0
    N, fs = 256, 200e6
    k_lo, k_hi = oracle.band(N, fs, g.n_freq, g.freq0_hz, g.dfreq_hz)
    k = np.arange(k_lo, k_hi + 1)
    w = np.exp(-0.5 * ((k * fs / N - 55e6) / 12.5e6) ** 2)
    A, n0, psi, alpha = 100.0, 100, 1.1, 0.4
    Eh = A * (N / (2 * w.sum())) * w * np.exp(-2j * np.pi * k * n0 / N + 1j * psi)
    v = oracle.fold_station(g, H, N, fs, Eh * np.cos(alpha), Eh * np.sin(alpha), 0.0, 0.0)
    r = oracle.unfold_batch(g, H, fs, v[None], np.array([[0.0, 0.0]]))
    assert r["idx"][0] == n0
    assert abs(r["amp"][0] - A) < 1e-10


def test_peak_tie_takes_lowest_index():
    zt = np.array([0, 3, 0, 3, 1], dtype=complex); zp = np.array([0, 4j, 0, -4, 0], dtype=complex)
    env2, amp, idx = oracle.peak(zt, zp)
    assert idx == 1 and amp == 5.0 and np.array_equal(env2, [0, 25, 0, 25, 1])


# ---------------------------------------------------------------- scan == batch per direction
def test_scan_equals_batch_per_direction(small_grid, small_table):
    g, H = small_grid, small_table
    wl = ai.WORKLOADS[0]
    ev = ai.make_event(wl, 0)
    dirs = np.array([[0.0, 0.0], [12.0, 358.0], [44.0, 91.0], [80.0, 180.0]])
    amp, idx = oracle.scan(g, H, wl.fs_hz, ev.traces, dirs)
    for d in range(len(dirs)):
        r = oracle.unfold_batch(g, H, wl.fs_hz, ev.traces, np.repeat(dirs[d][None], wl.n_stations, axis=0))
        assert np.array_equal(idx[d], r["idx"])
        assert np.max(np.abs(amp[d] - r["amp"])) <= 1e-13 * np.max(r["amp"])
    # the optional squared-envelope output (used by the scan parity tests for the near-tie rule) is the batch
    # oracle's env2 and is consistent with the returned peaks
    amp2, idx2, e2 = oracle.scan(g, H, wl.fs_hz, ev.traces, dirs, want_env2=True)
    assert np.array_equal(amp2, amp) and np.array_equal(idx2, idx) and e2.shape == (len(dirs), wl.n_stations, wl.n_samples)
    for d in range(len(dirs)):
        r = oracle.unfold_batch(g, H, wl.fs_hz, ev.traces, np.repeat(dirs[d][None], wl.n_stations, axis=0), want_env2=True)
        assert np.max(np.abs(e2[d] - r["env2"])) <= 1e-12 * np.max(r["env2"])
    assert np.array_equal(np.argmax(e2, axis=-1), idx) and np.array_equal(np.sqrt(np.max(e2, axis=-1)), amp)


# ---------------------------------------------------------------- generator sanity (no method arithmetic)
def test_generator_is_seeded_and_shaped():
    wl = ai.WORKLOADS[0]
    a = ai.make_event(wl, 0); b = ai.make_event(wl, 0); c = ai.make_event(wl, 1)
    assert a.traces.shape == (7, 2, 256) and a.traces.dtype == np.float32
    assert np.array_equal(a.traces, b.traces) and not np.array_equal(a.traces, c.traces)
    H = ai.pattern_table(wl.grid, np.complex64)
    assert H.shape == (2, 2, 19, 73, 41) and H.dtype == np.complex64
    assert np.array_equal(H[:, :, :, 72, :], H[:, :, :, 0, :])
    d = ai.scan_directions()
    assert d.shape == (7380, 2) and d[0].tolist() == [0.0, 0.0] and d[-1].tolist() == [80.0, 358.0]


def test_strong_pulses_recovered_near_injection(small_grid, small_table):
    """Plausibility of the whole chain on config-0 data (table is a 5 % perturbed version of the
    response used for synthesis): strong pulses peak within a few samples of n0, amplitude within 15 %."""
    wl = ai.WORKLOADS[0]
    tr, dirs, A, n0 = ai.make_batch(wl, range(6))
    U = tr.shape[0] * tr.shape[1]
    r = oracle.unfold_batch(small_grid, small_table, wl.fs_hz, tr.reshape(U, 2, -1),
                            np.repeat(dirs, wl.n_stations, axis=0), want_efield=False)
    strong = A.ravel() > 300.0
    assert strong.sum() >= 5
    assert np.all(np.abs(r["idx"][strong] - n0.ravel()[strong]) <= 3)
    assert np.all(np.abs(r["amp"][strong] / A.ravel()[strong] - 1.0) < 0.15)
