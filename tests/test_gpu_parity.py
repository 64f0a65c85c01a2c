"""GPU parity tests: the CUDA path (through the C ABI) against the CPU oracle on identical seeded
inputs. Run on the B200 box: python -m pytest tests -m gpu -x -q
"""
import numpy as np
import pytest
import torch

import aera_inputs as ai

pytestmark = pytest.mark.gpu

from parity import TOL, assert_peaks, compare, compare_peaks  # noqa: E402


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


@pytest.fixture(scope="module")
def orc():
    import oracle
    return oracle


_tables = {}


def table_for(wl):
    key = (wl.grid, wl.dtype)
    if key not in _tables:
        _tables[key] = ai.pattern_table(wl.grid, wl.complex_dtype)
    return _tables[key]


def run_gpu_batch(B, wl, H, traces, dirs, variant=0, inplace=False, want_efield=True):
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        tr = torch.from_numpy(traces).cuda()
        dd = torch.from_numpy(dirs).cuda()
        ef, amp, idx = B.aera_unfold_batch(pat, tr, dd, wl.fs_hz, efield=tr if inplace else None, want_efield=want_efield)
        torch.cuda.synchronize()
        out = (ef.cpu().numpy() if ef is not None else None, amp.cpu().numpy(), idx.cpu().numpy())
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    return out


def oracle_batch(orc, wl, H, traces, dirs):
    E, S = traces.shape[:2]
    return orc.unfold_batch(wl.grid, H, wl.fs_hz, traces.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0), want_env2=True)


def check(wl, gpu, ref):
    ef, amp, idx = gpu
    U = len(ref["amp"])
    rep = compare(wl.dtype, ef.reshape(U, 2, -1) if ef is not None else None, amp.ravel(), idx.ravel(), ref)
    print(f"\n[parity cfg{wl.config}] {rep}")
    assert rep.ok(TOL[wl.dtype]), str(rep)
    return rep


@pytest.mark.parametrize("variant", [0, 1])
def test_config0_all_units(B, orc, variant):
    wl = ai.WORKLOADS[0]
    H = table_for(wl)
    tr, dirs, _, _ = ai.make_batch(wl, [0])
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, variant), oracle_batch(orc, wl, H, tr, dirs))


@pytest.mark.parametrize("variant", [0, 1])
def test_config1_subsample(B, orc, variant):
    wl = ai.WORKLOADS[1]
    H = table_for(wl)
    events = [0, 1, 17, 999]
    tr, dirs, _, _ = ai.make_batch(wl, events)
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, variant), oracle_batch(orc, wl, H, tr, dirs))


@pytest.mark.parametrize("variant", [0, 1])
def test_config3_fp64_subsample(B, orc, variant):
    wl = ai.WORKLOADS[3]
    H = table_for(wl)
    events = [0, 1, 2, 3, 5000, 9999, 42]
    tr, dirs, _, _ = ai.make_batch(wl, events)
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, variant), oracle_batch(orc, wl, H, tr, dirs))


@pytest.mark.parametrize("variant", [0, 1])
def test_config4_long_trace_subsample(B, orc, variant):
    wl = ai.WORKLOADS[4]
    H = table_for(wl)
    n_st = 8 if variant == 0 else 4
    tr, dirs, _, _ = ai.make_batch(wl, [0], n_stations=n_st)
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, variant), oracle_batch(orc, wl, H, tr, dirs))


@pytest.mark.parametrize("variant", [0, 1])
def test_config2_scan(B, orc, variant):
    wl = ai.WORKLOADS[2]
    H = table_for(wl)
    ev = ai.make_event(wl, 0)
    alld = ai.scan_directions()
    rng = np.random.default_rng(2)
    pick = set(rng.choice(len(alld), size=58, replace=False).tolist())
    # the four grid corners, phi = 358 (periodic wrap) and a theta = 80 row
    pick |= {0, 179, len(alld) - 180, len(alld) - 1, 20 * 180 + 179, 40 * 180 + 90}
    dirs = alld[sorted(pick)]
    assert len(dirs) >= 64
    dt = B.AERA_F32
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(ev.traces).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    oamp, oidx, oe2 = orc.scan(wl.grid, H, wl.fs_hz, ev.traces, dirs, want_env2=True)
    rep = compare_peaks(wl.dtype, amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2)
    print(f"\n[parity cfg2 scan variant {variant}: {len(dirs)} directions x {ev.traces.shape[0]} stations] {rep}")
    assert_peaks(rep, wl.dtype)


def test_config2_scan_ragged_tiles(B, orc):
    """Scan tiles are 4 stations x 3 directions: 7 stations x 10 directions leaves both tails ragged."""
    wl = ai.WORKLOADS[2]
    H = table_for(wl)
    ev = ai.make_event(wl, 0)
    tr = np.ascontiguousarray(ev.traces[5:12])
    dirs = ai.scan_directions()[[3, 181, 400, 777, 1500, 2999, 3000, 5000, 7000, 7379]]
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
    finally:
        pat.free()
    oamp, oidx, oe2 = orc.scan(wl.grid, H, wl.fs_hz, tr, dirs, want_env2=True)
    rep = compare_peaks(wl.dtype, amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2)
    print(f"\n[parity cfg2 scan ragged] {rep}")
    assert_peaks(rep, wl.dtype)


# ------------------------------------------------------------------ sizes and edge cases
@pytest.mark.parametrize("dtype", ["f32", "f64"])
@pytest.mark.parametrize("N", [64, 128, 256, 512, 1024, 2048, 4096, 8192])
def test_all_sizes_small_batch(B, orc, N, dtype):
    """Every supported power of two up to 8192 (16384-65536 are covered by config 4), ragged batch:
    3 events x 5 stations; fs chosen so the band keeps ~N/4 bins."""
    base = ai.WORKLOADS[0]
    wl = ai.Workload(90, "sizes", 3, 5, N, 200e6, dtype, base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(3))
    check(wl, run_gpu_batch(B, wl, H, tr, dirs), oracle_batch(orc, wl, H, tr, dirs))


def test_directions_wrap_clamp_and_nodes(B, orc):
    wl = ai.WORKLOADS[0]
    H = table_for(wl)
    tr, _, _, _ = ai.make_batch(wl, range(8))
    dirs = np.array([[35.0, 125.0],      # exactly a grid node
                     [12.3, 359.9],      # last azimuth cell, wraps to node 0
                     [12.3, -10.0],      # negative azimuth
                     [45.0, 725.0],      # two periods up
                     [0.0, 0.0],         # table corner
                     [60.0, 360.0],      # phi == period
                     [89.0, 200.0],      # near the singular theta = 90 nodes (still regular)
                     [-5.0, 10.0]])      # clamped zenith
    check(wl, run_gpu_batch(B, wl, H, tr, dirs), oracle_batch(orc, wl, H, tr, dirs))


def test_inplace_and_peaks_only(B, orc):
    wl = ai.WORKLOADS[1]
    H = table_for(wl)
    tr, dirs, _, _ = ai.make_batch(wl, [3], n_stations=9)
    ref = oracle_batch(orc, wl, H, tr, dirs)
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, inplace=True), ref)
    ef, amp, idx = run_gpu_batch(B, wl, H, tr, dirs, want_efield=False)
    assert ef is None
    check(wl, (None, amp, idx), ref)


def test_zero_events_and_errors(B):
    wl = ai.WORKLOADS[0]
    H = table_for(wl)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        tr = torch.zeros((0, 7, 2, 256), device="cuda")
        dd = torch.zeros((0, 2), dtype=torch.float64, device="cuda")
        ef, amp, idx = B.aera_unfold_batch(pat, tr, dd, wl.fs_hz)
        assert amp.numel() == 0
        tr = torch.zeros((1, 7, 2, 256), device="cuda")
        dd = torch.zeros((1, 2), dtype=torch.float64, device="cuda")
        with pytest.raises(B.AeraError) as e:
            B.aera_unfold_batch(pat, torch.zeros((1, 7, 2, 200), device="cuda"), dd, wl.fs_hz, workspace=B.alloc_workspace(1 << 20))
        assert e.value.status == 2
        with pytest.raises(B.AeraError) as e:
            B.aera_unfold_batch(pat, tr.double(), dd, wl.fs_hz, workspace=B.alloc_workspace(1 << 20))
        assert e.value.status == 3
        with pytest.raises(B.AeraError) as e:
            B.aera_unfold_batch(pat, tr, dd, wl.fs_hz, workspace=B.alloc_workspace(256))
        assert e.value.status == 4
        with pytest.raises(B.AeraError) as e:  # band reaches Nyquist: fs = 150 MHz < 2 * 80 MHz
            B.aera_unfold_batch(pat, tr, dd, 150e6, workspace=B.alloc_workspace(1 << 20))
        assert e.value.status == 7
        with pytest.raises(B.AeraError) as e:  # misaligned traces
            B.aera_unfold_batch(pat, torch.zeros(1 * 7 * 2 * 256 + 1, device="cuda")[1:].view(1, 7, 2, 256), dd, wl.fs_hz)
        assert e.value.status == 1
        assert B.aera_band(pat, 256, 200e6) == (39, 102)
    finally:
        pat.free()


def test_host_pipeline_matches_device_path(B):
    wl = ai.WORKLOADS[1]
    H = table_for(wl)
    tr, dirs, _, _ = ai.make_batch(wl, range(6), n_stations=31)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        t_h = torch.from_numpy(tr).pin_memory(); d_h = torch.from_numpy(dirs).pin_memory()
        ef_h, amp_h, idx_h = B.aera_unfold_batch_host(pat, t_h, d_h, wl.fs_hz)
        ef_d, amp_d, idx_d = B.aera_unfold_batch(pat, t_h.cuda(), d_h.cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef_h, ef_d.cpu()) and torch.equal(amp_h, amp_d.cpu()) and torch.equal(idx_h, idx_d.cpu())
    finally:
        pat.free()


def test_library_is_loaded_and_counts_launches(B):
    n0 = B.aera_launch_count()
    wl = ai.WORKLOADS[0]
    tr, dirs, _, _ = ai.make_batch(wl, [0])
    run_gpu_batch(B, wl, table_for(wl), tr, dirs)
    assert B.aera_launch_count() >= n0 + 3  # repack + minv + unfold
    assert B.LIBRARY_PATH.endswith("libaera_unfold.so")


# ------------------------------------------------------------------ full sizes, bench.py's launch configuration
def _full_size_case(B, orc, cfg, n_events, sample_units, n_canon):
    """The whole batch of a config in ONE call, exactly as bench.py launches it (same input builder: a
    canonical block of seeded events tiled to the batch); sampled units are checked one by one against the
    oracle, every unit against properties that hold at any size (finite, index in range, tiled copies of the
    same event give bit-identical results)."""
    import bench
    wl = ai.WORKLOADS[cfg]
    H = table_for(wl)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    # same builders as bench.py: the whole batch staged on the host, or (configs[3], 26 GB) the canonical block
    # tiled on the device; host_tr holds the events 0 .. n_host-1, and event e equals event e % n_canon
    n_canon = min(n_canon, n_events)
    if n_events * wl.n_stations * 2 * wl.n_samples * (4 if wl.dtype == "f32" else 8) <= bench.HOST_BATCH_LIMIT:
        host_tr, host_dirs, _, _ = bench.build_inputs(wl, n_events, 0, pinned=False, n_canon=n_canon)
        d_tr = host_tr.cuda()
    else:
        host_tr, d_tr, host_dirs, _, _ = bench.build_inputs_device(wl, n_events, 0, n_canon=n_canon)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        ef, amp, idx = B.aera_unfold_batch(pat, d_tr, host_dirs.cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        amp_h = amp.cpu().numpy(); idx_h = idx.cpu().numpy()
        assert np.isfinite(amp_h).all() and (amp_h > 0).all()
        assert (idx_h >= 0).all() and (idx_h < wl.n_samples).all()
        if n_events >= 2 * n_canon:     # event e and e + n_canon are the same input at different addresses
            assert np.array_equal(amp_h[:n_canon], amp_h[n_canon:2 * n_canon])
            assert np.array_equal(idx_h[:n_canon], idx_h[n_canon:2 * n_canon])
            assert torch.equal(ef[0], ef[n_canon])
        S = wl.n_stations
        ev_ids = sorted({u // S for u in sample_units})
        tr_s = np.stack([host_tr[(u // S) % n_canon, u % S].numpy() for u in sample_units])
        dirs_s = np.stack([host_dirs[u // S].numpy() for u in sample_units])
        ref = orc.unfold_batch(wl.grid, H, wl.fs_hz, tr_s, dirs_s, want_env2=True)
        ef_s = np.stack([ef[u // S, u % S].cpu().numpy() for u in sample_units])
        rep = compare(wl.dtype, ef_s, np.array([amp_h[u // S, u % S] for u in sample_units]),
                      np.array([idx_h[u // S, u % S] for u in sample_units]), ref)
        print(f"\n[full-size cfg{cfg}: {n_events} events x {S} stations, {len(sample_units)} sampled units, events {ev_ids[:4]}..] {rep}")
        assert rep.ok(TOL[wl.dtype]), str(rep)
    finally:
        pat.free()


def test_full_size_config1(B, orc):
    rng = np.random.default_rng(11)
    units = sorted(set(rng.integers(0, 124000, size=2048).tolist()) | {0, 123999, 837, 838})   # incl. a CTA boundary
    _full_size_case(B, orc, 1, 1000, units, n_canon=200)


def test_full_size_config3(B, orc):
    """BASELINE configs[3] at its stated size: 10 000 events x 40 stations = 400 000 units (26 GB in, 26 GB out)."""
    rng = np.random.default_rng(13)
    units = sorted(set(rng.integers(0, 10000 * 40, size=512).tolist()) | {0, 399999, 2702, 2703})   # incl. a CTA boundary
    _full_size_case(B, orc, 3, 10000, units, n_canon=1000)    # bench.py's builder and size for configs[3]


def test_full_size_config4(B, orc):
    rng = np.random.default_rng(17)
    units = sorted(set(rng.integers(0, 12400, size=13).tolist()) | {0, 5000, 12399})
    _full_size_case(B, orc, 4, 100, units, n_canon=100)


@pytest.mark.parametrize("cfg,n_events,n_st", [(1, 40, 124), (3, 30, 40), (4, 2, 124)])
def test_repeated_runs_are_bit_identical(B, cfg, n_events, n_st):
    """Race check by determinism (compute-sanitizer is not available on the GPU pool): the kernels have no
    atomics on floating-point data, so repeated launches on the same input must agree bit for bit; a missing
    barrier between the shared-memory / tensor-memory / L2-scratch phases would show up as a mismatch."""
    wl = ai.WORKLOADS[cfg]
    H = table_for(wl)
    tr, dirs, _, _ = ai.make_batch(wl, range(min(n_events, 4)), n_stations=n_st)
    reps = -(-n_events // tr.shape[0])
    tr = np.concatenate([tr] * reps)[:n_events]; dirs = np.concatenate([dirs] * reps)[:n_events]
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        d_tr = torch.from_numpy(tr).cuda(); d_dirs = torch.from_numpy(dirs).cuda()
        ref = None
        for _ in range(6):
            ef, amp, idx = B.aera_unfold_batch(pat, d_tr, d_dirs, wl.fs_hz)
            torch.cuda.synchronize()
            if ref is None:
                ref = (ef.clone(), amp.clone(), idx.clone())
            else:
                assert torch.equal(ef, ref[0]) and torch.equal(amp, ref[1]) and torch.equal(idx, ref[2])
    finally:
        pat.free()


@pytest.mark.parametrize("cfg,n_st", [(3, 3), (4, 2)])
def test_team_and_cluster_kernels_inplace_and_peaks_only(B, orc, cfg, n_st):
    """The fp64 team kernel and the long-trace cluster kernel: E-field written over the input traces
    (efield aliases traces), peaks only (efield NULL), and fewer stations than warps / teams / CTAs."""
    wl = ai.WORKLOADS[cfg]
    H = table_for(wl)
    tr, dirs, _, _ = ai.make_batch(wl, [1], n_stations=n_st)
    ref = oracle_batch(orc, wl, H, tr, dirs)
    check(wl, run_gpu_batch(B, wl, H, tr, dirs, inplace=True), ref)
    ef, amp, idx = run_gpu_batch(B, wl, H, tr, dirs, want_efield=False)
    assert ef is None
    check(wl, (None, amp, idx), ref)


def test_scan_single_direction_and_station(B, orc):
    wl = ai.WORKLOADS[2]
    H = table_for(wl)
    ev = ai.make_event(wl, 0)
    for n_s, d_sel in ((1, [4242]), (2, [0, 7379]), (5, [17])):
        tr = np.ascontiguousarray(ev.traces[:n_s]); dirs = ai.scan_directions()[d_sel]
        pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
        try:
            amp, idx = B.aera_scan_directions(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
            torch.cuda.synchronize()
        finally:
            pat.free()
        oamp, oidx, oe2 = orc.scan(wl.grid, H, wl.fs_hz, tr, dirs, want_env2=True)
        rep = compare_peaks(wl.dtype, amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2)
        assert_peaks(rep, wl.dtype)


# ------------------------------------------------------------------ R8: exactly singular bins
def _table_with_dead_cell(wl, j0):
    """The seeded table with frequency nodes j0 and j0 + 1 set to zero: every DFT bin inside that frequency cell
    interpolates between zero matrices, so its response is exactly singular (det == 0) at every direction."""
    H = ai.pattern_table(wl.grid, wl.complex_dtype).copy()
    H[..., j0:j0 + 2] = 0
    return H


@pytest.mark.parametrize("cfg,events,n_st,variant,kernel", [
    (1, [0, 7], 9, 0, "unfold_w32"), (1, [0], 5, 1, "generic"), (0, [0, 1], 7, 0, "generic"),
    (3, [0], 5, 0, "unfold_t4k_f64"), (4, [0], 2, 0, "unfold_long_f32")])
def test_singular_bins_are_zeroed_like_the_oracle(B, orc, cfg, events, n_st, variant, kernel):
    """DESIGN.md reading R8: a bin whose 2x2 response has det == 0 contributes nothing (E[k] = 0). The oracle does this
    in oracle_solve2x2; here the CUDA branch runs on hardware against it, on every kernel family."""
    wl = ai.WORKLOADS[cfg]
    j0 = 6 if cfg != 4 else 50
    H = _table_with_dead_cell(wl, j0)
    f_lo = wl.grid.freq0_hz + j0 * wl.grid.dfreq_hz
    k_dead = [k for k in range(1, wl.n_samples // 2) if f_lo <= k * wl.fs_hz / wl.n_samples <= f_lo + wl.grid.dfreq_hz]
    assert len(k_dead) >= 2                                   # the cell really holds DFT bins of this (N, fs)
    tr, dirs, _, _ = ai.make_batch(wl, events, n_stations=n_st)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        ef, amp, idx = B.aera_unfold_batch(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    efn = ef.cpu().numpy()
    assert np.isfinite(efn).all() and np.isfinite(amp.cpu().numpy()).all()
    # the dead bins carry no power in the output: compare with the live neighbours (fp32 round-off floor ~1e-7 of the band)
    spec = np.abs(np.fft.rfft(efn.astype(np.float64), axis=-1))
    live = spec[..., k_dead[0] - 12:k_dead[0] - 2].mean()
    assert spec[..., k_dead].max() <= (1e-5 if wl.dtype == "f32" else 1e-12) * live, (spec[..., k_dead].max(), live)
    check(wl, (efn, amp.cpu().numpy(), idx.cpu().numpy()), oracle_batch(orc, wl, H, tr, dirs))


def test_singular_bins_in_the_scan(B, orc):
    wl = ai.WORKLOADS[2]
    H = _table_with_dead_cell(wl, 6)
    ev = ai.make_event(wl, 0)
    tr = np.ascontiguousarray(ev.traces[:9]); dirs = ai.scan_directions()[[0, 500, 3333, 7379]]
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "scan_w32"
    finally:
        pat.free()
    oamp, oidx, oe2 = orc.scan(wl.grid, H, wl.fs_hz, tr, dirs, want_env2=True)
    assert_peaks(compare_peaks(wl.dtype, amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2), wl.dtype)
