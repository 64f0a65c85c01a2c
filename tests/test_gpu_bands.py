"""The specialised kernels on band geometries other than the three benchmark ones (a user at another sampling rate
must not fall silently to the generic radix-2 path): which kernel family ran is read back with aera_last_kernel()."""
import numpy as np
import pytest
import torch

import aera_inputs as ai
from parity import TOL, assert_peaks, compare, compare_peaks

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


@pytest.mark.parametrize("dtype,N,fs,kernel", [("f32", 2048, 200e6, "unfold_w32"), ("f32", 2048, 250e6, "unfold_w32"),
                                               ("f64", 4096, 250e6, "unfold_t4k_f64"), ("f64", 4096, 180e6, "unfold_t4k_f64"),
                                               ("f32", 4096, 200e6, "unfold_t4k_f32"), ("f32", 4096, 250e6, "unfold_t4k_f32"),
                                               ("f32", 1024, 200e6, "unfold_t1k_f32"), ("f32", 1024, 180e6, "unfold_t1k_f32"),
                                               ("f64", 2048, 200e6, "unfold_t2k_f64"), ("f64", 2048, 250e6, "unfold_t2k_f64"),
                                               ("f64", 1024, 200e6, "unfold_t1k_f64"), ("f64", 1024, 180e6, "unfold_t1k_f64"),
                                               ("f32", 8192, 200e6, "unfold_t8k_f32"), ("f32", 8192, 250e6, "unfold_t8k_f32"),
                                               ("f64", 8192, 200e6, "unfold_t8k_f64"), ("f64", 8192, 180e6, "unfold_t8k_f64"),
                                               ("f32", 16384, 200e6, "unfold_t16k_f32"), ("f32", 16384, 180e6, "unfold_t16k_f32"),
                                               ("f32", 512, 200e6, "generic"), ("f64", 16384, 200e6, "generic")])
def test_batch_other_bands(B, dtype, N, fs, kernel):
    import oracle
    base = ai.WORKLOADS[0]
    wl = ai.Workload(91, "bands", 3, 7, N, fs, dtype, base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(3))
    dt = B.AERA_F32 if dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        ef, amp, idx = B.aera_unfold_batch(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), fs)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel
    finally:
        pat.free()
    E, S = tr.shape[:2]
    ref = oracle.unfold_batch(wl.grid, H, fs, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0), want_env2=True)
    rep = compare(dtype, ef.cpu().numpy().reshape(E * S, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref)
    print(f"\n[bands {dtype} N={N} fs={fs / 1e6:.0f} MHz -> {kernel}] {rep}")
    assert rep.ok(TOL[dtype]), str(rep)


@pytest.mark.parametrize("fs", [1e9, 500e6])
def test_long_trace_other_band(B, fs):
    """N = 65536 with the 30-80 MHz table (configs[4]'s is 20-200 MHz): the cluster kernel's any-band instantiation."""
    import oracle
    base = ai.WORKLOADS[0]
    N = 65536
    wl = ai.Workload(94, "long-band", 1, 3, N, fs, "f32", base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(1))
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        ef, amp, idx = B.aera_unfold_batch(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), fs)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "unfold_long_f32"
    finally:
        pat.free()
    E, S = tr.shape[:2]
    ref = oracle.unfold_batch(wl.grid, H, fs, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0), want_env2=True)
    rep = compare("f32", ef.cpu().numpy().reshape(E * S, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref)
    print(f"\n[long trace, 30-80 MHz table, fs={fs / 1e6:.0f} MHz] {rep}")
    assert rep.ok(TOL["f32"]), str(rep)


def test_scan_other_band_runs_the_warp_kernels(B):
    import oracle
    base = ai.WORKLOADS[2]
    fs = 200e6                                     # band rows 9..25 instead of configs[2]'s 10..28
    wl = ai.Workload(92, "scan-band", 1, 9, 2048, fs, "f32", base.grid, 75.0, 512, 1536, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    ev = ai.make_event(wl, 0)
    dirs = ai.scan_directions()[[0, 91, 1234, 4000, 7379]]
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(ev.traces).cuda(), torch.from_numpy(dirs).cuda(), fs)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "scan_w32"
    finally:
        pat.free()
    oamp, oidx, oe2 = oracle.scan(wl.grid, H, fs, ev.traces, dirs, want_env2=True)
    rep = compare_peaks("f32", amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2)
    print(f"\n[scan fs=200 MHz] {rep}")
    assert_peaks(rep, "f32")


def test_spectrum_reuse_on_another_band_is_bit_identical(B):
    wl0 = ai.WORKLOADS[1]
    fs = 200e6
    wl = ai.Workload(93, "loop-band", 3, 21, 2048, fs, "f32", wl0.grid, 75.0, 512, 1536, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    pos = ai.station_positions(21)
    tr = np.stack([ai.make_event(wl, e, n_stations=21, positions=pos).traces for e in range(3)])
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        d_tr = torch.from_numpy(tr).cuda(); d_pos = torch.from_numpy(pos).cuda()
        small = B.alloc_workspace(B.aera_workspace_bytes(B.AERA_OP_UNFOLD, pat, B.AERA_F32, 3, 21, 2048, fs))
        big = B.alloc_workspace(B.aera_workspace_bytes(B.AERA_OP_RECONSTRUCT, pat, B.AERA_F32, 3, 21, 2048, fs))
        assert big.numel() > small.numel()
        a = B.aera_reconstruct_batch(pat, d_tr, d_pos, fs, 3, workspace=small)
        b = B.aera_reconstruct_batch(pat, d_tr, d_pos, fs, 3, workspace=big)
        torch.cuda.synchronize()
        for k in ("dirs_hist", "efield", "amp_hist", "idx_hist", "idx0", "w0"):
            assert torch.equal(a[k], b[k]), k
    finally:
        pat.free()


@pytest.mark.parametrize("dtype,N,kernel", [("f64", 1024, "unfold_t1k_f64"), ("f64", 2048, "unfold_t2k_f64"), ("f32", 1024, "unfold_t1k_f32"),
                                            ("f32", 8192, "unfold_t8k_f32"), ("f64", 8192, "unfold_t8k_f64"), ("f32", 16384, "unfold_t16k_f32")])
def test_team_sizes_fold_inplace_peaks_only_and_tables(B, dtype, N, kernel):
    """Teams of one and two warps (N = 1024 / 2048) through every entry point that shares the team kernel: the forward
    model against the oracle's fold, E-field written over the traces, peaks only, and two identical tables reproducing
    the single-table call bit for bit; 3 x 7 = 21 stations do not fill the CTA's teams evenly."""
    import oracle
    base = ai.WORKLOADS[0]
    fs = 200e6
    wl = ai.Workload(95, "team-sizes", 3, 7, N, fs, dtype, base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(3))
    dt = B.AERA_F32 if dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    pat2 = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        d_tr = torch.from_numpy(tr).cuda(); d_dirs = torch.from_numpy(dirs).cuda()
        ef, amp, idx = B.aera_unfold_batch(pat, d_tr, d_dirs, fs)
        assert B.aera_last_kernel() == kernel
        # peaks only
        _, amp1, idx1 = B.aera_unfold_batch(pat, d_tr, d_dirs, fs, want_efield=False)
        assert torch.equal(amp, amp1) and torch.equal(idx, idx1)
        # two identical tables, stations alternating between them
        pid = torch.tensor([s & 1 for s in range(7)], dtype=torch.int32, device="cuda")
        ef2, amp2, idx2 = B.aera_unfold_batch_multi([pat, pat2], pid, d_tr, d_dirs, fs)
        assert B.aera_last_kernel() == kernel
        assert torch.equal(ef, ef2) and torch.equal(amp, amp2) and torch.equal(idx, idx2)
        # in place
        d_io = d_tr.clone()
        ef3, amp3, idx3 = B.aera_unfold_batch(pat, d_io, d_dirs, fs, efield=d_io)
        assert torch.equal(ef, ef3) and torch.equal(amp, amp3) and torch.equal(idx, idx3)
        # forward model on the same kernels
        rng = np.random.default_rng([78, N])
        e_in = rng.standard_normal((2, 5, 2, N)).astype(wl.real_dtype)
        v = B.aera_fold_batch(pat, torch.from_numpy(e_in).cuda(), d_dirs[:2].contiguous(), fs)
        assert B.aera_last_kernel() == kernel
        torch.cuda.synchronize()
        v_h = v.cpu().numpy()
    finally:
        pat.free(); pat2.free()
    k_lo, k_hi = oracle.band(N, fs, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    worst = 0.0
    for e in range(2):
        for s in range(5):
            Et = oracle.dft_band(e_in[e, s, 0], k_lo, k_hi); Ep = oracle.dft_band(e_in[e, s, 1], k_lo, k_hi)
            ref = oracle.fold_station(wl.grid, H, N, fs, Et, Ep, dirs[e, 0], dirs[e, 1])
            worst = max(worst, np.linalg.norm(v_h[e, s] - ref) / np.linalg.norm(ref))
    print(f"\n[team sizes {dtype} N={N}] fold max rel L2 vs oracle = {worst:.3e}")
    assert worst <= TOL[dtype]["l2"], worst
