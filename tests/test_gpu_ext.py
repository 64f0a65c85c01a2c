"""GPU parity of the remaining "next" rows against oracle/aera_ext.py:
per-station pattern tables (aera_unfold_batch_multi), int16 ADC-count input (aera_unfold_batch_i16) and spectral
up-sampling (aera_unfold_batch_upsampled); every kernel family they can run on."""
import numpy as np
import pytest
import torch

import aera_inputs as ai
from parity import TOL, compare

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


def _check(wl, rep, what):
    print(f"\n[{what}] {rep}")
    assert rep.ok(TOL[wl.dtype]), f"{what}: {rep}"


# ------------------------------------------------------------------ row 2: three antenna types
@pytest.mark.parametrize("cfg,events,n_st,variant,kernel", [
    (1, [0, 5, 999], 124, 0, "unfold_w32"), (1, [0, 1], 9, 1, "generic"), (0, [0, 1], 7, 0, "generic"),
    (3, [0, 42], 7, 0, "unfold_t4k_f64"), (4, [0], 3, 0, "unfold_long_f32")])
def test_multi_pattern_matches_oracle(B, cfg, events, n_st, variant, kernel):
    from oracle import aera_ext as ox
    wl = ai.WORKLOADS[cfg]
    tables = [ai.pattern_table(wl.grid, wl.complex_dtype, seed=sd) for sd in (1507, 99, 4242)]   # three antenna types
    rng = np.random.default_rng([5, cfg])
    pid = rng.integers(0, 3, size=n_st).astype(np.int32); pid[:3] = [0, 1, 2]
    tr, dirs, _, _ = ai.make_batch(wl, events, n_stations=n_st)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pats = [B.aera_pattern_upload(B.make_desc(wl.grid, dt), H) for H in tables]
    old = B.aera_set_kernel_variant(variant)
    try:
        ef, amp, idx = B.aera_unfold_batch_multi(pats, torch.from_numpy(pid).cuda(), torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel
        # identical tables -> the single-table call, bit for bit (same kernels, same matrices)
        ef1, amp1, idx1 = B.aera_unfold_batch_multi([pats[0], pats[0]], torch.from_numpy((pid % 2).astype(np.int32)).cuda(), torch.from_numpy(tr).cuda(),
                                                   torch.from_numpy(dirs).cuda(), wl.fs_hz)
        ef0, amp0, idx0 = B.aera_unfold_batch(pats[0], torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef1, ef0) and torch.equal(amp1, amp0) and torch.equal(idx1, idx0)
    finally:
        B.aera_set_kernel_variant(old)
        for p in pats:
            p.free()
    ref = ox.unfold_batch_multi(wl.grid, tables, pid, wl.fs_hz, tr, dirs, want_env2=True)
    U = len(ref["amp"])
    _check(wl, compare(wl.dtype, ef.cpu().numpy().reshape(U, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref), f"multi cfg{cfg} {kernel}")


# ------------------------------------------------------------------ row 4: int16 ADC counts
@pytest.mark.parametrize("cfg,events,n_st,variant,kernel", [(1, [0, 3, 17], 124, 0, "unfold_w32"), (1, [1], 5, 1, "generic"), (0, [0, 1], 7, 0, "generic")])
def test_int16_input_matches_oracle(B, cfg, events, n_st, variant, kernel):
    from oracle import aera_ext as ox
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, events, n_stations=n_st)
    g = (0.0625, 0.05)                                                   # microvolt per ADC count, per channel
    counts = np.stack([np.clip(np.round(tr[:, :, c] / g[c]), -32768, 32767) for c in (0, 1)], axis=2).astype(np.int16)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        ef, amp, idx = B.aera_unfold_batch_i16(pat, torch.from_numpy(counts).cuda(), g, torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel and ef.dtype == torch.float32
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    E, S = counts.shape[:2]
    ref = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, counts.reshape(E * S, 2, -1), g, np.repeat(dirs, S, axis=0), want_env2=True)
    _check(wl, compare("f32", ef.cpu().numpy().reshape(E * S, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref), f"int16 cfg{cfg} {kernel}")


# ------------------------------------------------------------------ row 4: spectral up-sampling
@pytest.mark.parametrize("cfg,events,n_st,u", [(0, [0, 1], 7, 2), (0, [2], 7, 4), (1, [0], 6, 2), (3, [1], 3, 2), (0, [0], 3, 1),
                                               (1, [0, 1], 124, 2)])   # N = 2048 x all 124 stations of an event
def test_upsampled_matches_oracle(B, cfg, events, n_st, u):
    from oracle import aera_ext as ox
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, events, n_stations=n_st)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        ef, amp, idx = B.aera_unfold_batch_upsampled(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz, u)
        torch.cuda.synchronize()
        assert tuple(ef.shape) == (len(events), n_st, 2, u * wl.n_samples)
        with pytest.raises(B.AeraError) as e:
            B.aera_unfold_batch_upsampled(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz, 3)
        assert e.value.status == 1
    finally:
        pat.free()
    E, S = tr.shape[:2]
    ref = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0), u)
    _check(wl, compare(wl.dtype, ef.cpu().numpy().reshape(E * S, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref), f"upsampled x{u} cfg{cfg}")


@pytest.mark.parametrize("N,fs,kernel", [(4096, 200e6, "unfold_t4k_f32"), (4096, 250e6, "unfold_t4k_f32"), (1024, 200e6, "unfold_t1k_f32"), (8192, 200e6, "unfold_t8k_f32")])
def test_int16_input_on_the_team_kernels(B, N, fs, kernel):
    """int16 ADC counts at the other register-resident trace lengths (fp32 out): the team kernel's templated load."""
    from oracle import aera_ext as ox
    base = ai.WORKLOADS[0]
    wl = ai.Workload(96, "i16-team", 2, 9, N, fs, "f32", base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(2))
    g = (0.0625, 0.05)
    counts = np.stack([np.clip(np.round(tr[:, :, c] / g[c]), -32768, 32767) for c in (0, 1)], axis=2).astype(np.int16)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        ef, amp, idx = B.aera_unfold_batch_i16(pat, torch.from_numpy(counts).cuda(), g, torch.from_numpy(dirs).cuda(), fs)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel and ef.dtype == torch.float32
    finally:
        pat.free()
    E, S = counts.shape[:2]
    ref = ox.unfold_batch_i16(wl.grid, H, fs, counts.reshape(E * S, 2, -1), g, np.repeat(dirs, S, axis=0), want_env2=True)
    _check(wl, compare("f32", ef.cpu().numpy().reshape(E * S, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref), f"int16 N={N} {kernel}")


def test_upsampled_short_trace_many_units_global_scratch(B):
    """Up-sampling a short trace far enough that N + 2 N U leaves shared memory (fp32 N = 512, U = 32) on more units than
    the kernel has scratch slices (4 per SM): the launch must stay on the grid the scratch was sized for. Checked three
    ways: bytes around an exactly sized workspace stay untouched, every event equals its own single-event call (few
    enough units that every CTA has a slice under any grid rule), and sampled units match the oracle."""
    from oracle import aera_ext as ox
    N, U, E, S = 512, 32, 8, 128
    base = ai.WORKLOADS[0]
    wl = ai.Workload(91, "upsampled-many", E, S, N, 200e6, "f32", base.grid, 60.0, N // 4, 3 * N // 4, 5.0)
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, range(E))
    trd, dd = torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda()
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        wsb = B.aera_workspace_bytes_ex(B.AERA_OP_UNFOLD, pat, B.AERA_F32, E, S, N, wl.fs_hz, 1, U)
        guard = 1 << 20
        raw = torch.full((wsb + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
        ef, amp, idx = B.aera_unfold_batch_upsampled(pat, trd, dd, wl.fs_hz, U, workspace=raw[guard:guard + wsb])
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "generic"
        assert bool((raw[:guard] == 0xA5).all()) and bool((raw[guard + wsb:] == 0xA5).all()), "write outside the workspace"
        for e in range(E):
            ef1, amp1, idx1 = B.aera_unfold_batch_upsampled(pat, trd[e:e + 1], dd[e:e + 1], wl.fs_hz, U)
            assert torch.equal(ef1[0], ef[e]) and torch.equal(amp1[0], amp[e]) and torch.equal(idx1[0], idx[e]), e
    finally:
        pat.free()
    units = np.array([0, 1, 127, 128, 500, 591, 592, 593, 700, 901, 1022, 1023])      # on both sides of 4 x 148 slices
    ref = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr.reshape(E * S, 2, -1)[units], np.repeat(dirs, S, axis=0)[units], U)
    _check(wl, compare("f32", ef.cpu().numpy().reshape(E * S, 2, -1)[units], amp.cpu().numpy().ravel()[units],
                       idx.cpu().numpy().ravel()[units], ref), "upsampled x32 N=512, 1024 units")


@pytest.mark.parametrize("cfg,n_st,u", [(0, 7, 4), (1, 5, 2), (3, 3, 2)])
def test_band_filter_applies_to_upsampling(B, cfg, n_st, u):
    """aera_pattern_set_band_filter + aera_unfold_batch_upsampled: the weights belong to (n_samples, fs), not to one plan,
    so they reach the up-sampled call whether its plan was built before or after the filter was set, and removing the
    filter restores the unfiltered fine-grid result bit for bit. Against oracle/aera_ext.py with the same weights."""
    from oracle import aera_ext as ox
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, [0, 1], n_stations=n_st)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    d_tr, d_dirs = torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda()
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    try:
        k_lo, k_hi = B.aera_band(pat, wl.n_samples, wl.fs_hz)
        rng = np.random.default_rng([7, cfg])
        w = 0.2 + 0.8 * rng.uniform(size=k_hi - k_lo + 1); w[rng.choice(len(w), 4, replace=False)] = 0.0
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, w)                       # filter first, then the U-plan
        ef_a, amp_a, idx_a = B.aera_unfold_batch_upsampled(pat, d_tr, d_dirs, wl.fs_hz, u)
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, None)
        ef_0, amp_0, idx_0 = B.aera_unfold_batch_upsampled(pat, d_tr, d_dirs, wl.fs_hz, u)   # unfiltered, U-plan exists now
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, w)                       # filter after the U-plan
        ef_b, amp_b, idx_b = B.aera_unfold_batch_upsampled(pat, d_tr, d_dirs, wl.fs_hz, u)
        torch.cuda.synchronize()
    finally:
        pat.free()
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)                                  # a handle that never saw a filter
    try:
        ef_p, amp_p, idx_p = B.aera_unfold_batch_upsampled(pat, d_tr, d_dirs, wl.fs_hz, u)
        torch.cuda.synchronize()
    finally:
        pat.free()
    assert torch.equal(ef_a, ef_b) and torch.equal(amp_a, amp_b) and torch.equal(idx_a, idx_b)
    assert torch.equal(ef_0, ef_p) and torch.equal(amp_0, amp_p) and torch.equal(idx_0, idx_p)
    assert not torch.equal(ef_a, ef_0)
    E, S = tr.shape[:2]
    ref = ox.unfold_batch_upsampled(wl.grid, H, wl.fs_hz, tr.reshape(E * S, 2, -1), np.repeat(dirs, S, axis=0), u, w)
    _check(wl, compare(wl.dtype, ef_a.cpu().numpy().reshape(E * S, 2, -1), amp_a.cpu().numpy().ravel(), idx_a.cpu().numpy().ravel(), ref),
           f"filtered + upsampled x{u} cfg{cfg}")


@pytest.mark.parametrize("cfg,n_st,kernel", [(1, 37, "unfold_w32"), (0, 7, "generic"), (3, 5, "unfold_t4k_f64"), (4, 2, "unfold_long_f32")])
def test_multi_pattern_ids_out_of_range_are_clamped(B, cfg, n_st, kernel):
    """pattern_id values outside 0 .. n_patterns-1 cannot be reported by an asynchronous call; they must not index outside
    the workspace either: they are clamped, so the result equals the call with the clamped ids bit for bit (and the bytes
    around an exactly sized workspace stay untouched)."""
    wl = ai.WORKLOADS[cfg]
    tables = [ai.pattern_table(wl.grid, wl.complex_dtype, seed=sd) for sd in (1507, 99, 4242)]
    tr, dirs, _, _ = ai.make_batch(wl, [0, 1] if cfg != 4 else [0], n_stations=n_st)
    E = tr.shape[0]
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    bad = (np.arange(n_st) % 3).astype(np.int32); bad[0] = -7; bad[-1] = 1 << 20
    if n_st > 3:
        bad[2] = 3; bad[3] = -(1 << 30)
    good = np.clip(bad, 0, 2).astype(np.int32)
    pats = [B.aera_pattern_upload(B.make_desc(wl.grid, dt), H) for H in tables]
    try:
        d_tr, d_dirs = torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda()
        wsb = B.aera_workspace_bytes_ex(B.AERA_OP_UNFOLD, pats[0], dt, E, n_st, wl.n_samples, wl.fs_hz, 3, 1)
        guard = 1 << 20
        raw = torch.full((wsb + 2 * guard,), 0xA5, dtype=torch.uint8, device="cuda")
        ef_b, amp_b, idx_b = B.aera_unfold_batch_multi(pats, torch.from_numpy(bad).cuda(), d_tr, d_dirs, wl.fs_hz, workspace=raw[guard:guard + wsb])
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel
        assert bool((raw[:guard] == 0xA5).all()) and bool((raw[guard + wsb:] == 0xA5).all())
        ef_g, amp_g, idx_g = B.aera_unfold_batch_multi(pats, torch.from_numpy(good).cuda(), d_tr, d_dirs, wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef_b, ef_g) and torch.equal(amp_b, amp_g) and torch.equal(idx_b, idx_g)
        assert torch.isfinite(ef_b).all()
    finally:
        for p in pats:
            p.free()


def test_host_pipeline_int16_matches_device_path_and_oracle(B):
    """aera_unfold_batch_host_i16: int16 counts from host memory through the chunked 3-stream pipeline. Bit-equal to the
    device call aera_unfold_batch_i16 (the same kernels on the same chunks' data), against the int16 oracle on a sample,
    peaks-only mode (no E-field staged or copied), and the staging buffers shared with the fp32 host call grow as needed."""
    from oracle import aera_ext as ox
    wl = ai.WORKLOADS[1]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    E, S = 70, 124                                        # 70 events x 124 stations x 16 KB of E-field = 139 MB: three 64 MB chunks
    tr, dirs, _, _ = ai.make_batch_parallel(wl, range(10))
    tr = np.ascontiguousarray(np.tile(tr, (7, 1, 1, 1))); dirs = np.ascontiguousarray(np.tile(dirs, (7, 1)))
    g = (0.0625, 0.05)
    counts = np.stack([np.clip(np.round(tr[:, :, c] / g[c]), -32768, 32767) for c in (0, 1)], axis=2).astype(np.int16)
    c_h = torch.from_numpy(counts).pin_memory(); d_h = torch.from_numpy(dirs).pin_memory()
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        _, amp_p, idx_p = B.aera_unfold_batch_host_i16(pat, c_h, g, d_h, wl.fs_hz, want_efield=False)     # peaks only first: no d_out yet
        ef_h, amp_h, idx_h = B.aera_unfold_batch_host_i16(pat, c_h, g, d_h, wl.fs_hz)                    # staging grows for the E-field
        ef_d, amp_d, idx_d = B.aera_unfold_batch_i16(pat, c_h.cuda(), g, d_h.cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef_h, ef_d.cpu()) and torch.equal(amp_h, amp_d.cpu()) and torch.equal(idx_h, idx_d.cpu())
        assert torch.equal(amp_p, amp_h) and torch.equal(idx_p, idx_h)
        t_h = torch.from_numpy(tr[:3]).pin_memory()                                                      # the fp32 host call on the same handle
        ef_f, amp_f, idx_f = B.aera_unfold_batch_host(pat, t_h, d_h[:3].clone().pin_memory(), wl.fs_hz)
        ef_g, amp_g, idx_g = B.aera_unfold_batch(pat, t_h.cuda(), d_h[:3].cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef_f, ef_g.cpu()) and torch.equal(idx_f, idx_g.cpu())
        with pytest.raises(B.AeraError):
            B.aera_unfold_batch_host_i16(pat, c_h, (float("nan"), 1.0), d_h, wl.fs_hz)
    finally:
        pat.free()
    ev, st = np.array([0, 9, 33, 69]), np.array([0, 57, 123])
    sel = counts[ev][:, st].reshape(-1, 2, wl.n_samples)
    ref = ox.unfold_batch_i16(wl.grid, H, wl.fs_hz, sel, g, np.repeat(dirs[ev], len(st), axis=0), want_env2=True)
    _check(wl, compare("f32", ef_h.numpy()[ev][:, st].reshape(-1, 2, wl.n_samples), amp_h.numpy()[ev][:, st].ravel(),
                       idx_h.numpy()[ev][:, st].ravel(), ref), "host int16 pipeline")
