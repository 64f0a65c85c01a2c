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
@pytest.mark.parametrize("cfg,events,n_st,u", [(0, [0, 1], 7, 2), (0, [2], 7, 4), (1, [0], 6, 2), (3, [1], 3, 2), (0, [0], 3, 1)])
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
