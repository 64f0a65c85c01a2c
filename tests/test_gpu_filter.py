"""GPU parity of the fused pre-filter (aera_pattern_set_band_filter) against
oracle/aera_filter.py, for the batch unfold (specialised and generic kernels, fp32 and fp64) and the scan;
removing the filter restores the unfiltered results bit for bit."""
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


def _weights(K, seed):
    rng = np.random.default_rng(seed)
    w = 0.2 + 0.8 * rng.uniform(size=K)
    w[: K // 10] *= np.linspace(0.0, 1.0, K // 10)           # band-pass taper at the lower edge
    w[rng.choice(K, size=5, replace=False)] = 0.0            # notches
    return w


@pytest.mark.parametrize("cfg,n_st,variant", [(1, 9, 0), (1, 4, 1), (0, 7, 0), (3, 5, 0)])
def test_filtered_unfold_matches_oracle(B, cfg, n_st, variant):
    from oracle import aera_filter as of
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tr, dirs, _, _ = ai.make_batch(wl, [0, 1], n_stations=n_st)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        k_lo, k_hi = B.aera_band(pat, wl.n_samples, wl.fs_hz)
        w = _weights(k_hi - k_lo + 1, cfg)
        d_tr = torch.from_numpy(tr).cuda(); d_dirs = torch.from_numpy(dirs).cuda()
        ef0, amp0, idx0 = B.aera_unfold_batch(pat, d_tr, d_dirs, wl.fs_hz)
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, w)
        ef, amp, idx = B.aera_unfold_batch(pat, d_tr, d_dirs, wl.fs_hz)
        with pytest.raises(B.AeraError):
            B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, w[:-1])
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, None)
        ef1, amp1, idx1 = B.aera_unfold_batch(pat, d_tr, d_dirs, wl.fs_hz)
        torch.cuda.synchronize()
        assert torch.equal(ef0, ef1) and torch.equal(idx0, idx1) and torch.equal(amp0, amp1)
        assert not torch.equal(ef0, ef)
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    U = tr.shape[0] * n_st
    ref = of.unfold_batch_filtered(wl.grid, H, wl.fs_hz, tr.reshape(U, 2, -1), np.repeat(dirs, n_st, axis=0), w)
    rep = compare(wl.dtype, ef.cpu().numpy().reshape(U, 2, -1), amp.cpu().numpy().ravel(), idx.cpu().numpy().ravel(), ref)
    print(f"\n[filter cfg{cfg} variant {variant}] {rep}")
    assert rep.ok(TOL[wl.dtype]), str(rep)


def test_filtered_scan_matches_oracle(B):
    from oracle import aera_filter as of
    wl = ai.WORKLOADS[2]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    ev = ai.make_event(wl, 0)
    tr = np.ascontiguousarray(ev.traces[:6]); dirs = ai.scan_directions()[[5, 900, 4000, 7001]]
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        k_lo, k_hi = B.aera_band(pat, wl.n_samples, wl.fs_hz)
        w = _weights(k_hi - k_lo + 1, 2)
        B.aera_pattern_set_band_filter(pat, wl.n_samples, wl.fs_hz, w)
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
    finally:
        pat.free()
    oamp = np.empty((len(dirs), len(tr))); oidx = np.empty((len(dirs), len(tr)), dtype=np.int32)
    oe2 = np.empty((len(dirs), len(tr), wl.n_samples))
    for d in range(len(dirs)):
        r = of.unfold_batch_filtered(wl.grid, H, wl.fs_hz, tr, np.tile(dirs[d], (len(tr), 1)), w)
        oamp[d] = r["amp"]; oidx[d] = r["idx"]; oe2[d] = r["env2"]
    rep = compare_peaks(wl.dtype, amp.cpu().numpy(), idx.cpu().numpy(), oamp, oidx, oe2)
    assert_peaks(rep, wl.dtype)
