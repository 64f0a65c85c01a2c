"""GPU parity of the on-device forward model (aera_fold_batch) against the oracle's
fold (oracle.dft_band + oracle.fold_station: the plain definition V = H E on the band, inverse real DFT),
and the round trip unfold(fold(e)) = band-limited e on the device."""
import numpy as np
import pytest
import torch

import aera_inputs as ai
from parity import TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


@pytest.mark.parametrize("cfg,n_events,n_st,variant", [(0, 2, 7, 0), (1, 2, 9, 0), (1, 1, 5, 1), (3, 2, 5, 0), (4, 1, 2, 0)])
def test_fold_matches_oracle_and_round_trips(B, cfg, n_events, n_st, variant):
    import oracle
    wl = ai.WORKLOADS[cfg]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    rng = np.random.default_rng([77, cfg])
    N = wl.n_samples
    ef = rng.standard_normal((n_events, n_st, 2, N)).astype(wl.real_dtype)          # white E-field: every band bin is exercised
    dirs = np.stack([rng.uniform(0, wl.zenith_max_deg, n_events), rng.uniform(0, 360, n_events)], axis=1)
    dt = B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, dt), H)
    old = B.aera_set_kernel_variant(variant)
    try:
        d_ef = torch.from_numpy(ef).cuda(); d_dirs = torch.from_numpy(dirs).cuda()
        v = B.aera_fold_batch(pat, d_ef, d_dirs, wl.fs_hz)
        ef2, amp, idx = B.aera_unfold_batch(pat, v, d_dirs, wl.fs_hz)
        torch.cuda.synchronize()
        v_h = v.cpu().numpy(); ef2_h = ef2.cpu().numpy()
    finally:
        B.aera_set_kernel_variant(old)
        pat.free()
    k_lo, k_hi = oracle.band(N, wl.fs_hz, wl.grid.n_freq, wl.grid.freq0_hz, wl.grid.dfreq_hz)
    tol = TOL[wl.dtype]["l2"]
    worst = 0.0
    for e in range(n_events):
        for s in range(n_st):
            Et = oracle.dft_band(ef[e, s, 0], k_lo, k_hi); Ep = oracle.dft_band(ef[e, s, 1], k_lo, k_hi)
            ref = oracle.fold_station(wl.grid, H, N, wl.fs_hz, Et, Ep, dirs[e, 0], dirs[e, 1])
            worst = max(worst, np.linalg.norm(v_h[e, s] - ref) / np.linalg.norm(ref))
            # round trip: the band-limited part of e comes back (Re of the analytic signal of the band spectrum)
            zt = oracle.analytic_from_band(Et, N, k_lo, k_hi); zp = oracle.analytic_from_band(Ep, N, k_lo, k_hi)
            back = np.stack([np.real(zt), np.real(zp)])
            rt = np.linalg.norm(ef2_h[e, s] - back) / np.linalg.norm(back)
            assert rt <= 20 * tol, (e, s, rt)      # two passes through H and H^-1 (cond <= 6.4)
    print(f"\n[fold cfg{cfg}] max rel L2 vs oracle = {worst:.3e}")
    assert worst <= tol, worst
