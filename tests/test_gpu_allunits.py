"""Full-coverage GPU parity (SURVEY.md 8c-B "secondary full-coverage check", A9): EVERY unit of the big batch
configs, in the launch configuration bench.py times (one call over the whole batch), against the harness-side
numpy float64 pipeline of fastref.py -- itself pinned to the oracle in tests/test_fastref_vs_oracle.py.
The oracle-sampled full-size tests stay in test_gpu_parity.py; this file adds the coverage the O(N K) oracle
cannot afford, and reports how many peak indices were exact / near-tie +-1 / ambiguous (non-adjacent near-tie).

Where the batch is larger than its block of distinct seeded events, the block is tiled on the device and the
copies are required to be bit-identical to their originals, so every unit is covered either way."""
import numpy as np
import pytest
import torch

import aera_inputs as ai
import fastref
from parity import TOL

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


def device_batch(wl, n_events, n_canon):
    """Canonical seeded events 0 .. n_canon-1 on the host, tiled to n_events on the device."""
    n_canon = min(n_canon, n_events)
    canon, dirs_c, _, _ = ai.make_batch_parallel(wl, range(n_canon))
    tdt = torch.float32 if wl.dtype == "f32" else torch.float64
    d_tr = torch.empty((n_events, wl.n_stations, 2, wl.n_samples), dtype=tdt, device="cuda")
    src = torch.from_numpy(canon)
    for lo in range(0, n_events, n_canon):
        hi = min(n_events, lo + n_canon)
        d_tr[lo:hi].copy_(src[: hi - lo])
    reps = -(-n_events // n_canon)
    dirs = np.ascontiguousarray(np.tile(dirs_c, (reps, 1))[:n_events])
    return canon, dirs_c, d_tr, torch.from_numpy(dirs).cuda()


@pytest.mark.parametrize("cfg,n_events,n_canon", [(1, 1000, 1000), (3, 10000, 2500), (4, 100, 100)])
def test_every_unit_against_float64_pipeline(B, cfg, n_events, n_canon):
    wl = ai.WORKLOADS[cfg]
    assert n_events == wl.n_events                       # BASELINE.json's stated size
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    tol = TOL[wl.dtype]
    canon, dirs_c, d_tr, d_dirs = device_batch(wl, n_events, n_canon)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32 if wl.dtype == "f32" else B.AERA_F64), H)
    try:
        l0 = B.aera_launch_count()
        ef, amp, idx = B.aera_unfold_batch(pat, d_tr, d_dirs, wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_launch_count() - l0 == 2           # one Minv launch + ONE unfold launch over the whole batch
        for lo in range(n_canon, n_events, n_canon):     # tiled copies: bit-identical to their originals
            hi = min(n_events, lo + n_canon)
            assert torch.equal(ef[lo:hi], ef[: hi - lo]) and torch.equal(amp[lo:hi], amp[: hi - lo]) and torch.equal(idx[lo:hi], idx[: hi - lo])
        r = fastref.check_all_units(wl.grid, H, wl.fs_hz, canon, dirs_c, ef[:n_canon].cpu().numpy(), amp[:n_canon].cpu().numpy(),
                                    idx[:n_canon].cpu().numpy(), tol)
    finally:
        pat.free()
    print(f"\n[all units cfg{cfg}: {n_events} events x {wl.n_stations} stations = {n_events * wl.n_stations} units, {r['n']} distinct] "
          f"relL2 max={r['max_l2']:.3e} amp max={r['max_amp']:.3e} idx exact={r['exact']} tie+-1={r['tie_pm1']} "
          f"ambiguous={r['ambiguous']} miss={r['miss']} bad={r['bad'][:6]}")
    assert r["max_l2"] <= tol["l2"] and r["max_amp"] <= tol["amp"], r
    assert r["miss"] == 0, r["bad"][:10]
    # SURVEY A9 predicts ~1 near-tie per 1e5 fp32 units, about half of them non-adjacent ("ambiguous": both samples are
    # maxima to working precision). Strict reading (R9): none tolerated on these seeded inputs.
    assert r["ambiguous"] == 0, r["bad"][:10]


def test_every_pair_of_the_full_scan_against_float64_pipeline(B):
    """BASELINE configs[2] at its stated size, in the one call bench.py --config 2 times: all 7 380 directions x 124
    stations = 915 120 (direction, station) pairs against the float64 pipeline (each direction is one "event" over the
    same 124 traces), with the same exact / near-tie / ambiguous count as the batch configs."""
    wl = ai.WORKLOADS[2]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    ev = ai.make_event(wl, 0)
    dirs = ai.scan_directions()
    D, S = len(dirs), ev.traces.shape[0]
    assert (D, S) == (41 * 180, 124)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        l0 = B.aera_launch_count()
        amp, idx = B.aera_scan_directions(pat, torch.from_numpy(ev.traces).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "scan_w32" and B.aera_launch_count() - l0 == 3   # Minv + forward + ONE inverse launch
    finally:
        pat.free()
    tol = TOL["f32"]
    traces = np.broadcast_to(ev.traces, (D,) + ev.traces.shape)                         # a view: no 7 380 copies
    r = fastref.check_all_units(wl.grid, H, wl.fs_hz, traces, dirs, None, amp.cpu().numpy(), idx.cpu().numpy(), tol)
    print(f"\n[all pairs cfg2: {D} directions x {S} stations = {r['n']} pairs] amp max={r['max_amp']:.3e} idx exact={r['exact']} "
          f"tie+-1={r['tie_pm1']} ambiguous={r['ambiguous']} miss={r['miss']} bad={r['bad'][:6]}")
    assert r["n"] == D * S
    assert r["max_amp"] <= tol["amp"], r["max_amp"]
    assert r["miss"] == 0, r["bad"][:10]
    # Directions far from the true one smear the pulse, so a few near-ties among 915 120 pairs are expected (SURVEY A9:
    # ~1 per 1e5 fp32 units); adjacent ones are allowed by the north_star rule, non-adjacent ones are counted and bounded
    assert r["tie_pm1"] + r["ambiguous"] <= 40, (r["tie_pm1"], r["ambiguous"], r["bad"][:10])
