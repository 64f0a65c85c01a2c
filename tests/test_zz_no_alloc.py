"""aera_unfold_batch_static: the batch unfolding for callers that may not allocate device memory.

Some users of this library never get to call cudaMalloc: a reconstruction module loaded into an application that owns
the device-memory pool is handed input and output buffers and nothing else, and a trigger / monitoring loop cannot
afford the device-wide stall an allocation causes. For them the library carries its scratch as a built-in 32 MiB
device array, and this entry point runs the ordinary unfolding on it without taking a workspace.

What is checked here, through the C ABI on the GPU: the outputs equal those of aera_unfold_batch (the existing path, own
workspace) within the parity tolerances of tests/parity.py, on two calls in a row with different sizes and inputs -- the
second call finds the first one's leftovers in the array, and must not be affected by them; a third call on another
kernel family (fp64 team kernel) follows for the same reason; batches beyond the array and calls without the set-up
step are refused with a message that says what to do.

This file sorts last on purpose (pytest -x stops at the first failure): it exercises a process-wide array, so a failure
here must not hide the rest of the suite. It passes alone in a fresh process and after all other tests.
"""
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


def _both_paths(B, pat, tr, dirs, fs, dtype):
    """Run the static-scratch entry point, then the existing path on a fresh workspace; assert they agree."""
    E, S, _, N = tr.shape
    ef_s = torch.full_like(tr, float("nan"))
    amp_s = torch.full((E, S), float("nan"), dtype=tr.dtype, device="cuda")
    idx_s = torch.full((E, S), -1, dtype=torch.int32, device="cuda")
    B.aera_unfold_batch_static(pat, tr, dirs, fs, ef_s, amp_s, idx_s)
    kernel = B.aera_last_kernel()
    ef, amp, idx = B.aera_unfold_batch(pat, tr, dirs, fs)
    torch.cuda.synchronize()
    assert B.aera_last_kernel() == kernel
    tol = TOL[dtype]
    a, b = ef_s.double().reshape(E * S, -1), ef.double().reshape(E * S, -1)
    assert torch.isfinite(a).all() and torch.isfinite(amp_s).all()
    rel_l2 = ((a - b).norm(dim=1) / b.norm(dim=1)).max().item()
    rel_amp = ((amp_s.double() - amp.double()).abs() / amp.double()).max().item()
    assert rel_l2 <= tol["l2"], (kernel, rel_l2)
    assert rel_amp <= tol["amp"], (kernel, rel_amp)
    assert torch.equal(idx_s, idx), kernel
    return kernel


def test_static_scratch_matches_workspace_path_on_consecutive_calls(B):
    wl = ai.WORKLOADS[1]                                    # N = 2048 fp32 at fs = 180 MHz: the warp kernel
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        B.aera_pattern_prepare(pat, wl.n_samples, wl.fs_hz)
        tr, dirs, _, _ = ai.make_batch(wl, [0, 1, 2, 3, 4], n_stations=9)
        tr, dirs = torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda()
        # call 1: five events; call 2: two other events at other directions, so the array still holds call 1's
        # matrices of events 2..4 behind (and different ones under) what call 2 writes
        assert _both_paths(B, pat, tr, dirs, wl.fs_hz, "f32") == "unfold_w32"
        tr2 = tr[3:5].flip(1).contiguous()
        dirs2 = torch.tensor([[71.5, 358.7], [0.0, 12.25]], dtype=torch.float64, device="cuda")
        assert _both_paths(B, pat, tr2, dirs2, wl.fs_hz, "f32") == "unfold_w32"
        # and once more with the first inputs: same answer as the first time
        assert _both_paths(B, pat, tr, dirs, wl.fs_hz, "f32") == "unfold_w32"
    finally:
        pat.free()
    # another dtype and kernel family on the same array right afterwards
    wl = ai.WORKLOADS[3]                                    # N = 4096 fp64: the team kernel
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F64), H)
    try:
        B.aera_pattern_prepare(pat, wl.n_samples, wl.fs_hz)
        tr, dirs, _, _ = ai.make_batch(wl, [0, 1], n_stations=5)
        assert _both_paths(B, pat, torch.from_numpy(tr).cuda(), torch.from_numpy(dirs).cuda(), wl.fs_hz, "f64") == "unfold_t4k_f64"
    finally:
        pat.free()


def test_static_scratch_refuses_what_it_cannot_serve(B):
    wl = ai.WORKLOADS[1]
    H = ai.pattern_table(wl.grid, wl.complex_dtype)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        limit = B.aera_static_scratch_bytes()
        assert limit == 32 << 20
        S, N = 1, wl.n_samples
        amp = lambda E: torch.empty((E, S), dtype=torch.float32, device="cuda")
        idx = lambda E: torch.empty((E, S), dtype=torch.int32, device="cuda")
        tr = torch.zeros((1, S, 2, N), dtype=torch.float32, device="cuda")
        dirs = torch.zeros((1, 2), dtype=torch.float64, device="cuda")
        # no plan yet: the call must not build one (that would be an allocation) and says which set-up call is missing
        with pytest.raises(B.AeraError) as ei:
            B.aera_unfold_batch_static(pat, tr, dirs, wl.fs_hz, None, amp(1), idx(1))
        assert ei.value.status == 1 and "aera_pattern_prepare" in str(ei.value)
        B.aera_pattern_prepare(pat, N, wl.fs_hz)
        B.aera_pattern_prepare(pat, N, wl.fs_hz)           # idempotent
        B.aera_unfold_batch_static(pat, tr, dirs, wl.fs_hz, None, amp(1), idx(1))
        # the largest batch that fits, and the first that does not (peaks only, one station per event: small buffers)
        e_max = 1656                                       # 20 256 bytes of matrices per event (include/aera_unfold.h)
        assert B.aera_workspace_bytes(B.AERA_OP_UNFOLD, pat, B.AERA_F32, e_max, S, N, wl.fs_hz) <= limit
        assert B.aera_workspace_bytes(B.AERA_OP_UNFOLD, pat, B.AERA_F32, e_max + 1, S, N, wl.fs_hz) > limit
        g = torch.Generator(device="cuda"); g.manual_seed(5)
        big = torch.randn((e_max + 1, S, 2, N), dtype=torch.float32, device="cuda", generator=g)
        bdirs = torch.stack([torch.linspace(0, 75, e_max + 1, dtype=torch.float64), torch.linspace(0, 359, e_max + 1, dtype=torch.float64)], 1).cuda()
        a_s, i_s = amp(e_max), idx(e_max)
        B.aera_unfold_batch_static(pat, big[:e_max], bdirs[:e_max], wl.fs_hz, None, a_s, i_s)
        _, a, i = B.aera_unfold_batch(pat, big[:e_max], bdirs[:e_max], wl.fs_hz, want_efield=False)
        torch.cuda.synchronize()
        assert ((a_s - a).abs() <= TOL["f32"]["amp"] * a).all() and torch.equal(i_s, i)
        with pytest.raises(B.AeraError) as ei:
            B.aera_unfold_batch_static(pat, big, bdirs, wl.fs_hz, None, amp(e_max + 1), idx(e_max + 1))
        assert ei.value.status == 4 and str(limit) in str(ei.value) and "split the events" in str(ei.value)
    finally:
        pat.free()
