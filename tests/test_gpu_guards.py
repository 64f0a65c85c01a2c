"""Out-of-bounds WRITES of every kernel family: outputs and workspace are carved out of larger buffers whose
surroundings carry a byte pattern; after the call the surroundings must be untouched and a workspace of exactly
aera_workspace_bytes must suffice (compute-sanitizer is not available on the GPU pool, so this is the bounds check)."""
import numpy as np
import pytest
import torch

import aera_inputs as ai

pytestmark = pytest.mark.gpu

GUARD = 1 << 16          # bytes on either side
PATTERN = 0xA5


@pytest.fixture(scope="module")
def B():
    import paper_1507_07733_b200.binding as b
    assert torch.cuda.is_available()
    return b


def guarded(nbytes, dtype, shape):
    """A tensor view of `shape` in the middle of a uint8 buffer filled with PATTERN (256-byte aligned start)."""
    raw = torch.full((nbytes + 2 * GUARD,), PATTERN, dtype=torch.uint8, device="cuda")
    view = raw[GUARD:GUARD + nbytes].view(dtype).view(shape)
    return raw, view


def intact(raw, nbytes):
    return bool((raw[:GUARD] == PATTERN).all().item() and (raw[GUARD + nbytes:] == PATTERN).all().item())


CASES = [  # dtype, N, fs, events, stations, expected kernel
    ("f32", 2048, 180e6, 3, 37, "unfold_w32"), ("f32", 2048, 200e6, 2, 13, "unfold_w32"), ("f32", 2048, 500e6, 2, 5, "unfold_w32"),
    ("f64", 4096, 200e6, 2, 7, "unfold_t4k_f64"), ("f32", 4096, 250e6, 2, 9, "unfold_t4k_f32"),
    ("f64", 2048, 200e6, 3, 5, "unfold_t2k_f64"), ("f64", 1024, 250e6, 3, 11, "unfold_t1k_f64"), ("f32", 1024, 200e6, 1, 19, "unfold_t1k_f32"),
    ("f32", 65536, 1e9, 1, 3, "unfold_long_f32"), ("f32", 256, 200e6, 2, 7, "generic"), ("f64", 16384, 200e6, 1, 2, "generic"),
    ("f32", 8192, 200e6, 2, 5, "unfold_t8k_f32"), ("f64", 8192, 250e6, 1, 3, "unfold_t8k_f64"), ("f32", 16384, 180e6, 1, 3, "unfold_t16k_f32"),
]


@pytest.mark.parametrize("dtype,N,fs,E,S,kernel", CASES)
def test_batch_writes_stay_inside_their_buffers(B, dtype, N, fs, E, S, kernel):
    grid = ai.WORKLOADS[4].grid if N == 65536 else ai.WORKLOADS[0].grid
    td = torch.float32 if dtype == "f32" else torch.float64
    dt = B.AERA_F32 if dtype == "f32" else B.AERA_F64
    H = ai.pattern_table(grid, np.complex64 if dtype == "f32" else np.complex128)
    pat = B.aera_pattern_upload(B.make_desc(grid, dt), H)
    try:
        g = torch.Generator(device="cuda"); g.manual_seed(N + S)
        tr = torch.randn(E, S, 2, N, dtype=td, device="cuda", generator=g)
        dirs = torch.tensor([[10.0 + 7 * e, 33.0 + 100 * e] for e in range(E)], dtype=torch.float64, device="cuda")
        es = tr.element_size()
        raw_ef, ef = guarded(E * S * 2 * N * es, td, (E, S, 2, N))
        raw_a, amp = guarded(E * S * es, td, (E, S))
        raw_i, idx = guarded(E * S * 4, torch.int32, (E, S))
        wsb = B.aera_workspace_bytes(B.AERA_OP_UNFOLD, pat, dt, E, S, N, fs)
        raw_w, ws = guarded(wsb, torch.uint8, (wsb,))
        B.aera_unfold_batch(pat, tr, dirs, fs, efield=ef, peak_amp=amp, peak_idx=idx, workspace=ws)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == kernel
        assert intact(raw_ef, E * S * 2 * N * es) and intact(raw_a, E * S * es) and intact(raw_i, E * S * 4) and intact(raw_w, wsb)
        assert torch.isfinite(ef).all() and torch.isfinite(amp).all()
        assert int(idx.min()) >= 0 and int(idx.max()) < N
        # the same call with the plain allocation gives the same bits (the guarded views change nothing but the addresses)
        ef2, amp2, idx2 = B.aera_unfold_batch(pat, tr, dirs, fs)
        torch.cuda.synchronize()
        assert torch.equal(ef, ef2) and torch.equal(amp, amp2) and torch.equal(idx, idx2)
    finally:
        pat.free()


@pytest.mark.parametrize("fs,D,S", [(180e6, 50, 9), (200e6, 31, 6), (500e6, 7, 5)])
def test_scan_writes_stay_inside_their_buffers(B, fs, D, S):
    wl = ai.WORKLOADS[2]
    H = ai.pattern_table(wl.grid, np.complex64)
    pat = B.aera_pattern_upload(B.make_desc(wl.grid, B.AERA_F32), H)
    try:
        g = torch.Generator(device="cuda"); g.manual_seed(D)
        tr = torch.randn(S, 2, 2048, dtype=torch.float32, device="cuda", generator=g)
        dirs = torch.from_numpy(ai.scan_directions()[::7380 // D][:D].copy()).cuda()
        raw_a, amp = guarded(D * S * 4, torch.float32, (D, S))
        raw_i, idx = guarded(D * S * 4, torch.int32, (D, S))
        wsb = B.aera_workspace_bytes(B.AERA_OP_SCAN, pat, B.AERA_F32, D, S, 2048, fs)
        raw_w, ws = guarded(wsb, torch.uint8, (wsb,))
        B.aera_scan_directions(pat, tr, dirs, fs, peak_amp=amp, peak_idx=idx, workspace=ws)
        torch.cuda.synchronize()
        assert B.aera_last_kernel() == "scan_w32"
        assert intact(raw_a, D * S * 4) and intact(raw_i, D * S * 4) and intact(raw_w, wsb)
        assert torch.isfinite(amp).all() and int(idx.min()) >= 0 and int(idx.max()) < 2048
    finally:
        pat.free()
