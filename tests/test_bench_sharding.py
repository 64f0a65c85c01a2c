"""Host-side multi-GPU logic on CPU: world_size-2 gloo processes exercise the event sharding, the
max-over-ranks timing / whole-job throughput aggregation and the optional peak gather
(paper_1507_07733_b200/sharding.py, used by bench.py). No kernels run here."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_1507_07733_b200 import sharding


def test_shard_range_tiles_exactly():
    for n in (0, 1, 7, 124, 1000, 7380):
        for world in (1, 2, 3, 4, 8):
            got = []
            sizes = []
            for r in range(world):
                sh = sharding.shard_range(n, r, world)
                got.extend(sh)
                sizes.append(len(sh))
            assert got == list(range(n))
            assert max(sizes) - min(sizes) <= 1
    with pytest.raises(ValueError):
        sharding.shard_range(10, 2, 2)


def test_weak_events_are_disjoint():
    a, b = sharding.weak_events(200, 0), sharding.weak_events(200, 1)
    assert set(a).isdisjoint(b) and len(a) == len(b) == 200 and b[0] == 200


def test_scan_shards_reassemble_in_direction_order():
    import numpy as np
    import aera_inputs as ai
    dirs = ai.scan_directions()
    for world in (1, 2, 3, 8):
        parts = [sharding.scan_shard(dirs, r, world) for r in range(world)]
        assert np.array_equal(np.concatenate(parts), dirs)
        assert max(len(p) for p in parts) - min(len(p) for p in parts) <= 1


def test_aggregate_single_process():
    u, ms, v = sharding.aggregate_throughput(124000, 1.0)
    assert (u, ms) == (124000, 1.0) and abs(v - 1.24e8) < 1e-3


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    try:
        n_events = 11
        sh = sharding.shard_range(n_events, rank, world)
        # fake per-event "results": amp = event id, idx = 10 * event id, 3 stations each
        amp = torch.tensor([[float(e)] * 3 for e in sh], dtype=torch.float32).reshape(len(sh), 3)
        idx = torch.tensor([[10 * e] * 3 for e in sh], dtype=torch.int32).reshape(len(sh), 3)
        A, I = sharding.gather_peaks(amp, idx)
        ms_local = 2.0 if rank == 0 else 5.0     # the slower rank must decide
        units, ms, val = sharding.aggregate_throughput(len(sh) * 3, ms_local)
        q.put((rank, A[:, 0].tolist(), I[:, 0].tolist(), units, ms, val))
    finally:
        dist.destroy_process_group()


def test_world_size_2_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = [q.get(timeout=120) for _ in procs]
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, A, I, units, ms, val in res:
        assert A == [float(e) for e in range(11)]          # rank order, ragged shards (5 + 6)
        assert I == [10 * e for e in range(11)]
        assert units == 33 and ms == 5.0
        assert abs(val - 33 / 5e-3) < 1e-6
