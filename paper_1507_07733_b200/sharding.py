"""Multi-GPU plumbing (one process per GPU): how a batch is split across ranks and how the
per-rank timings become one whole-job number.

The method has no exchange step (units are independent, PAPER.md L29 gives one
direction per event), so nothing here touches the data path: `aera_unfold_batch` is sharded by
EVENT (keeps each event's Minv local to one rank), `aera_scan_directions` by DIRECTION, the
pattern table is replicated by each rank's own upload, and the only collectives are a barrier and
a MAX/SUM reduction of a few scalars. Works on any torch.distributed backend (nccl on the GPU box,
gloo in the CPU tests).
"""
from __future__ import annotations


def shard_range(n_items: int, rank: int, world: int) -> range:
    """Contiguous, balanced split of range(n_items): rank r gets [r n/W, (r+1) n/W) (integer floor),
    so sizes differ by at most one and the shards tile the range exactly, in rank order."""
    if world < 1 or not (0 <= rank < world):
        raise ValueError(f"rank {rank} / world {world}")
    if n_items < 0:
        raise ValueError("n_items < 0")
    return range(n_items * rank // world, n_items * (rank + 1) // world)


def scan_shard(dirs, rank: int, world: int):
    """`aera_scan_directions` across ranks: rank r scans the contiguous block shard_range(n_dirs, r, world) of the
    direction list against ALL stations (the forward spectra are recomputed per rank: 124 transforms against
    ~10^5 pairs). The peaks are [n_dirs][n_stations], direction-major, so the ranks' outputs concatenated in rank
    order (gather_peaks) are the single-GPU result. The total work is fixed as the ranks grow: strong scaling."""
    sh = shard_range(int(dirs.shape[0]), rank, world)
    return dirs[sh.start:sh.stop]


def weak_events(n_events_per_gpu: int, rank: int) -> range:
    """Weak scaling (bench.py): every rank processes its own n_events_per_gpu canonical events."""
    return range(rank * n_events_per_gpu, (rank + 1) * n_events_per_gpu)


def aggregate_throughput(units_local: int, ms_local: float, device=None):
    """(total units over all ranks, max time over ranks in ms, units per second of the whole job).
    With no process group initialised this is the single-rank answer."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return units_local, ms_local, units_local / (ms_local * 1e-3)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return int(u.item()), float(t.item()), float(u.item()) / (float(t.item()) * 1e-3)


def gather_peaks(amp_local, idx_local):
    """Optional result exchange (8 B per unit): all ranks' (amp, idx) concatenated in rank order.
    Shards may have different lengths (shard_range), so sizes are exchanged first."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return amp_local, idx_local
    world = dist.get_world_size()
    n = torch.tensor([amp_local.shape[0]], dtype=torch.int64, device=amp_local.device)
    sizes = [torch.zeros_like(n) for _ in range(world)]
    dist.all_gather(sizes, n)
    sizes = [int(s.item()) for s in sizes]
    m = max(sizes)
    tail = amp_local.shape[1:]

    def padded(x):
        out = x.new_zeros((m,) + tuple(tail))
        out[: x.shape[0]] = x
        return out

    amps = [amp_local.new_zeros((m,) + tuple(tail)) for _ in range(world)]
    idxs = [idx_local.new_zeros((m,) + tuple(tail)) for _ in range(world)]
    dist.all_gather(amps, padded(amp_local))
    dist.all_gather(idxs, padded(idx_local))
    return (torch.cat([a[:s] for a, s in zip(amps, sizes)]), torch.cat([i[:s] for i, s in zip(idxs, sizes)]))
