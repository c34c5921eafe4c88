"""Host-side logic of the N > 1 path.

Every output node is independent, so the path shards by batch with NO
data-path collective: rank r runs the same step on its own seeded batch.  The only communication is
the timing/metric reduction of bench.py: the step time is the MAX over ranks, the node count the SUM.
This module holds that logic so that it can be tested on CPU with the gloo backend.
"""
from __future__ import annotations


def rank_seed(base_seed: int, rank: int) -> int:
    """Seed of rank `rank`'s batch: distinct, reproducible batches per rank."""
    return int(base_seed) + 100 * int(rank)


def tile_owner(tile_index: int, world: int) -> int:
    """Round-robin owner of an output tile when ONE survey is split across ranks (replicated index,
    sharded output tiles; not used by bench.py, which runs whole batches per rank)."""
    return int(tile_index) % max(int(world), 1)


def tiles_of_rank(tiles, rank: int, world: int):
    """The tiles of ONE survey that rank `rank` predicts (replicated index, output
    tiles dealt round-robin in arrival order).  Every tile has exactly one owner."""
    return [t for i, t in enumerate(tiles) if tile_owner(i, world) == int(rank)]


def broadcast_soundings(x, y, z, dist=None, src: int = 0):
    """Replicates the sounding set of rank `src` on every rank (one broadcast of <= 64 MB over NCCL / NVLink on
    GPUs, gloo on CPU): the only data-plane communication of the one-survey sharding.  x, y, z: float32 tensors
    of equal length on every rank (contents are only read on `src`).  Returns the three tensors."""
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        for t in (x, y, z):
            dist.broadcast(t, src=src)
    return x, y, z


def reduce_step_times(times_ms, dist=None, device=None):
    """MAX over ranks of each entry of `times_ms` (list of floats).  `dist` is torch.distributed (or
    None for a single process)."""
    import torch
    t = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def whole_job_throughput(units_per_rank: float, world: int, max_ms_per_step: float) -> float:
    """Whole-job units per second: the units all ranks processed divided by the slowest rank's time."""
    return float(world) * float(units_per_rank) / (float(max_ms_per_step) * 1e-3)
