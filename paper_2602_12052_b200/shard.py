"""Host-side sharding of the path over ranks.

The path shards over independent events / drift volumes (the paper processes TPC volumes
"independently in sequence"): one process per GPU, every rank simulates
its own events and there is NO data-path collective.  The only communication is the
reduction of the timing record (max of the per-rank times, sum of the units processed),
which is what this module holds; it has none of the method's arithmetic.
"""
from __future__ import annotations


def event_seed(cfg_id: int, event: int) -> int:
    """Seed of the synthetic event `event` of a configuration (event 0 = the BASELINE one)."""
    return 1000 + int(cfg_id) + int(event)


def shard_events(n_events: int, world: int, rank: int) -> range:
    """Contiguous, balanced split of event ids 0..n_events-1: the first n_events % world
    ranks get one more.  Every event belongs to exactly one rank."""
    if world < 1 or not (0 <= rank < world) or n_events < 0:
        raise ValueError("bad shard arguments")
    q, r = divmod(n_events, world)
    lo = rank * q + min(rank, r)
    return range(lo, lo + q + (1 if rank < r else 0))


def reduce_timing(ms_local, units_local: float, device=None):
    """(max over ranks of every entry of ms_local, sum over ranks of units_local).
    Works without an initialised process group (world 1), on gloo (CPU tensors) and on
    nccl (pass the rank's CUDA device)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x) for x in ms_local], dtype=torch.float64, device=device)
    n = torch.tensor([float(units_local)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        dist.all_reduce(n, op=dist.ReduceOp.SUM)
    return [float(x) for x in t.tolist()], float(n.item())
