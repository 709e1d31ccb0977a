"""Host-side plumbing for running the path on several GPUs (one process per GPU, torch.distributed).

Events are independent ("assigns different events to different computing threads") and the smearing
stream is keyed by the GLOBAL event index (hepf_events_t.event_base), so the path shards with no data-path
collective: rank r owns a contiguous range of events and runs hepf_select + hepf_reconstruct_tth on it.  The only
exchange a global result needs is tiny and latency-bound: the survivor counts (all-gather of one int64 per rank ->
each rank's offset into the global survivor list) and the cutflow (all-reduce of <= 32 int64).  DESIGN.md §8.
"""
from __future__ import annotations


def shard_range(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range [lo, hi) of rank `rank`.  The unit is a PAIR of events, so every boundary is even and a slice
    of an even-stride SoA store keeps its 16-byte row alignment; sizes differ by at most three events."""
    pairs = (n_events + 1) // 2
    base, rem = divmod(pairs, world)
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return min(2 * lo, n_events), min(2 * hi, n_events)


def global_survivor_offset(local_count: int, group=None, device="cpu") -> tuple[int, int]:
    """(offset of this rank's survivors in the global ascending list, global survivor count)."""
    import torch
    import torch.distributed as dist
    world, rank = dist.get_world_size(group), dist.get_rank(group)
    mine = torch.tensor([int(local_count)], dtype=torch.int64, device=device)
    allc = [torch.zeros_like(mine) for _ in range(world)]
    dist.all_gather(allc, mine, group=group)
    counts = [int(c.item()) for c in allc]
    return sum(counts[:rank]), sum(counts)


def global_cutflow(local_cutflow, group=None):
    """Sum of the per-rank cutflow vectors (int64 tensor, reduced in place and returned)."""
    import torch.distributed as dist
    dist.all_reduce(local_cutflow, op=dist.ReduceOp.SUM, group=group)
    return local_cutflow
