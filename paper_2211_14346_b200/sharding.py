"""Host-side plumbing for running the path on several GPUs (one process per GPU, torch.distributed).

Events are independent ("assigns different events to different computing threads") and the smearing
stream is keyed by the GLOBAL event index (hepf_events_t.event_base), so the path shards with no data-path
collective: rank r owns a contiguous range of events and runs hepf_select + hepf_reconstruct_tth on it.  The only
exchange a global result needs is tiny and latency-bound: the survivor counts (all-gather of one int64 per rank ->
each rank's offset into the global survivor list) and the cutflow (all-reduce of <= 32 int64).  DESIGN.md §8.
"""
from __future__ import annotations


def shard_range(n_events: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous range [lo, hi) of rank `rank`.  The unit is FOUR events, so every boundary is a multiple of 4: a
    pointer-offset view of a resident store (DeviceEvents.subview) then keeps the 16-byte alignment hepf_events_t asks
    of every column, the 4-byte flags column included; sizes differ by at most seven events."""
    quads = (n_events + 3) // 4
    base, rem = divmod(quads, world)
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return min(4 * lo, n_events), min(4 * hi, n_events)


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
