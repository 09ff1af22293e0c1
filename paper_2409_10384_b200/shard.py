"""Host-side multi-GPU plumbing: MeshBlocks are independent units, so the block
list shards across ranks with no collective on the data path.  The only communication is the
reduction of timings / counters for reporting."""
import numpy as np


def shard_blocks(nmb, rank, world):
    """contiguous, near-equal ranges of block ids: rank r owns [lo, hi)."""
    if not (0 <= rank < world):
        raise ValueError("rank %d outside world %d" % (rank, world))
    base, rem = divmod(nmb, world)
    lo = rank * base + min(rank, rem)
    hi = lo + base + (1 if rank < rem else 0)
    return lo, hi


def rank_block_ids(all_ids, rank, world, strong):
    """block ids a rank works on: its shard of the list (strong scaling) or the whole list
    (weak scaling: every rank runs its own batch of the same shape)."""
    all_ids = np.asarray(all_ids)
    if not strong:
        return all_ids
    lo, hi = shard_blocks(len(all_ids), rank, world)
    return all_ids[lo:hi]


def reduce_max(value, device=None):
    """max over ranks of a scalar (timings are reported as the slowest rank's)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def reduce_sum(value, device=None):
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return float(t.item())
