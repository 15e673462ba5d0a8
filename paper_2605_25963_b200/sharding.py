"""Multi-GPU sharding of histories: histories are independent and the RNG is keyed by the global
history index, so rank r transports a contiguous range and the only exchange is one integer sum of the tallies
(spectrum + per-line counters, ~33 KB) -- bit-identical for any number of ranks.  One process per GPU."""
from __future__ import annotations


def history_range(n_total: int, rank: int, world: int, first: int = 0):
    """Contiguous split of [first, first + n_total) over `world` ranks; the first n_total % world ranks get one more."""
    if world <= 0 or not (0 <= rank < world) or n_total < 0:
        raise ValueError("bad shard request")
    base, rem = divmod(n_total, world)
    count = base + (1 if rank < rem else 0)
    start = first + rank * base + min(rank, rem)
    return start, count


def allreduce_tallies(tally, group=None):
    """In-place integer SUM of a tally tensor (int64 view of the uint64 tallies) over the process group.
    `tally` lives on the GPU for the nccl backend and on the CPU for gloo (tests)."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(tally, op=dist.ReduceOp.SUM, group=group)
    return tally
