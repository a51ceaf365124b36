"""Multi-GPU plan: particles are independent, so every rank owns a contiguous index range of
the population, keeps its own copy of the tables and runs the single-GPU path on its shard.  There is no
data-path collective; the only exchanges are host-side: the max over ranks of a timing, and (for a globally
ordered secondary buffer) one count per rank per step, whose exclusive scan gives the rank's output offset."""
import torch
import torch.distributed as dist


def shard_range(rank, world, n_total):
    """contiguous, balanced [lo, hi) of rank; the particle id of local index i is lo + i (id_base = lo)"""
    base, rem = divmod(int(n_total), int(world))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def max_over_ranks(value, device="cpu"):
    """max of a host scalar over all ranks (timings are reported as the slowest rank's)"""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def secondary_offsets(n_local, device="cpu"):
    """(offset of this rank's secondaries in the globally index-ordered buffer, global total): an all-gather of
    one count per rank and an exclusive scan; ranks hold ascending index ranges, so rank order = index order"""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return 0, int(n_local)
    world, rank = dist.get_world_size(), dist.get_rank()
    mine = torch.tensor([int(n_local)], dtype=torch.int64, device=device)
    counts = [torch.zeros(1, dtype=torch.int64, device=device) for _ in range(world)]
    dist.all_gather(counts, mine)
    counts = [int(c.item()) for c in counts]
    return sum(counts[:rank]), sum(counts)
