"""Multi-GPU plumbing of the benchmark/driver layer: galaxies are independent
(PAPER.md:107), so ranks hold disjoint galaxy shards, replicate the tables and exchange nothing on the data
path; only the timings are combined (MAX over ranks) with one all-reduce.  Pure host logic: works on any
torch.distributed backend (nccl on GPUs, gloo in the CPU tests)."""
from __future__ import annotations


def galaxy_shard(n_gal_total: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous shard [start, stop) of a catalogue of n_gal_total galaxies (strong scaling split)."""
    base, rem = divmod(n_gal_total, world)
    start = rank * base + min(rank, rem)
    return start, start + base + (1 if rank < rem else 0)


def rank_seed(seed: int, rank: int) -> int:
    """Seed of a rank's synthetic galaxies in the weak-scaling benchmark (every rank draws its own catalogue)."""
    return seed + 1000 * rank


def max_over_ranks(values, dist=None, device="cpu"):
    """Element-wise MAX of a list of floats over all ranks (identity without a process group)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return [float(v) for v in values]
    import torch
    t = torch.tensor(list(values), dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return t.tolist()


def aggregate_throughput(units_per_rank: float, world: int, seconds_max: float) -> float:
    """Whole-job throughput: all ranks' units over the slowest rank's time."""
    return units_per_rank * world / seconds_max
