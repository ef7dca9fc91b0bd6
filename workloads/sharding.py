"""Data-parallel sharding of the hot path over ranks (each device generates its own
data, multi-device brings no data-path exchange).  No arithmetic of the method lives here.

Two ways to use N ranks, both without a data-path collective:
  * weak scaling (bench.py): every rank assembles its own batch of the full per-GPU size from its own seed;
  * strong split: one global batch is cut into contiguous per-rank slices (the per-detector PSD is recomputed on every
    rank from the same background: 189 small FFTs, cheaper than any exchange).
The only collective is the MAX over ranks of the measured time (timing plumbing, not data path).
"""


def rank_seed(base_seed, rank):
    """Seed of the synthetic workload of `rank` (weak scaling: independent data per rank)."""
    return int(base_seed) + int(rank)


def shard_batch(global_batch, world, rank):
    """Contiguous slice [start, start + count) of a global batch owned by `rank`; slices are disjoint, ordered by rank,
    cover [0, global_batch) and differ in size by at most one."""
    if world < 1 or not (0 <= rank < world) or global_batch < 0:
        raise ValueError("need world >= 1, 0 <= rank < world, global_batch >= 0")
    base, rem = divmod(global_batch, world)
    start = rank * base + min(rank, rem)
    return start, base + (1 if rank < rem else 0)


def max_over_ranks(value, dist=None, device=None):
    """MAX of a python float over all ranks (identity without a process group)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(units_per_rank, world, ms_per_step_max):
    """Whole-job throughput: the units all ranks processed in a step / the slowest rank's step time."""
    return world * units_per_rank / (ms_per_step_max * 1e-3)
