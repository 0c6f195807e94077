"""Batch partitioning for more than one GPU: the B matrices are independent 64-byte units
(PAPER.md:170-172), so the batch dimension is cut into contiguous, near-equal shards, one per rank, and no
data-path collective exists.  Host logic only; holds none of the method's arithmetic.
"""


def shard_bounds(B, world_size, rank):
    """[lo, hi) of rank's shard: the first B % world_size ranks get one matrix more."""
    if world_size < 1 or not 0 <= rank < world_size or B < 0:
        raise ValueError("bad shard request")
    q, r = divmod(B, world_size)
    lo = rank * q + min(rank, r)
    return lo, lo + q + (1 if rank < r else 0)


def reduce_max_time(ms, dist=None):
    """max over ranks of a per-rank duration (the only cross-rank traffic of bench.py: timing, not data)."""
    if dist is None or not dist.is_initialized() or dist.get_world_size() == 1:
        return float(ms)
    import torch
    dev = "cuda" if dist.get_backend() == "nccl" else "cpu"
    t = torch.tensor([float(ms)], dtype=torch.float64, device=dev)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())
