"""Multi-GPU plumbing: photons are independent, so the path shards by contiguous
global photon-id ranges with the scene and BVH replicated on every GPU.  Philox is keyed by the global
id, hence results do not depend on the number of ranks.  The only exchange is one sum all-reduce of
the pixel hit-map and of the 8 counters; hit records stay sharded.  No arithmetic of the method here.
"""


def shard_range(n_total, rank, world):
    """Contiguous id range [start, start + count) of `rank`: the first n_total % world ranks get one
    extra photon, so counts differ by at most one and the ranges tile [0, n_total) exactly."""
    if not (0 <= rank < world):
        raise ValueError("rank out of range")
    base, extra = divmod(int(n_total), int(world))
    start = rank * base + min(rank, extra)
    return start, base + (1 if rank < extra else 0)


def allreduce_accumulators(hitmap, counters, group=None):
    """Sum the per-rank hit-maps (uint32 bit pattern in an int32 tensor) and counters (int64) over the
    process group, in place.  NCCL on GPUs, gloo in the CPU tests."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(hitmap, op=dist.ReduceOp.SUM, group=group)
        dist.all_reduce(counters, op=dist.ReduceOp.SUM, group=group)
    return hitmap, counters
