"""Event sharding across GPUs: events are independent, so every rank reweights a contiguous range of
the sample with no data-path collective; only the three scalar sums of eqs.(6)-(7) would cross ranks."""


def shard_range(n, rank, world_size):
    """[lo, hi) of the events rank `rank` owns: contiguous, disjoint, covering, sizes differ by at most one."""
    if not (0 <= rank < world_size):
        raise ValueError("rank %d outside world of %d" % (rank, world_size))
    base, rem = divmod(int(n), int(world_size))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)
