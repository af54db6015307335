"""Event sharding across GPUs: events are independent, so every rank reweights a contiguous range of
the sample with no data-path collective; only the three scalar sums of eqs.(6)-(7) would cross ranks."""


def shard_range(n, rank, world_size):
    """[lo, hi) of the events rank `rank` owns: contiguous, disjoint, covering, sizes differ by at most one."""
    if not (0 <= rank < world_size):
        raise ValueError("rank %d outside world of %d" % (rank, world_size))
    base, rem = divmod(int(n), int(world_size))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def xsec_all_ranks(moments, C, sigma, dsigma, group=None):
    """Reweighted cross section of a sample sharded over ranks: every rank passes the moments of ITS events
    (`trex_xsec_moments`), the four numbers are all-gathered (the only exchange of the path, 32 B per rank) and every
    rank combines them in rank order with `trex_xsec_finish` -- same result on all ranks, independent of timing."""
    import numpy as np
    import torch
    import torch.distributed as dist
    from .binding import trex_xsec_finish
    mine = torch.from_numpy(np.asarray(moments, dtype=np.float64).reshape(4).copy())
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        backend = dist.get_backend(group)
        dev = torch.device("cuda", torch.cuda.current_device()) if backend == "nccl" else torch.device("cpu")
        parts = [torch.empty(4, dtype=torch.float64, device=dev) for _ in range(dist.get_world_size(group))]
        dist.all_gather(parts, mine.to(dev), group=group)
        allm = torch.stack(parts).cpu().numpy()
    else:
        allm = mine.numpy().reshape(1, 4)
    return trex_xsec_finish(allm, C, sigma, dsigma)
