"""Event sharding across GPUs: events are independent, so every rank reweights a contiguous range of
the sample with no data-path collective; only the scalar sums of eqs.(6)-(7) cross ranks.

`launch_ranks` starts one process per GPU (torch.distributed.run, rendezvous on 127.0.0.1); `python -m
paper_2510_05100_b200.shard` is the small self-check those ranks can run on CPU (gloo) or GPU (nccl)."""
import json
import os
import socket
import subprocess
import sys


def shard_range(n, rank, world_size):
    """[lo, hi) of the events rank `rank` owns: contiguous, disjoint, covering, sizes differ by at most one."""
    if not (0 <= rank < world_size):
        raise ValueError("rank %d outside world of %d" % (rank, world_size))
    base, rem = divmod(int(n), int(world_size))
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def shard_arrays(n, rank, world_size, *arrays):
    """This rank's contiguous slice [lo, hi) of every array along its LAST axis (the event axis of the SoA layout)."""
    import numpy as np
    lo, hi = shard_range(n, rank, world_size)
    out = []
    for a in arrays:
        if a.shape[-1] != n:
            raise ValueError("event axis has %d entries, expected %d" % (a.shape[-1], n))
        out.append(np.ascontiguousarray(a[..., lo:hi]))
    return out


def free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def launch_ranks(script, nranks, argv, port=None, timeout=None, env=None, module=False):
    """Run `script argv...` as `nranks` ranks of one node (one process per GPU): torch.distributed.run with the
    rendezvous on 127.0.0.1 (the container hostname may not resolve). Returns the exit code; the ranks' stdout/stderr
    are inherited, so rank 0's JSON line is the launcher's output."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(int(nranks)),
           "--master-addr", "127.0.0.1", "--master-port", str(port or free_port())]
    cmd += (["-m", script] if module else [script]) + list(argv)
    e = dict(os.environ)
    e.setdefault("NCCL_DEBUG", "WARN")
    e.setdefault("OMP_NUM_THREADS", str(max(1, (os.cpu_count() or 1) // max(1, int(nranks)))))
    if env:
        e.update(env)
    return subprocess.call(cmd, env=e, timeout=timeout)


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


def _selfcheck(argv):
    """What every rank of a launch does with its shard, without the GPU kernels: slice a seeded sample, all-reduce the
    coverage, combine the eq.(6)-(7) moments of the shards. Rank 0 prints one JSON line."""
    import numpy as np
    import torch
    import torch.distributed as dist
    n = int(argv[0]) if argv else 1001
    out = argv[1] if len(argv) > 1 else None
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    backend = "nccl" if torch.cuda.is_available() and os.environ.get("TREX_SHARD_BACKEND", "") != "gloo" else "gloo"
    if backend == "nccl":
        torch.cuda.set_device(int(os.environ.get("LOCAL_RANK", "0")))
    dist.init_process_group(backend)
    rng = np.random.default_rng(21)
    w = rng.lognormal(0, 0.5, n)
    wo = w * rng.uniform(0.5, 2.0, n)
    idx = np.arange(n)
    a, b, mine = shard_arrays(n, rank, world, w, wo, idx)
    dev = torch.device("cuda") if backend == "nccl" else torch.device("cpu")
    cover = torch.zeros(n, dtype=torch.int64, device=dev)
    cover[torch.from_numpy(mine).to(dev)] = 1
    dist.all_reduce(cover)
    mean = b.mean() if len(b) else 0.0
    mom = [float(len(b)), float(b.sum()), float((b / a).sum()), float(((b - mean) ** 2).sum())]
    res = xsec_all_ranks(mom, 0.1, 5.0, 0.2)
    gathered = [None] * world
    dist.all_gather_object(gathered, [float(res[0]), float(res[1]), bool(res[2])])
    if rank == 0:
        line = json.dumps({"world": world, "backend": backend, "n": n, "covered_once": bool((cover == 1).all().item()),
                           "xsec": gathered})
        if out:
            with open(out, "w") as fh:
                fh.write(line + "\n")
        print(line)
    dist.barrier()
    dist.destroy_process_group()


if __name__ == "__main__":
    _selfcheck(sys.argv[1:])
