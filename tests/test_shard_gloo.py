"""N > 1 host logic on CPU: world_size-2 gloo run of the sharding used by bench.py. The data path has
no collective; the ranks only agree on disjoint covering ranges and on the max-over-ranks timing reduction."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2510_05100_b200.shard import shard_range


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, n, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_range(n, rank, world)
    mine = torch.zeros(n, dtype=torch.int64)
    mine[lo:hi] = 1
    dist.all_reduce(mine)                                   # coverage count per event
    t = torch.tensor([float(rank + 1)], dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)                # bench.py: time = max over ranks
    cnt = torch.tensor([hi - lo], dtype=torch.int64)
    dist.all_reduce(cnt)
    if rank == 0:
        out.put((mine.numpy().copy(), float(t.item()), int(cnt.item())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_covers_every_event_once():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    n, world, port = 1001, 2, _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, n, q)) for r in range(world)]
    for p in procs:
        p.start()
    cover, tmax, total = q.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert np.all(cover == 1) and tmax == 2.0 and total == n


def test_shard_range_properties():
    for n in (0, 1, 7, 64, 1001):
        for world in (1, 2, 3, 8):
            r = [shard_range(n, k, world) for k in range(world)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(world - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def _xsec_worker(rank, world, port, n, out):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from paper_2510_05100_b200.shard import xsec_all_ranks
    rng = np.random.default_rng(21)
    w = rng.lognormal(0, 0.5, n)
    wo = w * rng.uniform(0.5, 2.0, n)
    lo, hi = shard_range(n, rank, world)
    a, b = w[lo:hi], wo[lo:hi]
    mom = [float(hi - lo), float(b.sum()), float((b / a).sum()), float(((b - b.mean()) ** 2).sum())]
    res = xsec_all_ranks(mom, 0.1, 5.0, 0.2)
    gathered = [None] * world
    dist.all_gather_object(gathered, res)
    if rank == 0:
        out.put(gathered)
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_cross_section_equals_the_single_rank_definition():
    """eqs.(6)-(7) over a sharded sample: the all-gather of four moments per rank is the only exchange."""
    from oracle import oracle as O
    n = 1001
    ctx = mp.get_context("spawn")
    out = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_xsec_worker, args=(r, 2, port, n, out)) for r in range(2)]
    for p in procs:
        p.start()
    res = out.get(timeout=120)
    for p in procs:
        p.join(timeout=60)
    rng = np.random.default_rng(21)
    w = rng.lognormal(0, 0.5, n)
    wo = w * rng.uniform(0.5, 2.0, n)
    ref = O.xsec(w, wo, 0.1, 5.0, 0.2)
    assert res[0] == res[1]                                    # every rank holds the same numbers
    assert abs(res[0][0] / ref[0] - 1) < 1e-13 and abs(res[0][1] / ref[1] - 1) < 1e-12 and not res[0][2]


def test_launcher_starts_two_ranks_that_shard_and_combine(tmp_path):
    """bench.py --gpus N uses shard.launch_ranks when it is not already under torchrun: the same launcher, world_size 2,
    gloo on CPU, running the package's shard self-check (slices, coverage all-reduce, eq.(6)-(7) all-gather)."""
    import json
    from oracle import oracle as O
    from paper_2510_05100_b200.shard import launch_ranks
    n = 1001
    out = tmp_path / "shard.json"
    rc = launch_ranks("paper_2510_05100_b200.shard", 2, [str(n), str(out)], module=True, timeout=300,
                      env={"TREX_SHARD_BACKEND": "gloo", "CUDA_VISIBLE_DEVICES": ""})
    assert rc == 0
    res = json.loads(out.read_text())
    assert res["world"] == 2 and res["backend"] == "gloo" and res["covered_once"] is True
    rng = np.random.default_rng(21)
    w = rng.lognormal(0, 0.5, n)
    wo = w * rng.uniform(0.5, 2.0, n)
    ref = O.xsec(w, wo, 0.1, 5.0, 0.2)
    assert res["xsec"][0] == res["xsec"][1]
    assert abs(res["xsec"][0][0] / ref[0] - 1) < 1e-13 and abs(res["xsec"][0][1] / ref[1] - 1) < 1e-12


def test_shard_arrays_slices_the_event_axis():
    from paper_2510_05100_b200.shard import shard_arrays
    n = 37
    keys = np.arange(n, dtype=np.uint64)
    mom = np.arange(5 * 4 * n, dtype=np.float64).reshape(5, 4, n)
    got = [shard_arrays(n, r, 3, keys, mom) for r in range(3)]
    assert np.array_equal(np.concatenate([g[0] for g in got]), keys)
    assert np.array_equal(np.concatenate([g[1] for g in got], axis=2), mom)
    assert all(g[1].flags.c_contiguous for g in got)
