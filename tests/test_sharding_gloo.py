"""N > 1 host logic on CPU: world_size-2 gloo processes (the data path itself has no collective)."""
import os
import sys

import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from paper_1206_1779_b200.sharding import shard_systems, max_over_ranks, aggregate_throughput
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    lo, hi = shard_systems(257, world, rank)
    tmax = max_over_ranks(1.0 + rank)
    thr = aggregate_throughput(hi - lo, 1.0 + rank)
    q.put((rank, lo, hi, tmax, thr))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_sharding_and_timing():
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, lo0, hi0, t0, th0), (r1, lo1, hi1, t1, th1) = out
    assert (lo0, hi0, lo1, hi1) == (0, 129, 129, 257)          # contiguous, balanced, covers everything once
    assert t0 == t1 == 2.0                                      # max over ranks
    assert abs(th0 - 257 / 2.0) < 1e-12 and th0 == th1          # all ranks' units / max time


def test_shard_systems_properties():
    sys.path.insert(0, ROOT)
    from paper_1206_1779_b200.sharding import shard_systems
    for n in (1, 5, 256, 257):
        for world in (1, 2, 3, 8):
            cuts = [shard_systems(n, world, r) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n
            assert all(cuts[i][1] == cuts[i + 1][0] for i in range(world - 1))
            sizes = [b - a for a, b in cuts]
            assert max(sizes) - min(sizes) <= 1
