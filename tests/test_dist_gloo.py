"""The N > 1 host logic of bench.py (plan sharding over ranks, max-over-ranks time, summed work) with
world_size 2 on the gloo backend.  CPU only."""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    from workloads import weight_grid
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    _, _, weights = weight_grid(9)
    mine = bench.rank_weights(weights, rank, world)
    # every rank times its own shard; the job time is the max, the work is the sum
    ms = 100.0 + 50.0 * rank
    plan_iters = 1000 * (rank + 1)
    (tmax,), (total, launches) = bench.reduce_max_sum(dist, torch.device("cpu"), [ms], [plan_iters, 7])
    dist.barrier()
    q.put((rank, mine[:, 1].tolist(), mine[:, 2].tolist(), tmax, total, launches))
    dist.destroy_process_group()


def test_two_rank_sharding_and_reduction():
    world, port = 2, 29517 + (os.getpid() % 200)
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, a0, b0, t0, s0, l0), (r1, a1, b1, t1, s1, l1) = got
    assert t0 == t1 == 150.0 and s0 == s1 == 3000.0 and l0 == l1 == 14.0
    assert b0 == b1                                  # same beam-on-time weights
    assert a0 != a1 and max(a1) <= 1.0 and min(a1) > min(a0) - 1e-12
    assert np.allclose(np.array(a1)[:72] - np.array(a0)[:72], 1.0 / 16.0 / 8.0)
    # rank 0 of any world keeps the unshifted grid
    sys.path.insert(0, ROOT)
    import bench
    from workloads import weight_grid
    _, _, weights = weight_grid(9)
    assert np.array_equal(bench.rank_weights(weights, 0, 8), weights)
