"""The N > 1 path of bench.py on CPU: two gloo ranks take disjoint attitudes of the sweep and the
only collective (MAX of times, SUM of totals, after the timed region) gives the whole-job numbers.
The hot path itself needs no collective: attitudes are independent problems."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, out):
    sys.path.insert(0, ROOT)
    import bench
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    mine = [bench.attitude_index(k, rank, world, 64) for k in range(8)]
    times, totals = bench.reduce_over_ranks([100.0 + 7 * rank, 1.0 + rank], [1000 * (rank + 1), 10 * (rank + 1), 5], world)
    out.put((rank, mine, times, totals))
    dist.destroy_process_group()


def test_two_ranks_shard_attitudes_and_reduce():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (r0, a0, t0, s0), (r1, a1, t1, s1) = res
    assert not set(a0) & set(a1) and sorted(a0 + a1) == list(range(16))       # disjoint, contiguous coverage
    assert t0 == t1 == [107.0, 2.0]                                            # max over ranks
    assert s0 == s1 == [3000.0, 30.0, 10.0]                                    # sums over ranks


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks([3.0], [4.0, 5.0], 1) == ([3.0], [4.0, 5.0])
    assert [bench.attitude_index(k, 0, 1, 64) for k in (0, 1, 63, 64)] == [0, 1, 63, 0]
