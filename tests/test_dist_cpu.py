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


def _slice_worker(rank, world, port, out):
    """SURVEY 8(e), the particle-range split: each rank runs its (first, count) slice of ONE run and the outputs are
    summed across ranks.  On the CPU box the slice results come from the oracle (slices are additive on both sides)."""
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    import oracle
    import tpmc_inputs as ti
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    cfg = ti.config("C4")[5].with_(N=30_000, mesh_fn=lambda: ti.satellite(4, 0.25))
    cfg._mesh_cache = []
    m = cfg.mesh()
    om = oracle.OracleMesh(m.vertices, m.indices, m.flags)
    first, count = bench.slice_of(rank, world, cfg.N)
    # bench.py --split slices: the plan of a step (same sweep point on every rank, this rank's particle range) ...
    assert bench.split_plan("slices", 70, rank, world, 64, cfg.N) == (6, first, count)
    assert bench.split_plan("attitudes", 70, rank, world, 64, cfg.N) == (bench.attitude_index(70, rank, world, 64), 0, cfg.N)
    r = om.run(cfg, first=first, count=count, debug=False)
    F, Tq, P, hits = bench.sum_slices([r.force, r.torque, r.facet_momentum, np.array([float(r.hits)])], world)
    # ... and its exchange step: the in-place all-reduce of the three output buffers, as the bench loop calls it
    bufs = [torch.tensor(r.force), torch.tensor(r.torque), torch.tensor(r.facet_momentum)]
    same = bench.allreduce_outputs(bufs, world)
    assert same[0] is bufs[0] and torch.equal(bufs[0], F) and torch.equal(bufs[1], Tq) and torch.equal(bufs[2], P)
    res = None
    if rank == 0:
        full = om.run(cfg, debug=False)
        res = (float(np.abs(F.numpy() - full.force).max() / np.abs(full.force).max()),
               float(np.abs(Tq.numpy() - full.torque).max() / max(np.abs(full.torque).max(), 1e-30)),
               float(np.abs(P.numpy() - full.facet_momentum).max() / np.abs(full.facet_momentum).max()),
               int(hits.item()) == full.hits, (first, count))
    out.put((rank, (first, count), res))
    dist.destroy_process_group()


def test_two_ranks_sum_particle_slices_of_one_run():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_slice_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    (_, s0, r0), (_, s1, _) = res
    assert s0 == (0, 15_000) and s1 == (15_000, 15_000)                       # disjoint cover of [0, N)
    eF, eT, eP, same_hits, _ = r0
    assert eF < 1e-12 and eT < 1e-11 and eP < 1e-12 and same_hits


def test_slices_cover_the_stream():
    sys.path.insert(0, ROOT)
    import bench
    t = [torch.ones(3)]
    assert bench.allreduce_outputs(t, 1)[0] is t[0] and bench.split_plan("slices", 3, 0, 1, 64, 10) == (3, 0, 10)
    for N, world in ((10, 3), (1_000_000_007, 8), (5, 8)):
        s = [bench.slice_of(r, world, N) for r in range(world)]
        assert s[0][0] == 0 and sum(c for _, c in s) == N
        assert all(s[k][0] + s[k][1] == s[k + 1][0] for k in range(world - 1))
