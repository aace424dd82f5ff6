"""N > 1 path of bench.py on CPU: world_size-2 gloo processes (no GPU work).

The path shards by independent samples (one lattice per rank, seed + rank), so the only
cross-rank logic is: which sample a rank runs, max-over-ranks of the timed region, and sums of the
work counters.  The oracle stands in for the GPU here only to show that the two ranks' samples are
different, reproducible chains.
"""
import os
import sys

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import workloads


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    import oracle
    dist.init_process_group("gloo", rank=rank, world_size=world)
    w = workloads.CONFIGS[1]
    seed = bench.rank_seed(w, rank)
    o = oracle.OraclePotts(w.L, w.q, seed, w.init)
    E, _ = o.sweep_measured(w.temperatures[0], 5, 1, hist=False)
    # rank r pretends its timed region took 10 + 5 r ms for 1000 (r + 1) updates and 3 launches
    ms, upd, launches = bench.reduce_over_ranks(dist, "cpu", 10.0 + 5.0 * rank, 1000 * (rank + 1), 3)
    q.put((rank, seed, [int(x) for x in E], ms, upd, launches))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_gloo_independent_samples_and_reduction():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 2000)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, s0, E0, ms0, u0, l0), (r1, s1, E1, ms1, u1, l1) = res
    w = workloads.CONFIGS[1]
    assert (s0, s1) == (w.seed, w.seed + 1)
    assert E0 != E1                                  # two different samples
    assert E0[0] == -1676                            # rank 0 runs the golden chain of config 1
    assert ms0 == ms1 == 15.0                        # max over ranks
    assert u0 == u1 == 3000 and l0 == l1 == 6        # sums over ranks
