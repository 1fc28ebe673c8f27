"""N > 1 host logic of bench.py (replicas: per-rank seeds, max-over-ranks time, summed updates),
exercised with world_size 2 over gloo on CPU."""
import os
import sys

import torch
import torch.distributed as dist
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import bench
    from paper_2107_05397_b200 import synth
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    p = synth.make_config("tiny", seed=bench.rank_seed(0, rank))
    ms_local = 10.0 + 5.0 * rank
    upd_local = float(p.n_pairs * 100 * (rank + 1))
    ms, upd = bench.reduce_over_ranks(ms_local, upd_local, world)
    q.put((rank, ms, upd, int(p.indices[:8].sum())))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_replica_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + (os.getpid() % 500)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (r0, ms0, u0, h0), (r1, ms1, u1, h1) = res
    assert ms0 == ms1 == 15.0                       # max over ranks
    assert u0 == u1 == 2016 * 100 * 3               # sum over ranks
    assert h0 != h1                                 # replicas work on different seeded problems


def test_single_rank_is_identity():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.reduce_over_ranks(3.5, 7.0, 1) == (3.5, 7.0)
