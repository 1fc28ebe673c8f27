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


def _shard_worker(rank, world, port, q):
    """Shard mode (unifrac_dm_shard): every pair is owned by exactly one rank, so summing the ranks' buffers (the
    merge of the paper's stripe pieces) reproduces the whole condensed matrix.  The owner map is the
    library's host helper; the stand-in 'distance' of pair k is k + 1."""
    sys.path.insert(0, ROOT)
    from paper_2107_05397_b200 import multigpu
    import numpy as np
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    n = 3300                                             # 26 tiles = 3 block rows of 12 tiles
    rng = np.random.default_rng(0)
    i = rng.integers(0, n - 1, size=4000)
    j = rng.integers(i + 1, n)
    pairs = np.unique(np.stack([i, j], 1), axis=0)
    own = np.array(multigpu.owner_of_pairs(pairs, world))
    buf = torch.zeros(len(pairs), dtype=torch.float64)
    mine = torch.from_numpy(own == rank)
    buf[mine] = torch.arange(1, len(pairs) + 1, dtype=torch.float64)[mine]
    multigpu.merge_shards(buf)                           # the routine bench.py calls on the NCCL path
    ok = bool(torch.equal(buf, torch.arange(1, len(pairs) + 1, dtype=torch.float64)))
    q.put((rank, ok, int(mine.sum()), len(pairs)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_shard_merge_by_sum():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 30100 + (os.getpid() % 500)
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, ok0, n0, tot), (_, ok1, n1, _) = res
    assert ok0 and ok1
    assert n0 + n1 == tot and n0 > 0 and n1 > 0      # disjoint, complete, both ranks own something
