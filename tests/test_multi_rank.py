"""world_size-2 gloo test of bench.py's multi-rank aggregation (replicas only: the ranks share no data;
value = total interactions / max-over-ranks time).  Calls bench.aggregate_ranks, the function bench.py itself runs."""
import os
import sys

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp


def _worker(rank, world, port, q):
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    # each rank: its own replica (different seed => different interaction count), its own step time
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    from workloads import make_workload
    from workloads.generators import SEED_BASE
    w = make_workload(1, N=512, seed=SEED_BASE + 1 + 1000 * rank if rank else None)
    inter = float(1000 + w.x[0] * 0 + 10 * rank)
    ms = 5.0 + rank
    import bench
    ms_step, e2e_ms, total = bench.aggregate_ranks(ms, 2.0 * ms, inter, dist, "cpu")
    assert e2e_ms == 12.0
    q.put((rank, ms_step, total, float(w.x[1])))
    dist.barrier()
    dist.destroy_process_group()


def test_two_rank_aggregation():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    ps = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    [p.start() for p in ps]
    res = sorted(q.get(timeout=120) for _ in range(2))
    [p.join(timeout=60) for p in ps]
    assert all(p.exitcode == 0 for p in ps)
    assert res[0][1] == res[1][1] == 6.0            # max over ranks
    assert res[0][2] == res[1][2] == 2010.0         # whole-job total
    assert res[0][3] != res[1][3]                   # replicas are independent inputs
