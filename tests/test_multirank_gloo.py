"""N > 1 is "replicas only": each rank runs the whole path on its own GPU and the only
communication is bench.py's MAX-over-ranks of the timed region.  Covered here with world_size 2 on CPU (gloo)."""
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
    t_local = 0.5 + 0.25 * rank  # rank 1 is the slow one
    t_max = bench.max_over_ranks(t_local, dist, torch.device("cpu"))
    rate = bench.whole_job_rate(1000, 4, world, t_max)
    out.put((rank, t_max, rate))
    dist.barrier()
    dist.destroy_process_group()


def test_max_over_ranks_and_whole_job_rate_world2():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 29500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    for rank, t_max, rate in res:
        assert t_max == 0.75  # both ranks see the slowest rank's time
        assert abs(rate - 2 * 1000 * 4 / 0.75 / 1e9) < 1e-18


def test_single_rank_needs_no_process_group():
    sys.path.insert(0, ROOT)
    import bench
    assert bench.max_over_ranks(0.125, None, torch.device("cpu")) == 0.125
    assert bench.whole_job_rate(10 ** 9, 2, 1, 0.5) == 4.0
