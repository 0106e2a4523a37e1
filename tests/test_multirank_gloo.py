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


def _shard_worker(rank, world, port, out):
    """bench.py --shard rows, end to end, with the oracle standing in for the kernels (they need a GPU): shard_job ->
    the rank's rows -> timed region -> max over ranks -> whole-job rate with ONE replica."""
    sys.path.insert(0, ROOT)
    import time
    import numpy as np
    import bench
    from oracle import oracle
    from paper_1205_1222_b200 import inputs
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    oracle.build()
    wl = inputs.make_custom(900, 333, 10, 64, seed_sub=5)   # 333 rows: shards of 256 and 77 at grain 128 (uneven)
    local, job_pairs, job_replicas, rows = bench.shard_job(wl, rank, world, "rows")
    xp, vp = oracle.predict_state(wl.state)                 # every rank predicts all j itself
    t0 = time.perf_counter()
    acc, jerk, cnt, _ = oracle.regular_force(xp, vp, wl.state.m, local.i_idx, local.r_s, list_stride=wl.cap)
    t_local = time.perf_counter() - t0 + 0.25 * rank        # rank 1 is the slow one
    t_max = bench.max_over_ranks(t_local, dist, torch.device("cpu"))
    rate = bench.whole_job_rate(job_pairs, 3, job_replicas, t_max)
    out.put((rank, rows, local.n_i, job_pairs, job_replicas, t_local, t_max, rate, acc))
    dist.barrier()
    dist.destroy_process_group()


def test_shard_rows_bookkeeping_world2():
    sys.path.insert(0, ROOT)
    import numpy as np
    import bench
    from oracle import oracle
    from paper_1205_1222_b200 import inputs
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000
    procs = [ctx.Process(target=_shard_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    wl = inputs.make_custom(900, 333, 10, 64, seed_sub=5)
    assert [r[1] for r in res] == [(0, 256), (256, 333)] and [r[2] for r in res] == [256, 77]
    t_slowest = max(r[5] for r in res)
    for rank, rows, n_loc, job_pairs, job_replicas, t_local, t_max, rate, acc in res:
        assert job_pairs == wl.pairs == 333 * 900 and job_replicas == 1      # ONE job: the block's pairs counted once
        assert t_max == t_slowest                                              # both ranks see the slowest rank's time
        assert abs(rate - wl.pairs * 3 / t_slowest / 1e9) <= 1e-12 * rate     # strong scaling: whole block / slowest rank
    # the two shards are the rows of the unsharded result, bit for bit
    xp, vp = oracle.predict_state(wl.state)
    acc_full, _, _, _ = oracle.regular_force(xp, vp, wl.state.m, wl.i_idx, wl.r_s, list_stride=wl.cap)
    assert np.array_equal(np.concatenate([res[0][8], res[1][8]]), acc_full)
    # replicas (the default): every rank runs everything, the job is `world` replicas
    same, pairs, replicas, rows = bench.shard_job(wl, 1, 2, "none")
    assert same is wl and pairs == wl.pairs and replicas == 2 and rows is None
