"""Row sharding over several GPUs (paper_1205_1222_b200/sharding.py, SURVEY.md 8(e) option 1 / NEXT-3).

CPU part: the partition's properties, and a world-size-2 gloo run in which each rank evaluates ITS rows with the
oracle (standing in for the kernels, which need a GPU) and the all-gather reassembles exactly the unsharded result.
GPU part (one GPU): the ranks of a 4-way job run one after the other on cuda:0; their rows together match the oracle."""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_1205_1222_b200 import inputs, sharding

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.parametrize("grain", [1, 32, 128])
def test_row_shard_partitions_the_block(grain):
    rng = np.random.default_rng(5)
    sizes = [0, 1, 127, 128, 129, 1000, 4096, 65536, 1048576] + [int(v) for v in rng.integers(0, 300000, 40)]
    for n_i in sizes:
        for world in (1, 2, 3, 4, 8):
            cuts = [sharding.row_shard(n_i, r, world, grain) for r in range(world)]
            assert cuts[0][0] == 0 and cuts[-1][1] == n_i
            for (lo, hi), (lo2, _) in zip(cuts, cuts[1:]):
                assert lo <= hi == lo2                       # contiguous, disjoint, in rank order
            lens = [hi - lo for lo, hi in cuts]
            assert sharding.shard_sizes(n_i, world, grain) == lens
            assert max(lens) - min(lens) < 2 * grain        # balanced: one grain, plus the block's ragged end
            assert all(lo % grain == 0 for lo, _ in cuts if lo < n_i)  # boundaries on CTA boundaries
            assert lens == sorted(lens, reverse=True)        # rank 0 owns a largest shard (ShardedContext sizes by it)


def test_shard_capacity_holds_every_block_up_to_n_i_max():
    """ShardedContext sizes its context by shard_capacity(n_i_max, world): every rank's shard of every block of up to
    n_i_max rows must fit, also when n_i is not a multiple of world x 128."""
    rng = np.random.default_rng(6)
    for world in (1, 2, 3, 4, 8):
        for n_i_max in [1, 127, 129, 333, 1000, 5000, 65537] + [int(v) for v in rng.integers(1, 200000, 10)]:
            cap = sharding.shard_capacity(n_i_max, world)
            assert cap >= 1
            for n_i in {n_i_max, max(1, n_i_max - 1), max(1, n_i_max // 2), max(1, n_i_max - 127), 1}:
                assert max(sharding.shard_sizes(n_i, world)) <= cap
            # tight: no more than one grain above an even split
            assert cap <= -(-n_i_max // world) + sharding.ROW_GRAIN


def test_row_shard_rejects_bad_arguments():
    for args in ((-1, 0, 1), (10, 1, 1), (10, -1, 2), (10, 0, 0)):
        with pytest.raises(ValueError):
            sharding.row_shard(*args)
    with pytest.raises(ValueError):
        sharding.row_shard(10, 0, 1, grain=0)


def _worker(rank, world, port, q):
    sys.path.insert(0, ROOT)
    import torch.distributed as dist
    from oracle import oracle
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK=str(rank), WORLD_SIZE=str(world))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    oracle.build()
    wl = inputs.make_custom(700, 333, 12, 64, seed_sub=3)   # 333 rows: shards of 256 and 77 at grain 128
    s = wl.state
    xp, vp = oracle.predict_state(s)
    lo, hi = sharding.row_shard(wl.n_i, rank, world)
    acc, jerk, cnt, _ = oracle.regular_force(xp, vp, s.m, wl.i_idx[lo:hi], wl.r_s[lo:hi], list_stride=wl.cap)
    full = {k: sharding.allgather_rows(torch.from_numpy(np.ascontiguousarray(v)), wl.n_i, rank, world)
            for k, v in (("acc", acc), ("jerk", jerk), ("nbr_count", cnt))}
    q.put((rank, (lo, hi), {k: v.numpy() for k, v in full.items()}))
    dist.barrier()
    dist.destroy_process_group()


def test_allgather_rows_world2_reassembles_the_unsharded_result(oracle):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    res = sorted((q.get(timeout=180) for _ in procs), key=lambda t: t[0])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [r[1] for r in res] == [(0, 256), (256, 333)]
    wl = inputs.make_custom(700, 333, 12, 64, seed_sub=3)
    s = wl.state
    xp, vp = oracle.predict_state(s)
    acc, jerk, cnt, _ = oracle.regular_force(xp, vp, s.m, wl.i_idx, wl.r_s, list_stride=wl.cap)
    for _, _, full in res:  # every rank holds all rows, bit for bit what one process computes
        assert np.array_equal(full["acc"], acc) and np.array_equal(full["jerk"], jerk)
        assert np.array_equal(full["nbr_count"], cnt)


def test_allgather_rows_single_rank_is_a_copy():
    t = torch.arange(12.0).reshape(4, 3)
    g = sharding.allgather_rows(t, 4, 0, 1)
    assert torch.equal(g, t) and g.data_ptr() != t.data_ptr()
    with pytest.raises(ValueError):
        sharding.allgather_rows(t[:2], 4, 0, 1)


@pytest.mark.gpu
@pytest.mark.parametrize("world", [1, 4])
def test_sharded_ranks_together_match_the_oracle(oracle, world):
    import parity

    wl = inputs.make_custom(5000, 1500, 24, 96, seed_sub=4, predict=lambda s: oracle.predict_state(s)[0])
    s = wl.state
    dev = torch.device("cuda:0")
    i_idx = torch.from_numpy(np.ascontiguousarray(wl.i_idx, dtype=np.int32)).to(dev)
    r_s = torch.from_numpy(np.ascontiguousarray(wl.r_s)).to(dev)
    gpu = {"acc": np.zeros((wl.n_i, 3)), "jerk": np.zeros((wl.n_i, 3)), "nbr_count": np.zeros(wl.n_i, np.int32),
           "nbr_list": np.full((wl.n_i, wl.cap), -7, np.int32), "n_overflow": np.zeros(1, np.int32)}
    covered = 0
    for rank in range(world):  # the ranks of one job, one after the other on the one GPU there is
        sc = sharding.ShardedContext(s.n, wl.n_i, wl.cap, rank, world)
        sc.set_state(s)
        out = sc.nb_regular_force(i_idx, r_s, s.t)
        torch.cuda.synchronize()
        lo, hi = sc.rows
        assert (lo, hi) == sharding.row_shard(wl.n_i, rank, world)
        for k in ("acc", "jerk", "nbr_count", "nbr_list"):
            gpu[k][lo:hi] = out[k][:hi - lo].cpu().numpy()
        gpu["n_overflow"] += out["n_overflow"].cpu().numpy()
        covered += hi - lo
        sc.close()
    assert covered == wl.n_i
    xp, vp = oracle.predict_state(s)
    parity.compare(oracle, xp, vp, s.m, wl.i_idx, wl.r_s, wl.cap, gpu)
