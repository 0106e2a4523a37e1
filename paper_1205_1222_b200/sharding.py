"""Row sharding of one regular-force call over several GPUs (SURVEY.md 8(e) option 1, 8(f) NEXT-3).

The paper splits the regular force over its two GPUs ("the j-particles are split ... partial
forces and partial neighbour lists", regular-force time 45 -> 23 s).  On one NVSwitch domain the
other axis is the natural one: the ROWS (active particles) are independent units, so every rank holds the whole
j-set, predicts it itself (25 us at N = 2^20: cheaper than receiving it) and evaluates a contiguous slice of the
active block.  The slices' outputs are disjoint rows of the result: the force path has NO collective.  What a host
integrator may want afterwards -- every rank seeing all rows' acc / jerk / counts -- is one all-gather of 52 B per
row (allgather_rows below), outside the force path.

Only plumbing here: which rows a rank owns, and the optional all-gather; every step of the method runs in the
kernels behind binding.Context.  The default of bench.py stays "replicas only": `north_star`
fixes one GPU.  `bench.py --shard rows` times this module (strong scaling: the same block over N GPUs)."""
from __future__ import annotations

import torch

ROW_GRAIN = 128  # rows per CTA of the preferred launch shape: shard boundaries fall on CTA boundaries


def row_shard(n_i: int, rank: int, world: int, grain: int = ROW_GRAIN) -> tuple[int, int]:
    """Rows [lo, hi) of an active block of n_i rows owned by `rank` of `world`.

    Contiguous, disjoint, covering [0, n_i), in rank order; sizes differ by less than two grains (one grain of
    imbalance, and the ragged end of the block goes to the last rank that owns any rows).  Blocks smaller than
    world * grain leave the trailing ranks empty: a CTA's worth of rows is not worth splitting."""
    if n_i < 0 or world < 1 or not (0 <= rank < world) or grain < 1:
        raise ValueError("row_shard: need n_i >= 0, 0 <= rank < world, grain >= 1")
    units = -(-n_i // grain)                   # grains, the last one possibly ragged
    base, extra = divmod(units, world)
    lo_u = rank * base + min(rank, extra)      # the first `extra` ranks own one grain more
    hi_u = lo_u + base + (1 if rank < extra else 0)
    return min(lo_u * grain, n_i), min(hi_u * grain, n_i)


def shard_sizes(n_i: int, world: int, grain: int = ROW_GRAIN) -> list[int]:
    return [hi - lo for lo, hi in (row_shard(n_i, r, world, grain) for r in range(world))]


def shard_capacity(n_i_max: int, world: int, grain: int = ROW_GRAIN) -> int:
    """Rows a rank's context must hold so that ANY block of up to n_i_max rows fits its shard: the largest shard of the
    largest block (rank 0's), which is also the largest shard of every smaller block (shard sizes grow with n_i)."""
    lo, hi = row_shard(n_i_max, 0, world, grain)
    return max(hi - lo, 1)


def allgather_rows(local: torch.Tensor, n_i: int, rank: int, world: int, group=None,
                   grain: int = ROW_GRAIN) -> torch.Tensor:
    """All ranks' row slices of a per-row output (acc, jerk, nbr_count, ...) -> the full [n_i, ...] tensor on every
    rank.  `local` holds this rank's rows [lo, hi) first (it may be longer).  Shards differ in length, so each is
    padded to the longest for the collective (one `all_gather_into_tensor`)."""
    import torch.distributed as dist

    sizes = shard_sizes(n_i, world, grain)
    if local.shape[0] < sizes[rank]:
        raise ValueError("allgather_rows: local tensor shorter than this rank's shard")
    if world == 1:
        return local[:n_i].clone()
    longest = max(sizes)
    send = torch.zeros((longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    send[:sizes[rank]] = local[:sizes[rank]]
    recv = torch.empty((world * longest,) + tuple(local.shape[1:]), dtype=local.dtype, device=local.device)
    dist.all_gather_into_tensor(recv, send, group=group)
    return torch.cat([recv[r * longest:r * longest + sizes[r]] for r in range(world)], dim=0)


class ShardedContext:
    """binding.Context for one rank of a row-sharded job.  Every rank registers the FULL j-state (nb_set_j) and
    passes the FULL active block to nb_regular_force*; the rank's slice is taken here.  Outputs are the slice's
    rows; `rows` says which."""

    def __init__(self, n_max: int, n_i_max: int, nbr_cap: int, rank: int, world: int, device: int = 0, group=None):
        from . import binding  # loads the CUDA library: fails loudly without it

        self.rank, self.world, self.group = rank, world, group
        self.ctx = binding.Context(n_max, shard_capacity(n_i_max, world), nbr_cap, device=device)
        self.rows = (0, 0)

    def set_state(self, state):
        return self.ctx.set_state(state)

    def nb_set_j(self, *arrays):
        return self.ctx.nb_set_j(*arrays)

    def nb_predict_j(self, t: float, stream=None):
        return self.ctx.nb_predict_j(t, stream=stream)

    def nb_regular_force_ex(self, i_idx, r_s, t: float, dtr=None, want_pot: bool = False, out=None, stream=None):
        lo, hi = row_shard(int(i_idx.shape[0]), self.rank, self.world)
        self.rows = (lo, hi)
        return self.ctx.nb_regular_force_ex(i_idx[lo:hi], r_s[lo:hi], t, dtr=None if dtr is None else dtr[lo:hi],
                                            want_pot=want_pot, out=out, stream=stream)

    def nb_regular_force(self, i_idx, r_s, t: float, out=None, stream=None):
        return self.nb_regular_force_ex(i_idx, r_s, t, out=out, stream=stream)

    def allgather(self, out: dict, n_i: int, keys=("acc", "jerk", "nbr_count")) -> dict:
        """Every rank's acc / jerk / counts for all n_i rows (the lists stay with their owners)."""
        return {k: allgather_rows(out[k], n_i, self.rank, self.world, self.group) for k in keys}

    def close(self):
        self.ctx.close()
