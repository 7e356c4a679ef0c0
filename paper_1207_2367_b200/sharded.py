"""j-sharded multi-GPU driver: the paper's own decomposition (Table 1 row 7).

One process per GPU (torch.distributed, NCCL over NVLink 5 / NVSwitch).  Every rank holds the whole
state (replicated: 21 doubles per particle, 1.4 GB at N = 2^23), predicts all N, evaluates the m
active particles against ITS slice [j_begin, j_end) of the predicted particles only
(nb_set_j_range), and the partial (acc, jerk, snap) are summed with ONE all-reduce of 9 m doubles
before every rank runs the (identical) corrector.  The exchange is the only collective on the path;
at m = 2^20 it moves 75 MB against ~4 s / n of evaluation, so it never binds.

The all-reduce result is bit-identical on all ranks, the scheduler and the corrector are
deterministic, so the replicated states stay bit-identical without any further exchange.

This module only marshals: slices, buffers and the collective.  All arithmetic is in libnb.
"""
from __future__ import annotations

TILE = 128  # slice boundaries are multiples of the largest j-tile (include/nb.h: nb_set_j_range)


def j_range(N: int, rank: int, world: int) -> tuple[int, int]:
    """Contiguous slice of rank `rank`: whole tiles, sizes differing by at most one tile; the last
    non-empty slice ends at N.  Ranks beyond the number of tiles get an empty slice (N, N)."""
    if not (0 <= rank < world) or N < 1:
        raise ValueError("need 0 <= rank < world and N >= 1")
    tiles = (N + TILE - 1) // TILE
    base, extra = divmod(tiles, world)
    t0 = rank * base + min(rank, extra)
    t1 = t0 + base + (1 if rank < extra else 0)
    return min(t0 * TILE, N), min(t1 * TILE, N)


class ShardedNBody:
    """Block-step loop over `world` ranks.  `reduce(buf)` must sum `buf` (a float64 CUDA tensor)
    in place over the ranks; the default uses torch.distributed.all_reduce on the default group."""

    def __init__(self, pos, vel, mass, eps, eta, rank=None, world=None, reduce=None, **kw):
        import torch
        from . import nb
        self._nb, self._torch = nb, torch
        if rank is None or world is None:
            import torch.distributed as dist
            rank, world = dist.get_rank(), dist.get_world_size()
        self.rank, self.world = rank, world
        self.g = nb.NBody(pos, vel, mass, eps, eta, **kw)
        self.N = self.g.N
        jb, je = j_range(self.N, rank, world)
        self.empty = jb >= je            # more ranks than tiles: this rank contributes zeros
        if not self.empty:
            nb.nb_set_j_range(self.g.ctx, jb, je)
        self.j_begin, self.j_end = jb, je
        self._reduce = reduce or self._all_reduce
        self._buf = torch.empty(9 * self.N, dtype=torch.float64, device="cuda")

    def _all_reduce(self, buf):
        import torch.distributed as dist
        dist.all_reduce(buf, op=dist.ReduceOp.SUM)

    def partial(self, n):
        """Evaluate the n particles of the current set against this rank's slice; returns the
        contiguous [9][n] buffer of partial (acc, jerk, snap) that the ranks must sum."""
        nb, ctx = self._nb, self.g.ctx
        buf = self._buf[:9 * n]
        nb.nb_force(ctx, None, n)
        if self.empty:
            buf.zero_()
        else:
            nb.nb_get_forces(ctx, buf)
        return buf

    def finish(self, buf):
        """Store the summed buffer back as the evaluated values."""
        self._nb.nb_set_forces(self.g.ctx, buf)

    def _evaluate(self, n):
        buf = self.partial(n)
        self._reduce(buf)
        self.finish(buf)

    def startup(self):
        nb, ctx = self._nb, self.g.ctx
        nb.nb_predict(ctx, 0.0)
        self._evaluate(self.N)
        nb.nb_startup_commit(ctx, 1)
        self._evaluate(self.N)
        nb.nb_startup_commit(ctx, 2)

    def step(self):
        """One block step; returns (t_next, n_active)."""
        nb, ctx = self._nb, self.g.ctx
        tn, n = nb.nb_next_block(ctx)
        nb.nb_predict(ctx, tn)
        self._evaluate(n)
        nb.nb_correct_and_step(ctx)
        return tn, n

    def run_until(self, t_end):
        nb, ctx = self._nb, self.g.ctx
        steps = 0
        while True:
            tn, n = nb.nb_next_block(ctx)
            if tn > t_end:
                return steps
            nb.nb_predict(ctx, tn)
            self._evaluate(n)
            nb.nb_correct_and_step(ctx)
            steps += 1

    def close(self):
        self.g.close()
