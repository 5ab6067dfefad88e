"""Multi-GPU gridding: shard the rows over the ranks, one reduce of the grid.

The paper's decomposition: visibility rows split among the ranks, a private full-size grid
per rank, the grids summed on the master.  Here: one process per GPU, `wpg_shard_rows` (C ABI) for the split,
`wpg_grid` for the rank's rows, and ONE collective — `torch.distributed.reduce` of the N x N complex grid, NCCL over
NVLink on GPUs (gloo in the CPU tests) — plus a 5-word all-reduce of the counters.  north_star keeps the product
single-GPU ("no sharding and no collectives"); this module is the §8(f) extension and is not on bench.py's default
path (which runs replicas).  Argument marshalling only: nothing of the method's arithmetic lives here.
"""
import ctypes

from . import wpgrid


def shard_rows(nrow, world, rank, row_block=0):
    """[row0, row1) of `rank`: contiguous, disjoint, covering [0, nrow); whole time steps if row_block > 0."""
    r0, r1 = ctypes.c_int64(), ctypes.c_int64()
    rc = wpgrid.load().wpg_shard_rows(int(nrow), int(row_block), int(world), int(rank), ctypes.byref(r0), ctypes.byref(r1))
    if rc:
        raise wpgrid.WpgError(rc, "wpg_shard_rows: bad arguments")
    return int(r0.value), int(r1.value)


def reduce_grid(grid, dist, group=None, dst=0):
    """Sum of the ranks' private grids on rank `dst` (in place there; the other ranks' grids are left as they are,
    as after the paper's send to the master).  One collective of the whole grid; complex tensors travel as their
    real view."""
    import torch
    buf = torch.view_as_real(grid) if grid.is_complex() else grid
    dist.reduce(buf, dst=dst, op=dist.ReduceOp.SUM, group=group)
    return grid


def reduce_stats(stats, dist, device, group=None):
    """The five counters summed over the ranks (every rank gets the totals)."""
    import torch
    t = torch.tensor([stats[k] for k in wpgrid.Stats().as_dict()], dtype=torch.int64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return {k: int(v) for k, v in zip(wpgrid.Stats().as_dict(), t.tolist())}


def grid_sharded(ctx, vis, uvw, weight, freq, stack, dist, group=None, dst=0, row_block=0, rows="local", stats=False):
    """Grid this rank's rows into a private grid and reduce the grids onto rank `dst`.

    rows="local": the arrays hold this rank's rows only (the paper's layout: every rank loads its own slice);
    rows="all": the arrays hold all rows on every rank and the rank's slice is taken here (wpg_shard_rows).
    Returns (grid — the sum on rank dst, this rank's part elsewhere —, summed counters or None)."""
    if rows == "all":
        r0, r1 = shard_rows(uvw.shape[0], dist.get_world_size(group), dist.get_rank(group), row_block)
        vis, uvw, weight = vis[r0:r1], uvw[r0:r1], weight[r0:r1]
    if row_block:
        ctx.set_option("row_block", row_block)
    g, s = ctx.grid(vis.contiguous(), uvw.contiguous(), weight.contiguous(), freq, stack, stats=True)
    reduce_grid(g, dist, group, dst)
    return g, (reduce_stats(s, dist, g.device, group) if stats else None)
