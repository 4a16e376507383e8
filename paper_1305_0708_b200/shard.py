"""Multi-GPU sharding of the Monte-Carlo integration.

Events are independent (one phase-space point per thread) and event k always uses Philox counter
k, so a batch [first, first + n) is split into contiguous counter ranges, one per rank; each rank runs
hg_integrate_step on its range and the only exchange is the sum of the four accumulators (sum w, sum w^2, n,
n_pass) -- one all-reduce of 4 doubles per step (NCCL on GPUs, gloo in the CPU tests), latency only.  A grid-optimisation
step (hg_set_grid with a histogram) has one more exchange: the histograms of w^2 per (draw, bin) of the ranks are
summed, [n_draws][n_bins] doubles (8 KB), so that every rank refines the same grid.
"""
import torch
import torch.distributed as dist


def shard_range(first_event, n_total, rank, world_size):
    """Contiguous split of [first_event, first_event + n_total): the first n_total % world ranks get one more."""
    base, extra = divmod(int(n_total), int(world_size))
    n = base + (1 if rank < extra else 0)
    start = int(first_event) + rank * base + min(rank, extra)
    return start, n


def combine_acc(acc, device=None, group=None):
    """All-reduce (sum) of (sum w, sum w^2, n, n_pass) over the ranks; identity without a process group."""
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return tuple(float(x) for x in acc)
    t = torch.tensor(list(acc), dtype=torch.float64, device=device or 'cpu')
    dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return tuple(t.tolist())


def combine_hist(hist, group=None):
    """All-reduce (sum) of the grid-optimisation histogram [n_draws, n_bins] over the ranks, in place; identity without
    a process group.  Every rank then calls hg_grid_refine on the same numbers and holds the same grid."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(hist, op=dist.ReduceOp.SUM, group=group)
    return hist
