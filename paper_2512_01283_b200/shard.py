"""Multi-GPU plan of the path: packets are independent and carry a global id,
so the job shards by id range with the grid and tables replicated; the only exchange is one sum of the
fp64 image maps at the end of the job.  This module is host logic only (no arithmetic of the method)
and works with any torch.distributed backend (NCCL on GPUs, gloo in the CPU tests).
"""


def step_id_range(step, rank, world, batch, id0=0):
    """Global packet ids of `rank` in step `step` when every rank transports `batch` packets per step
    (weak scaling): steps are laid out one after another, ranks side by side inside a step.
    Returns (first_id, count).  The union over ranks and steps is [id0, id0 + steps*world*batch)
    without gaps or overlaps, so the result equals a single-GPU run over that range."""
    if not (0 <= rank < world) or batch < 0 or step < 0:
        raise ValueError("bad shard arguments")
    return id0 + (step * world + rank) * batch, batch


def split_range(id0, n, rank, world):
    """Strong-scaling split of ids [id0, id0+n) into `world` contiguous parts whose sizes differ by at
    most one.  Returns (first_id, count) of `rank`."""
    if not (0 <= rank < world) or n < 0:
        raise ValueError("bad shard arguments")
    base, rem = divmod(n, world)
    first = id0 + rank * base + min(rank, rem)
    return first, base + (1 if rank < rem else 0)


def reduce_images(img, group=None):
    """Sum the per-rank image maps in place (torch tensor, fp64) across the process group: the single
    collective of the path.  With world size 1 or no initialised process group this is a no-op."""
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        dist.all_reduce(img, op=dist.ReduceOp.SUM, group=group)
    return img
